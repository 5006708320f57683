"""The five BASELINE.json workloads (C1..C5) as seeded synthetic generators.

Seeds: phantom = 1000 + config number, noise = 2000 + config number (+ projection index for C5).
Everything is generated in fp64; `d` is stored as fp32.  Sizes can be reduced (`n=`) for parity
tests — the phantom then has proportionally fewer ellipsoids and smaller semi-axes.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from .phantom import ellipsoid_phantom
from .simulate import HC_KEV_M, exit_wave, fresnel_detector, poisson_noise


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    batch: int
    pixel_m: float
    L_m: float
    energy_keV: np.ndarray
    weight: np.ndarray
    delta_over_beta: np.ndarray      # what the RETRIEVAL assumes (single-material hypothesis, R14)
    solver: str                      # "local" | "nonlocal"
    iterations: int
    step: float
    max_shift_px: float              # S (R6)
    target_shift_px: float
    d: np.ndarray = field(repr=False, default=None)          # [batch][ny][nx] float32
    thickness_px: np.ndarray = field(repr=False, default=None)  # [n_materials][ny][nx] of projection 0
    seed_noise: int = 0

    @property
    def n_bins(self):
        return int(np.size(self.energy_keV))


CONFIGS = {
    # name: (ny, nx, batch, n_ellipsoids, n_materials, shells, energies, solver, iterations, step, target, S, db@100keV)
    "C1": dict(ny=256, nx=256, batch=1, n_ell=20, n_mat=1, shells=False, poly=False, solver="local",
               iterations=10, step=1.0, target=0.3, S=16.0, db100=1000.0),
    "C2": dict(ny=2048, nx=2048, batch=1, n_ell=200, n_mat=2, shells=False, poly=False, solver="local",
               iterations=20, step=1.0, target=0.5, S=16.0, db100=1000.0),
    "C3": dict(ny=2048, nx=2048, batch=1, n_ell=200, n_mat=2, shells=True, poly=False, solver="nonlocal",
               iterations=20, step=0.4, target=5.0, S=16.0, db100=200.0),
    "C4": dict(ny=2048, nx=2048, batch=1, n_ell=200, n_mat=2, shells=True, poly=True, solver="nonlocal",
               iterations=20, step=0.4, target=5.0, S=16.0, db100=200.0),
    "C5": dict(ny=2160, nx=2560, batch=64, n_ell=200, n_mat=2, shells=True, poly=True, solver="nonlocal",
               iterations=20, step=0.4, target=8.0, S=24.0, db100=200.0),
}

PIXEL_M = 6.5e-6
PHOTONS = 1.0e4


def _spectrum(poly):
    if not poly:
        return np.array([100.0]), np.array([1.0])
    E = np.linspace(60.0, 140.0, 8)
    w = np.exp(-0.5 * ((E - 100.0) / 20.0) ** 2)
    return E, w / w.sum()


def _max_phase_gradient(t_px, pixel_m, energy_keV):
    _, phi = exit_wave(t_px, pixel_m, energy_keV)
    gx = np.abs(np.roll(phi, -1, 1) - np.roll(phi, 1, 1)) / 2.0
    gy = np.abs(np.roll(phi, -1, 0) - np.roll(phi, 1, 0)) / 2.0
    return float(max(gx.max(), gy.max()))


def make_workload(name, n=None, batch=None, noise=True, distinct=None, first=0):
    """Build workload `name` (C1..C5).  n: override grid (n x n, or (ny, nx)); batch: override batch.
    distinct: number of distinct simulated projections (the rest of the batch re-draws only the
    Poisson noise of projection j % distinct) — bounds host-side generation time for large batches.
    first: the batch is the slice [first, first + batch) of one larger seeded batch (projection j of that batch has the
    same image and the same noise whoever generates it): what rank k of a multi-GPU run gets from `shard_range`."""
    c = CONFIGS[name]
    num = int(name[1:])
    ny, nx = c["ny"], c["nx"]
    if n is not None:
        ny, nx = (n, n) if np.isscalar(n) else n
    B = c["batch"] if batch is None else batch
    n_ell = max(4, int(round(c["n_ell"] * (nx * ny) / float(c["nx"] * c["ny"]))))
    E, w = _spectrum(c["poly"])
    e_ref = float(E[np.argmin(np.abs(E - 100.0))])
    shells = 1 if c["shells"] else None
    n_distinct = B if distinct is None else min(distinct, B)

    rng_rot = np.random.default_rng(1000 + num)
    angles = np.degrees(rng_rot.uniform(0.0, np.pi, size=max(B, 1))) if name == "C5" else [None] * B

    phantoms = []
    for j in range(n_distinct):
        phantoms.append(ellipsoid_phantom(ny, nx, n_ell, c["n_mat"], 1000 + num, shells_for_material=shells,
                                          rotation_deg=angles[j], cylinder=(name == "C5")))
    gmax = max(_max_phase_gradient(t, PIXEL_M, e_ref) for t in phantoms)
    k_ref = 2.0 * np.pi * e_ref / HC_KEV_M
    L_m = c["target"] * k_ref * PIXEL_M ** 2 / gmax

    clean = [fresnel_detector(t, PIXEL_M, L_m, E, w) for t in phantoms]
    d = np.empty((B, ny, nx), dtype=np.float32)
    for j in range(B):
        g = int(first) + j                                # index in the global batch
        img = clean[g % n_distinct]
        d[j] = poisson_noise(img, PHOTONS, 2000 + num + 7919 * g) if noise else img.astype(np.float32)

    db = c["db100"] * E / 100.0
    return Workload(name=name, nx=nx, ny=ny, batch=B, pixel_m=PIXEL_M, L_m=L_m, energy_keV=E, weight=w,
                    delta_over_beta=db, solver=c["solver"], iterations=c["iterations"], step=c["step"],
                    max_shift_px=c["S"], target_shift_px=c["target"], d=d, thickness_px=phantoms[0],
                    seed_noise=2000 + num)


def shard_range(total, rank, world):
    """Contiguous, balanced split of `total` independent projections over `world` ranks (no exchange step:
    PAPER.md:231 is per radiograph).  Returns (start, stop) for `rank`."""
    base, rem = divmod(int(total), int(world))
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)
