"""Random-ellipsoid phantoms projected to thickness maps (closed-form chords).

Recipe (DESIGN.md §"Synthetic inputs", after SURVEY.md §8(d)): ellipsoid i has its centre uniform in
the central 60 % of the field, semi-axes uniform in [5, 40]·scale px, a uniformly random orientation
(unit quaternion) and a material drawn uniformly.  The projected thickness along z is the chord of
the rotated ellipsoid, 2·sqrt(disc)/M_zz, summed over ellipsoids.  A "shell" is an ellipsoid minus
its concentric copy scaled by 0.8 (sharp, unsmoothed edges).
"""
from __future__ import annotations

import numpy as np


def _random_rotation(rng):
    q = rng.normal(size=4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)],
    ])


def _add_chord(t, centre, M, sign=1.0):
    """Add sign * chord length (px) of the ellipsoid (r-c)^T M (r-c) <= 1 along z to t[y][x]."""
    ny, nx = t.shape
    Minv = np.linalg.inv(M)
    hx = np.sqrt(Minv[0, 0])
    hy = np.sqrt(Minv[1, 1])
    x_lo = max(int(np.floor(centre[0] - hx)) - 1, 0)
    x_hi = min(int(np.ceil(centre[0] + hx)) + 2, nx)
    y_lo = max(int(np.floor(centre[1] - hy)) - 1, 0)
    y_hi = min(int(np.ceil(centre[1] + hy)) + 2, ny)
    if x_hi <= x_lo or y_hi <= y_lo:
        return
    X = np.arange(x_lo, x_hi, dtype=np.float64)[None, :] - centre[0]
    Y = np.arange(y_lo, y_hi, dtype=np.float64)[:, None] - centre[1]
    B = M[0, 2] * X + M[1, 2] * Y
    C = M[0, 0] * X * X + 2.0 * M[0, 1] * X * Y + M[1, 1] * Y * Y - 1.0
    disc = B * B - M[2, 2] * C
    t[y_lo:y_hi, x_lo:x_hi] += sign * 2.0 * np.sqrt(np.maximum(disc, 0.0)) / M[2, 2]


def ellipsoid_phantom(ny, nx, n_ellipsoids, n_materials, seed, shells_for_material=None,
                      axis_scale=None, rotation_deg=None, cylinder=False):
    """Return thickness maps t[m][y][x] in PIXELS for each material m.

    shells_for_material: material index whose ellipsoids are hollow shells (or None).
    rotation_deg: rotate the whole 3-D phantom about the vertical (y) axis before projecting.
    cylinder: draw centres inside a vertical cylinder of radius 0.3*nx (3-D consistent phantom).
    """
    rng = np.random.default_rng(seed)
    if axis_scale is None:
        # semi-axes 5-40 px at 256^2, 20-160 px at 2048^2; linear in between
        axis_scale = max(nx / 512.0, min(1.0, nx / 256.0))
    t = np.zeros((n_materials, ny, nx), dtype=np.float64)
    Ry = np.eye(3)
    if rotation_deg is not None:
        c, s = np.cos(np.deg2rad(rotation_deg)), np.sin(np.deg2rad(rotation_deg))
        Ry = np.array([[c, 0.0, s], [0.0, 1.0, 0.0], [-s, 0.0, c]])
    mid = np.array([nx / 2.0, ny / 2.0, 0.0])
    for _ in range(n_ellipsoids):
        if cylinder:
            rad = 0.3 * nx * np.sqrt(rng.uniform())
            ang = rng.uniform(0.0, 2.0 * np.pi)
            centre = np.array([nx / 2.0 + rad * np.cos(ang), rng.uniform(0.2 * ny, 0.8 * ny), rad * np.sin(ang)])
        else:
            centre = np.array([rng.uniform(0.2 * nx, 0.8 * nx), rng.uniform(0.2 * ny, 0.8 * ny), 0.0])
        axes = rng.uniform(5.0, 40.0, size=3) * axis_scale
        R = _random_rotation(rng)
        m = int(rng.integers(0, n_materials))
        R = Ry @ R
        centre = mid + Ry @ (centre - mid)
        M = R @ np.diag(1.0 / axes ** 2) @ R.T
        _add_chord(t[m], centre, M, +1.0)
        if shells_for_material is not None and m == shells_for_material:
            _add_chord(t[m], centre, M / 0.64, -1.0)   # concentric copy scaled by 0.8
    return t
