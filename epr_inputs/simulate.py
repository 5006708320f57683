"""Detector-image simulator: paraxial Fresnel propagation + Poisson noise (numpy only).

This is the *physics* the EPR method inverts (Eq. (S5)-(S7)), not the method:
the paper's algorithm never evaluates a Fresnel integral.  It makes detector images
whose structure (edge-enhancement fringes, caustic-like peaks at sharp interfaces, Poisson noise
at 1e4 photons/px) matches the paper's beamline workloads, without touching any operator of the
method, so neither the oracle nor the CUDA path can inherit an error from it.
"""
from __future__ import annotations

import numpy as np

HC_KEV_M = 1.2398419843e-9


def material_constants(energy_keV):
    """Synthetic optical constants: soft A: delta = 2.0e-8 (100/E)^2, beta = 2.0e-11 (100/E)^3
    (delta/beta = 1000 at 100 keV); bone-like B: beta_B = 10 beta_A, delta_B = 200 beta_B."""
    E = float(energy_keV)
    dA = 2.0e-8 * (100.0 / E) ** 2
    bA = 2.0e-11 * (100.0 / E) ** 3
    bB = 10.0 * bA
    dB = 200.0 * bB * (E / 100.0)      # delta_B/beta_B = 200 at 100 keV, proportional to E like material A
    return np.array([dA, dB]), np.array([bA, bB])


def exit_wave(t_px, pixel_m, energy_keV):
    """Object-plane intensity and phase of one spectral line: I = exp(-sum_m mu_m t_m),
    phi = -k sum_m delta_m t_m, mu = 2 k beta (projection approximation)."""
    k = 2.0 * np.pi * energy_keV / HC_KEV_M
    delta, beta = material_constants(energy_keV)
    nm = t_px.shape[0]
    t_m = t_px * pixel_m
    phi = -k * np.tensordot(delta[:nm], t_m, axes=1)
    I = np.exp(-2.0 * k * np.tensordot(beta[:nm], t_m, axes=1))
    return I, phi


def fresnel_detector(t_px, pixel_m, L_m, energy_keV, weight):
    """Noise-free flat-field-normalised detector intensity sum_s f_s |Fresnel_L[sqrt(I_s) e^{i phi_s}]|^2
    on the periodic (ny, nx) grid (transfer function exp(-i pi lambda L |f|^2), Eq. (S5))."""
    E = np.atleast_1d(np.asarray(energy_keV, dtype=np.float64))
    w = np.atleast_1d(np.asarray(weight, dtype=np.float64))
    w = w / w.sum()
    ny, nx = t_px.shape[1:]
    fx = np.fft.fftfreq(nx, d=pixel_m)
    fy = np.fft.fftfreq(ny, d=pixel_m)
    f2 = fy[:, None] ** 2 + fx[None, :] ** 2
    out = np.zeros((ny, nx), dtype=np.float64)
    for s in range(E.size):
        lam = HC_KEV_M / E[s]
        I, phi = exit_wave(t_px, pixel_m, E[s])
        psi = np.sqrt(I) * np.exp(1j * phi)
        psi_L = np.fft.ifft2(np.fft.fft2(psi) * np.exp(-1j * np.pi * lam * L_m * f2))
        out += w[s] * (psi_L.real ** 2 + psi_L.imag ** 2)
    return out


def poisson_noise(I_det, photons_per_px, seed):
    """d = Poisson(N * max(I_det, 0)) / N, returned as float32 (what the detector delivers)."""
    rng = np.random.default_rng(seed)
    lam = photons_per_px * np.maximum(I_det, 0.0)
    return (rng.poisson(lam) / float(photons_per_px)).astype(np.float32)
