"""Pins for the fp64 oracle's operators (CPU only).

Each test checks `oracle/epr_oracle.py` against something the paper or the mathematics fixes —
closed forms, invariants, brute force from the printed definition, or a library routine used in a
different way — never against a retyped copy of the oracle's own formula.
"""
import math

import numpy as np
import pytest

from oracle import epr_oracle as O

RNG = np.random.default_rng(12345)


# ------------------------------------------------------------------ constants (Eq. (2), (S8), (6))
def test_lines_from_S8_form():
    """eps = lambda L / (2 pi) (Eq. (S8)) with lambda = hc/E; alpha = eps/p^2; a = alpha db/2."""
    E, p, L, db = 100.0, 6.5e-6, 4.6, 1000.0
    lam = 1.2398419843e-9 / E                       # 0.12398 Angstrom at 100 keV
    assert abs(lam - 1.2398419843e-11) < 1e-24
    eps = lam * L / (2.0 * math.pi)
    lines = O.derive_lines(p, L, [E], [1.0], [db])
    assert lines.alpha[0] == pytest.approx(eps / p ** 2, rel=1e-14)
    assert lines.a[0] == pytest.approx(eps / p ** 2 * db / 2.0, rel=1e-14)
    assert lines.a[0] == pytest.approx(107.42, rel=2e-4)      # tests/golden/c1_scalars.txt
    assert lines.f[0] == 1.0 and lines.gamma[0] == pytest.approx(1.0)


def test_gamma_normalisation_and_energy_scaling():
    """R11: mu_s ∝ 1/(E_s db_s); with delta ∝ E^-2 and beta ∝ E^-3 (db ∝ E) this is mu ∝ E^-2."""
    E = np.linspace(60.0, 140.0, 8)
    w = np.exp(-0.5 * ((E - 100.0) / 20.0) ** 2)
    lines = O.derive_lines(6.5e-6, 10.0, E, w, 200.0 * E / 100.0)
    assert np.sum(lines.f) == pytest.approx(1.0, abs=1e-15)
    assert np.sum(lines.f * lines.gamma) == pytest.approx(1.0, abs=1e-14)
    assert lines.gamma[0] / lines.gamma[-1] == pytest.approx((140.0 / 60.0) ** 2, rel=1e-13)
    # a_s = L delta_s/(mu_s p^2): delta ∝ E^-2 and mu ∝ E^-2 cancel
    assert np.ptp(lines.a) / lines.a[0] < 1e-13


# ------------------------------------------------------------------ splat / gather
def test_splat_zero_shift_is_identity():
    I = RNG.uniform(0.1, 2.0, size=(17, 23))
    z = np.zeros_like(I)
    assert np.array_equal(O.splat(I, z, z), I)
    assert np.array_equal(O.gather(I, z, z), I)


@pytest.mark.parametrize("mx,my", [(3, 0), (-2, 5), (0, -7), (23, 17)])
def test_splat_integer_shift_is_roll(mx, my):
    I = RNG.uniform(0.1, 2.0, size=(17, 23))
    ux = np.full_like(I, float(mx))
    uy = np.full_like(I, float(my))
    assert np.array_equal(O.splat(I, ux, uy), np.roll(I, (my, mx), axis=(0, 1)))
    # the adjoint of a rigid shift is the opposite shift
    assert np.array_equal(O.gather(I, ux, uy), np.roll(I, (-my, -mx), axis=(0, 1)))


def test_splat_fractional_shift_is_bilinear_mix_of_rolls():
    I = RNG.uniform(0.1, 2.0, size=(16, 20))
    sx, sy = 2.25, -1.5          # floor = (2, -2), frac = (0.25, 0.5): exactly representable
    P = O.splat(I, np.full_like(I, sx), np.full_like(I, sy))
    ref = (0.75 * 0.5 * np.roll(I, (-2, 2), (0, 1)) + 0.25 * 0.5 * np.roll(I, (-2, 3), (0, 1))
           + 0.75 * 0.5 * np.roll(I, (-1, 2), (0, 1)) + 0.25 * 0.5 * np.roll(I, (-1, 3), (0, 1)))
    assert np.max(np.abs(P - ref)) < 1e-15


def test_ray_map_constant_gradient_gives_closed_form_shift():
    """"a constant phase gradient gives a rigid detector shift by the closed-form number of pixels":
    I = exp(c x) => phi = (db/2) c x (Eq. (6)); shift = L dphi/dx /(k p) with dphi/dx = (db/2) c / p."""
    E, p, db, c = 100.0, 6.5e-6, 1000.0, -2.0e-3
    k = 2.0 * math.pi * E / 1.2398419843e-9
    shift_px = -3.0                                   # choose L so that the shift is exactly -3 px
    L = shift_px * k * p * p / ((db / 2.0) * c)
    lines = O.derive_lines(p, L, [E], [1.0], [db])
    ny, nx = 12, 64
    I = np.exp(c * np.arange(nx, dtype=np.float64))[None, :].repeat(ny, 0)
    ux, uy = O.ray_map(I, lines.a[0], 4.0)
    assert np.max(np.abs(ux[:, 1:-1] - shift_px)) < 1e-9   # interior: D0 of a linear function is exact
    assert np.max(np.abs(uy)) == 0.0
    P = O.splat(I, ux, uy)
    # interior source pixels land on x-3; the two wrap columns (x = 0, nx-1) see a jump in ln I, are
    # clamped to +4 px and land on detector columns 4 and 3 — outside the compared range
    assert np.max(np.abs(P[:, 8:nx - 5] - I[:, 11:nx - 2])) < 1e-9


def test_ray_map_clamps_to_S():
    I = np.exp(np.cumsum(RNG.normal(size=(8, 32)), axis=1))
    ux, uy = O.ray_map(I, 50.0, 4.0)
    assert ux.max() <= 4.0 and ux.min() >= -4.0 and uy.max() <= 4.0 and uy.min() >= -4.0
    assert (np.abs(ux) == 4.0).any()


def test_splat_mass_conservation_and_linearity():
    """for a fixed shift field M_s is linear in I_s and mass conserving."""
    I1 = RNG.uniform(0.0, 3.0, size=(33, 47))
    I2 = RNG.uniform(0.0, 3.0, size=(33, 47))
    ux = RNG.uniform(-8.0, 8.0, size=I1.shape)
    uy = RNG.uniform(-8.0, 8.0, size=I1.shape)
    P = O.splat(I1, ux, uy)
    assert abs(P.sum() - I1.sum()) <= 1e-12 * I1.sum()
    lin = O.splat(2.0 * I1 - 0.5 * I2, ux, uy) - (2.0 * P - 0.5 * O.splat(I2, ux, uy))
    assert np.max(np.abs(lin)) < 1e-13


def test_adjointness():
    """<M x, y> = <x, M* y>."""
    x = RNG.normal(size=(31, 29))
    y = RNG.normal(size=(31, 29))
    ux = RNG.uniform(-8.0, 8.0, size=x.shape)
    uy = RNG.uniform(-8.0, 8.0, size=x.shape)
    lhs = np.sum(O.splat(x, ux, uy) * y)
    rhs = np.sum(x * O.gather(y, ux, uy))
    assert abs(lhs - rhs) <= 1e-12 * max(1.0, abs(lhs))


def _dense_splat_matrix(ux, uy):
    """Brute force from the printed definition, pure Python, periodic wrap."""
    ny, nx = ux.shape
    M = np.zeros((ny * nx, ny * nx))
    for y in range(ny):
        for x in range(nx):
            xt, yt = x + ux[y, x], y + uy[y, x]
            x0, y0 = math.floor(xt), math.floor(yt)
            dx, dy = xt - x0, yt - y0
            src = y * nx + x
            for (yy, xx, w) in ((y0, x0, (1 - dx) * (1 - dy)), (y0, x0 + 1, dx * (1 - dy)),
                                (y0 + 1, x0, (1 - dx) * dy), (y0 + 1, x0 + 1, dx * dy)):
                M[(yy % ny) * nx + (xx % nx), src] += w
    return M


def test_splat_gather_against_dense_matrix():
    ny = nx = 8
    ux = RNG.uniform(-5.0, 5.0, size=(ny, nx))
    uy = RNG.uniform(-5.0, 5.0, size=(ny, nx))
    ux[0, 0], uy[0, 0] = -0.25, -3.0        # negative coordinates: floor, not truncation (R7)
    M = _dense_splat_matrix(ux, uy)
    I = RNG.uniform(0.0, 2.0, size=(ny, nx))
    e = RNG.normal(size=(ny, nx))
    assert np.max(np.abs(O.splat(I, ux, uy).ravel() - M @ I.ravel())) < 1e-14
    assert np.max(np.abs(O.gather(e, ux, uy).ravel() - M.T @ e.ravel())) < 1e-14
    assert np.max(np.abs(M.sum(axis=0) - 1.0)) < 1e-14     # every column distributes exactly one unit


def test_subpixel_splat_is_first_order_upwind():
    """For |u_x| < 1, u_y = 0 the splat is the conservative upwind scheme
    P[x] = I[x](1-|u[x]|) + (u+ I)[x-1] + (u- I)[x+1]   (exact identity)."""
    I = RNG.uniform(0.1, 2.0, size=(9, 40))
    u = RNG.uniform(-0.99, 0.99, size=I.shape)
    up, um = np.maximum(u, 0.0), np.maximum(-u, 0.0)
    ref = I * (1.0 - np.abs(u)) + np.roll(up * I, 1, axis=1) + np.roll(um * I, -1, axis=1)
    assert np.max(np.abs(O.splat(I, u, np.zeros_like(u)) - ref)) < 1e-14


# ------------------------------------------------------------------ preconditioner
@pytest.mark.parametrize("symbol", [0, 1])
def test_filter_single_mode_closed_form(symbol):
    """a single Fourier mode comes back scaled by 1/(1 + a lambda(theta))."""
    ny, nx, m, n, a = 24, 40, 3, 5, 57.3
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    thx, thy = 2 * math.pi * m / nx, 2 * math.pi * n / ny
    mode = np.cos(thx * x + thy * y + 0.3)
    lam = (2 - 2 * math.cos(thx)) + (2 - 2 * math.cos(thy)) if symbol == 0 else thx ** 2 + thy ** 2
    out = O.precondition(2.5 + mode, a, symbol)
    assert np.max(np.abs(out - (2.5 + mode / (1.0 + a * lam)))) < 1e-13     # DC gain 1


def test_filter_inverts_the_R1_linear_operator_and_matches_dense_dft():
    ny = nx = 16
    a = 11.0
    r = RNG.normal(size=(ny, nx))
    # (1) it is the exact inverse of I -> I - a lap5(I), evaluated with plain rolls
    q = O.precondition(r, a, 0)
    back = q - a * (np.roll(q, 1, 0) + np.roll(q, -1, 0) + np.roll(q, 1, 1) + np.roll(q, -1, 1) - 4 * q)
    assert np.max(np.abs(back - r)) < 1e-12
    # (2) O(N^2) dense DFT matrices instead of np.fft
    Fy = np.exp(-2j * np.pi * np.outer(np.arange(ny), np.arange(ny)) / ny)
    Fx = np.exp(-2j * np.pi * np.outer(np.arange(nx), np.arange(nx)) / nx)
    R = Fy @ r @ Fx.T
    ky = np.minimum(np.arange(ny), ny - np.arange(ny)) * 2 * np.pi / ny
    kx = np.minimum(np.arange(nx), nx - np.arange(nx)) * 2 * np.pi / nx
    for symbol in (0, 1):
        lam = ((2 - 2 * np.cos(ky))[:, None] + (2 - 2 * np.cos(kx))[None, :]) if symbol == 0 \
            else (ky ** 2)[:, None] + (kx ** 2)[None, :]
        dense = np.real(np.conj(Fy) @ (R / (1 + a * lam)) @ np.conj(Fx).T) / (ny * nx)
        assert np.max(np.abs(O.precondition(r, a, symbol) - dense)) < 1e-12


# ------------------------------------------------------------------ local closure
def test_closure_exponential_closed_form():
    """I = exp(cx + dy): interior P = I [1 - a(kc+kd) + (a^2/2)(c^2 kc + d^2 kd + 2cd sinh c sinh d)],
    k_c = 2 cosh c - 2; the WKB1 term vanishes because Q is constant."""
    ny, nx, c, d, a, alpha = 20, 24, 0.013, -0.021, 37.0, 0.9
    y, x = np.meshgrid(np.arange(ny, dtype=float), np.arange(nx, dtype=float), indexing="ij")
    I = np.exp(c * x + d * y)
    kc, kd = 2 * math.cosh(c) - 2, 2 * math.cosh(d) - 2
    fac = 1 - a * (kc + kd) + 0.5 * a * a * (c * c * kc + d * d * kd + 2 * c * d * math.sinh(c) * math.sinh(d))
    P = O.closure(I, a, alpha, order=2, wkb1=True)
    sl = (slice(3, ny - 3), slice(3, nx - 3))
    assert np.max(np.abs(P[sl] / I[sl] - fac)) < 1e-12
    P1 = O.closure(I, a, alpha, order=1)
    assert np.max(np.abs(P1[sl] / I[sl] - (1 - a * (kc + kd)))) < 1e-13


def _spectral_derivs(f):
    """Exact derivatives of a band-limited periodic field by FFT (independent of finite differences)."""
    ny, nx = f.shape
    kx = 2j * np.pi * np.fft.fftfreq(nx)[None, :]
    ky = 2j * np.pi * np.fft.fftfreq(ny)[:, None]
    F = np.fft.fft2(f)
    return (lambda px, py: np.real(np.fft.ifft2(F * kx ** px * ky ** py)))


def _continuum_closure_terms(I, db):
    """Eq. (1) PAPER.md:146 term by term with spectral derivatives, phi = (db/2) ln I, pixel units,
    eps = 1:  T1 = d_i(I d_i phi), T2 = d_i d_j(I d_i phi d_j phi), T3 = d_i(I d_i Q)."""
    D = _spectral_derivs
    phi = 0.5 * db * np.log(I)
    px, py = D(phi)(1, 0), D(phi)(0, 1)
    T1 = D(I * px)(1, 0) + D(I * py)(0, 1)
    T2 = D(I * px * px)(2, 0) + D(I * py * py)(0, 2) + 2 * D(I * px * py)(1, 1)
    A = np.sqrt(I)
    Q = (D(A)(2, 0) + D(A)(0, 2)) / A
    T3 = D(I * D(Q)(1, 0))(1, 0) + D(I * D(Q)(0, 1))(0, 1)
    return T1, T2, T3


@pytest.mark.parametrize("which", ["order1", "wkb0", "wkb1"])
def test_closure_converges_to_eq1_at_second_order(which):
    """The discrete closure tends to Eq. (1) evaluated with exact (spectral) derivatives, with O(h^2)
    error: refining the grid 2x divides the error of each term by ~4 (signs and coefficients pinned)."""
    db, alpha = 40.0, 3.0
    a = alpha * db / 2
    errs = []
    for n in (64, 128):
        y, x = np.meshgrid(np.arange(n) * 2 * np.pi / n, np.arange(n) * 2 * np.pi / n, indexing="ij")
        I = np.exp(0.2 * np.cos(x) + 0.15 * np.sin(y + 0.4) + 0.1 * np.cos(x + 2 * y))
        T1, T2, T3 = _continuum_closure_terms(I, db)
        P1 = O.closure(I, a, alpha, order=1)
        P2 = O.closure(I, a, alpha, order=2, wkb1=False)
        P3 = O.closure(I, a, alpha, order=2, wkb1=True)
        if which == "order1":
            got, ref = P1 - I, -alpha * T1
        elif which == "wkb0":
            got, ref = P2 - P1, 0.5 * alpha ** 2 * T2
        else:
            got, ref = P3 - P2, -0.25 * alpha ** 2 * T3
        errs.append(np.max(np.abs(got - ref)) / np.max(np.abs(ref)))
    assert errs[1] < 0.02
    assert 3.3 < errs[0] / errs[1] < 4.7


# ------------------------------------------------------------------ projection
def test_projection_against_scalar_root_finder():
    from scipy.optimize import brentq
    E = np.linspace(60.0, 140.0, 8)
    lines = O.derive_lines(6.5e-6, 10.0, E, np.exp(-0.5 * ((E - 100) / 20.0) ** 2), 200.0 * E / 100.0)
    T = RNG.uniform(0.05, 1.3, size=(5, 7))
    tau = O.project(T, lines)
    for idx in np.ndindex(T.shape):
        root = brentq(lambda t: float(np.sum(lines.f * np.exp(-lines.gamma * t))) - T[idx], -5.0, 50.0, xtol=1e-15)
        assert abs(tau[idx] - root) < 1e-12


def test_projection_invariants():
    E = np.array([70.0, 100.0, 130.0])
    lines = O.derive_lines(6.5e-6, 5.0, E, [0.2, 0.5, 0.3], [700.0, 1000.0, 1300.0])
    tau = RNG.uniform(-0.1, 2.0, size=(6, 6))
    Is = O.line_intensities(tau, lines)
    T = np.sum(Is, axis=0)
    tau2 = O.project(T, lines)
    assert np.max(np.abs(tau2 - tau)) < 1e-12                     # idempotent on the manifold
    off = [Is[s] * (1 + 0.05 * RNG.normal(size=tau.shape)) for s in range(3)]
    tau3 = O.project(np.sum(off, axis=0), lines)
    assert np.max(np.abs(np.sum(O.line_intensities(tau3, lines), axis=0) - np.sum(off, axis=0))) < 1e-13
    mono = O.derive_lines(6.5e-6, 5.0, [100.0], [1.0], [1000.0])
    assert np.max(np.abs(O.project(np.exp(-tau), mono) - tau)) < 1e-14
