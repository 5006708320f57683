"""fp64 CPU oracle for the fast Eikonal Phase Retrieval (EPR) hot path.

TEST INFRASTRUCTURE ONLY.  This module is a plain, slow, obviously-correct numpy
restatement of what the paper defines.  It shares no code with the CUDA path and must
never be imported by the product (`paper_2601_22793_b200/`); only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs may
import it.

Every function cites the PAPER.md passage (line, section / equation) it follows.  Where the
paper is silent the reading taken is the one listed in DESIGN.md ("Readings", R1..R16, which
restate SURVEY.md §8(c); R16 is the oversampled grid and R17 the x-dependent effective spectrum of SURVEY.md §8(f)).

Conventions: pixel units; arrays are `[row = y][col = x]`, x fastest
(PAPER.md:185-191 write `P_s(y0, x0)`); every index is periodic (R7).

Parity pins: every function below is pinned by `tests/test_oracle_operators.py`, `tests/test_oracle_loop.py`,
`tests/test_oracle_oversample.py` and `tests/test_oracle_profiles.py` against closed forms, invariants, brute force
from the definition or a library routine used in a different way (table in DESIGN.md §8; a mutation check of the pins is
described there).  The *readings* R1..R17 themselves (finite-difference scheme, weights, start, projection, oversampling
transfer, blockwise interpolation of an x-dependent spectrum) are "parity unpinned" against the paper's own (unavailable)
implementation: the paper prints no numeric intermediate or final value.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

HC_KEV_M = 1.2398419843e-9  # h*c in keV*m  (lambda = hc / E)


# --------------------------------------------------------------------------------------
# physical constants per spectral line
# --------------------------------------------------------------------------------------
@dataclass
class Lines:
    """Per-line scalars of the spectral discretisation (§4.3-4.4)."""

    n_bins: int
    energy_keV: np.ndarray
    k: np.ndarray        # wavenumber 2*pi/lambda, 1/m
    alpha: np.ndarray    # eps_s / p^2 = L/(k_s p^2), dimensionless
    db: np.ndarray       # delta_s / beta_s
    a: np.ndarray        # alpha_s * db_s / 2  (Paganin length^2 in px^2)
    f: np.ndarray        # spectral fraction, sum = 1
    gamma: np.ndarray    # per-line attenuation scaling, sum f*gamma = 1      PAPER.md:227-229 (R11)

    @property
    def abar(self) -> float:
        """Weighted-mean Paganin coefficient used by the initial guess (R9)."""
        return float(np.sum(self.f * self.a))


def derive_lines(pixel_m, L_m, energy_keV, weight, delta_over_beta, mu_rel=None) -> Lines:
    """k_s = 2 pi E_s/(hc); eps_s = L/k_s (Eq. (2), (S8) PAPER.md:349);
    in pixel units alpha_s = eps_s/p^2.  phi_s = (db_s/2) ln I_s (Eq. (6)
    PAPER.md:216) gives a_s = alpha_s db_s/2.  gamma_s (Eq. (7)) is not a plan
    argument; reading R11: mu_s ∝ 1/(E_s db_s), normalised so that sum_s f_s gamma_s = 1."""
    E = np.atleast_1d(np.asarray(energy_keV, dtype=np.float64))
    w = np.atleast_1d(np.asarray(weight, dtype=np.float64))
    db = np.atleast_1d(np.asarray(delta_over_beta, dtype=np.float64))
    n = E.size
    assert w.size == n and db.size == n
    k = 2.0 * np.pi * E / HC_KEV_M
    alpha = L_m / (k * pixel_m * pixel_m)
    a = alpha * db / 2.0
    f = w / w.sum()
    g = (1.0 / (E * db)) if mu_rel is None else np.asarray(mu_rel, dtype=np.float64)
    gamma = g / np.sum(f * g)
    return Lines(n, E, k, alpha, db, a, f, gamma)


# --------------------------------------------------------------------------------------
# periodic finite differences (R1-R3, R7); they act on the LAST TWO axes ([…][y][x]), so a stack of planes works too
# --------------------------------------------------------------------------------------
def _xp(g):  # g[y][x+1]
    return np.roll(g, -1, axis=-1)


def _xm(g):  # g[y][x-1]
    return np.roll(g, 1, axis=-1)


def _yp(g):  # g[y+1][x]
    return np.roll(g, -1, axis=-2)


def _ym(g):  # g[y-1][x]
    return np.roll(g, 1, axis=-2)


def d0x(g):
    return (_xp(g) - _xm(g)) / 2.0


def d0y(g):
    return (_yp(g) - _ym(g)) / 2.0


def d2x(g):
    return _xp(g) - 2.0 * g + _xm(g)


def d2y(g):
    return _yp(g) - 2.0 * g + _ym(g)


def lap5(g):
    return d2x(g) + d2y(g)


# --------------------------------------------------------------------------------------
# a1-L  local O(L^2) closure, Eq. (1)
# --------------------------------------------------------------------------------------
def wkb1_term(I, alpha):
    """The diffraction-pressure (WKB1) term of Eq. (1), (eps²/4) ∂i(I ∂iQ) with Q = ∇²√I/√I
    (Eq. (S15)): flux form on the 5-point stencils (R3), coefficient alpha²/4 in pixel units.
    Eq. (1) SUBTRACTS it from the prediction."""
    I = np.asarray(I, dtype=np.float64)
    A = np.sqrt(I)
    Q = lap5(A) / A
    Fx = 0.5 * (_xp(I) + I) * (_xp(Q) - Q)   # flux through the face x+1/2
    Fy = 0.5 * (_yp(I) + I) * (_yp(Q) - Q)   # flux through the face y+1/2
    return 0.25 * alpha * alpha * ((Fx - _xm(Fx)) + (Fy - _ym(Fy)))


def closure(I, a, alpha, order=2, wkb1=True):
    """P = I − eps ∂i(I ∂iφ) + (eps²/2) ∂i∂j(I ∂iφ ∂jφ) − (eps²/4) ∂i(I ∂iQ)   Eq. (1) PAPER.md:146.

    With Eq. (6) I ∂φ = (db/2) ∂I, so the O(L) term is −a ∇²I (R1, 5-point).
    WKB0 O(L²): g = D⁰ ln I, S_ij = I g_i g_j, coefficient a²/2 (R2).
    WKB1: Q = ∇²√I/√I (Eq. (S15)), flux form, coefficient alpha²/4 (R3).
    `order=1` is the L¹ truncation."""
    I = np.asarray(I, dtype=np.float64)
    P = I - a * lap5(I)
    if order == 2:
        lnI = np.log(I)
        gx = d0x(lnI)
        gy = d0y(lnI)
        Sxx = I * gx * gx
        Syy = I * gy * gy
        Sxy = I * gx * gy
        P = P + 0.5 * a * a * (d2x(Sxx) + d2y(Syy) + 2.0 * d0x(d0y(Sxy)))
        if wkb1:
            P = P - wkb1_term(I, alpha)
    return P


# --------------------------------------------------------------------------------------
# a1-N  eikonal ray map, Eq. (2), and splat
# --------------------------------------------------------------------------------------
def ray_map(I, a, S):
    """u_s = Δ_s/p = (eps_s/p²) ∇φ_s with φ_s = (db_s/2) ln I_s  →  u = a · D⁰ ln I
    (Eq. (2), Eq. (6)), each component clamped
    to [−S, S] (R6)."""
    lnI = np.log(np.asarray(I, dtype=np.float64))
    ux = np.clip(a * d0x(lnI), -S, S)
    uy = np.clip(a * d0y(lnI), -S, S)
    return ux, uy


def _bilinear_targets(ux, uy):
    """x_t = x + u_x, y_t = y + u_y; x0 = ⌊x_t⌋, y0 = ⌊y_t⌋, d = x_t − x0; the four weights of
    PAPER.md:177-181.  Indices wrap (R7)."""
    ny, nx = ux.shape
    Y, X = np.meshgrid(np.arange(ny, dtype=np.float64), np.arange(nx, dtype=np.float64), indexing="ij")
    xt = X + ux
    yt = Y + uy
    x0f = np.floor(xt)
    y0f = np.floor(yt)
    dx = xt - x0f
    dy = yt - y0f
    x0 = np.mod(x0f.astype(np.int64), nx)
    y0 = np.mod(y0f.astype(np.int64), ny)
    x1 = np.mod(x0 + 1, nx)
    y1 = np.mod(y0 + 1, ny)
    w00 = (1.0 - dx) * (1.0 - dy)
    w10 = dx * (1.0 - dy)
    w01 = (1.0 - dx) * dy
    w11 = dx * dy
    return (y0, y1, x0, x1), (w00, w10, w01, w11)


def splat(I, ux, uy):
    """Mass-conserving bilinear redistribution ℳ_s (Eq. (3), discrete form
    PAPER.md:175-191):  P(y0,x0) += I w00;  P(y0,x0+1) += I w10;  P(y0+1,x0) += I w01;
    P(y0+1,x0+1) += I w11."""
    I = np.asarray(I, dtype=np.float64)
    ny, nx = I.shape
    (y0, y1, x0, x1), (w00, w10, w01, w11) = _bilinear_targets(ux, uy)
    P = np.zeros(ny * nx, dtype=np.float64)
    for yy, xx, w in ((y0, x0, w00), (y0, x1, w10), (y1, x0, w01), (y1, x1, w11)):
        P += np.bincount((yy * nx + xx).ravel(), weights=(I * w).ravel(), minlength=ny * nx)
    return P.reshape(ny, nx)


def gather(e, ux, uy):
    """Adjoint ℳ*_s, Eq. (4) PAPER.md:197-203:
    (ℳ* e)(x,y) = w00 e(y0,x0) + w10 e(y0,x0+1) + w01 e(y0+1,x0) + w11 e(y0+1,x0+1)."""
    e = np.asarray(e, dtype=np.float64)
    (y0, y1, x0, x1), (w00, w10, w01, w11) = _bilinear_targets(ux, uy)
    return w00 * e[y0, x0] + w10 * e[y0, x1] + w01 * e[y1, x0] + w11 * e[y1, x1]


# --------------------------------------------------------------------------------------
# a4  FFT-diagonal Paganin-type preconditioner
# --------------------------------------------------------------------------------------
def symbol_lambda(ny, nx, symbol=0):
    """λ(θ): Fourier symbol of −∇² on the pixel grid.  symbol=0: discrete 5-point
    (2−2cosθx)+(2−2cosθy) (default, R5: makes P⁻¹₁ the exact inverse of the R1 O(L) operator);
    symbol=1: continuous θx²+θy² (textbook Paganin filter)."""
    thx = 2.0 * np.pi * np.fft.fftfreq(nx)
    thy = 2.0 * np.pi * np.fft.fftfreq(ny)
    if symbol == 0:
        lx = 2.0 - 2.0 * np.cos(thx)
        ly = 2.0 - 2.0 * np.cos(thy)
    else:
        lx = thx * thx
        ly = thy * thy
    return ly[:, None] + lx[None, :]


def precondition(r, a, symbol=0):
    """q = IFFT2( FFT2(r) / (1 + a λ) ): the FFT-diagonal inverse of the linearised O(L)
    per-line operator I ↦ I − a∇²I ("Paganin-type filter")."""
    r = np.asarray(r, dtype=np.float64)
    H = 1.0 / (1.0 + a * symbol_lambda(r.shape[0], r.shape[1], symbol))
    return np.real(np.fft.ifft2(np.fft.fft2(r) * H))


# --------------------------------------------------------------------------------------
# a6  projection to the single-thickness manifold, Eq. (7) PAPER.md:227, PAPER.md:233 (R10)
# --------------------------------------------------------------------------------------
def line_intensities(tau, lines: Lines):
    """I_s = f_s exp(−γ_s τ)   Eq. (7) PAPER.md:227."""
    tau = np.asarray(tau, dtype=np.float64)
    return [lines.f[s] * np.exp(-lines.gamma[s] * tau) for s in range(lines.n_bins)]


def project(T, lines: Lines, tol=1e-14, max_iter=200):
    """Solve Σ_s f_s exp(−γ_s τ) = T per pixel (R10: the projection keeps the total object-plane
    intensity).  Newton from τ0 = −ln(T/Σf)/γ̄, γ̄ = Σ f γ / Σ f; monotone by convexity."""
    T = np.asarray(T, dtype=np.float64)
    f, g = lines.f, lines.gamma
    gbar = np.sum(f * g) / np.sum(f)
    tau = -np.log(T / np.sum(f)) / gbar
    if lines.n_bins == 1:
        return -np.log(T / f[0]) / g[0]
    for _ in range(max_iter):
        F = -T.copy()
        dF = np.zeros_like(T)
        for s in range(lines.n_bins):
            E = f[s] * np.exp(-g[s] * tau)
            F += E
            dF -= g[s] * E
        step = F / dF
        tau = tau - step
        if np.max(np.abs(step)) < tol:
            break
    return tau


# --------------------------------------------------------------------------------------
# forward model  τ → Σ_s F_s[I_s]   Eq. (5)
# --------------------------------------------------------------------------------------
def forward(tau, lines: Lines, solver="local", order=2, wkb1=True, S=16.0, nonlocal_wkb1=False):
    """I_det ≈ Σ_s F_s[I_s], F_s ∈ {P_{m,s}, ℳ_s} (Eq. (5)) with
    I_s = f_s e^{−γ_s τ} (Eq. (7)).  Returns (P_sum, [P_s], [(ux_s, uy_s)] or None).
    nonlocal_wkb1 (variant of reading R4, off by default): the ray map carries the WKB0 transport to all orders; the
    leading wave-optics correction of Eq. (1), −(eps²/4) ∂i(I ∂iQ), is added to it as the same LOCAL term
    ("when complemented by the second-order corrections")."""
    Is = line_intensities(tau, lines)
    P_bins, maps = [], []
    for s in range(lines.n_bins):
        if solver == "local":
            P_bins.append(closure(Is[s], lines.a[s], lines.alpha[s], order=order, wkb1=wkb1))
        else:
            ux, uy = ray_map(Is[s], lines.a[s], S)
            maps.append((ux, uy))
            P_s = splat(Is[s], ux, uy)
            if nonlocal_wkb1:
                P_s = P_s - wkb1_term(Is[s], lines.alpha[s])
            P_bins.append(P_s)
    P = np.sum(P_bins, axis=0)
    return P, P_bins, (maps if solver != "local" else None)


def split_weights(P_bins, lines: Lines):
    """"positivity-weighted weights", reading R8: w_s = P_s⁺ / Σ_t P_t⁺,
    falling back to f_s where the denominator is not positive."""
    Pp = [np.maximum(P, 0.0) for P in P_bins]
    den = np.sum(Pp, axis=0)
    ok = den > 0.0
    safe = np.where(ok, den, 1.0)
    return [np.where(ok, Pp[s] / safe, lines.f[s]) for s in range(lines.n_bins)]


# --------------------------------------------------------------------------------------
# the iteration
# --------------------------------------------------------------------------------------
def paganin_init(d, lines: Lines, symbol=0, i_min=1e-6):
    """Initial guess (R9): one linear Paganin solve with the weighted-mean coefficient ā,
    floored at i_min, projected onto the manifold Eq. (7).  `iterations = 0` returns this —
    the L¹ / Paganin result of PAPER.md:124."""
    T0 = precondition(d, lines.abar, symbol)
    T0 = np.maximum(T0, i_min)
    return project(T0, lines)


def max_shift(tau, lines: Lines):
    """Regime indicator of PAPER.md:53-55 in the sup norm: the largest component of the eikonal shift
    u_s = a_s D⁰ ln I_s (Eq. (2), Eq. (6)) over pixels and lines, in pixels, NOT clamped
    (η(r) = ‖Δ(r)‖/p is its Euclidean version: η_sup ≤ η ≤ √2 η_sup)."""
    Is = line_intensities(tau, lines)
    m = 0.0
    for s in range(lines.n_bins):
        ux, uy = ray_map(Is[s], lines.a[s], np.inf)
        m = max(m, float(np.max(np.abs(ux))), float(np.max(np.abs(uy))))
    return m


def retrieve(d, lines: Lines, solver="local", iterations=10, step=1.0, order=2, wkb1=True,
             symbol=0, S=16.0, i_min=1e-6, tau0=None, history=None, shift_history=None, nonlocal_wkb1=False):
    """The batched per-projection correction loop for one projection:
    per-line predictions and their sum, detector residual, positivity-weighted split, transport
    back (identity | adjoint Eq. (4)), per-line FFT-diagonal preconditioner update, projection
    to the single-thickness manifold.  Returns τ."""
    d = np.asarray(d, dtype=np.float64)
    tau = paganin_init(d, lines, symbol, i_min) if tau0 is None else np.asarray(tau0, np.float64).copy()
    n = lines.n_bins
    for _ in range(iterations):
        Is = line_intensities(tau, lines)
        P, P_bins, maps = forward(tau, lines, solver, order, wkb1, S, nonlocal_wkb1)
        e = d - P
        if history is not None:
            history.append(float(np.sqrt(np.mean(e * e))))
        if shift_history is not None:
            shift_history.append(max_shift(tau, lines))
        w = split_weights(P_bins, lines)
        for s in range(n):
            r = w[s] * e
            if solver != "local":
                r = gather(r, maps[s][0], maps[s][1])
            Is[s] = Is[s] + step * precondition(r, lines.a[s], symbol)
        if n > 1:
            T = np.maximum(np.sum(Is, axis=0), i_min)
            tau = project(T, lines)
        else:
            I1 = np.maximum(Is[0], i_min)
            tau = -np.log(I1 / lines.f[0]) / lines.gamma[0]
    return tau


def phase(tau, lines: Lines, s=0):
    """φ_s = (db_s/2) ln(I_s/f_s) = −(db_s/2) γ_s τ   Eq. (6) PAPER.md:216 with Eq. (7)."""
    return -(lines.db[s] / 2.0) * lines.gamma[s] * np.asarray(tau, dtype=np.float64)


# --------------------------------------------------------------------------------------
# oversampled computational grid (reading R16)
# --------------------------------------------------------------------------------------
def upsample(d, m):
    """Detector image on the grid refined m times ("a pixel size reduced by a factor 2").
    The paper does not say how the data reach the fine grid; reading R16: each detector pixel measures the mean
    intensity over its area, so the fine image is constant over it — pixel replication."""
    d = np.asarray(d, dtype=np.float64)
    return np.repeat(np.repeat(d, m, axis=0), m, axis=1)


def downsample(t, m):
    """Back to the detector grid: mean over each m x m block of fine pixels (R16), the exact left inverse of
    `upsample` and mean-preserving."""
    t = np.asarray(t, dtype=np.float64)
    ny, nx = t.shape
    return t.reshape(ny // m, m, nx // m, m).mean(axis=(1, 3))


def retrieve_oversampled(d, lines_fine: Lines, m, solver="local", iterations=10, step=1.0, order=2, wkb1=True,
                         symbol=0, S=16.0, i_min=1e-6):
    """The correction loop on the m-times oversampled grid (factor 2 for the local solver, 4 for the
    non-local one): up-sample d, run `retrieve` with the per-line scalars of the FINE pixel (`lines_fine` =
    derive_lines(pixel/m, ...), so that shifts are counted in fine pixels; S is in fine pixels too),
    down-sample τ.  m = 1 is `retrieve`."""
    tau = retrieve(upsample(d, m), lines_fine, solver, iterations, step, order, wkb1, symbol, S, i_min)
    return downsample(tau, m)


# --------------------------------------------------------------------------------------
# x-dependent effective spectrum (Eq. (6) + remark, 227-229 Eq. (7), 431-441 §9.2;
# SURVEY.md §8(f) rank 2; reading R17)
# --------------------------------------------------------------------------------------
# The paper parameterises I_s(r) = f_s(x) exp(−γ_s(x) τ(r)) and φ_s = (db_s(x)/2) ln I_s with 1-D profiles in the
# horizontal detector coordinate x ("slow spatial variations of the effective spectrum", §9.2), and promises the
# "file format and the blockwise interpolation strategy" in a Supporting Information that PAPER.md does not contain
# (PAPER.md:221).  Reading R17:
#   (a) the profiles are given on n_blocks equal blocks of columns; the value of column x is the LINEAR interpolation
#       between the two nearest block centres, constant outside the outermost centres; one block = uniform spectrum
#       (§9.2 "single block");
#   (b) the variation is slow, so the per-line scalars are FROZEN at the pixel's own column: every stencil of the local
#       closure sees the neighbouring τ through the scalars of the centre column (no derivative of f_s, γ_s, db_s is
#       ever taken — the empty beam must stay d = 1), and a source pixel of the ray map carries the mass and the shift
#       of its own column's scalars;
#   (c) the FFT-diagonal preconditioner cannot have an x-dependent coefficient; it is applied once per block with that
#       block's a_s and the results are blended with the interpolation weights of (a): "blockwise interpolation".
@dataclass
class Profiles:
    n_bins: int
    n_blocks: int
    nx: int
    alpha: np.ndarray     # [n_bins]            L/(k_s p²): the lines keep their energies
    wblk: np.ndarray      # [n_blocks][nx]      interpolation weights of (a); Σ_b wblk[b][x] = 1
    f_blk: np.ndarray     # [n_blocks][n_bins]  per-block scalars
    gamma_blk: np.ndarray
    a_blk: np.ndarray
    abar_blk: np.ndarray  # [n_blocks]          Σ_s f_s a_s per block (initial guess, R9)
    f: np.ndarray         # [n_bins][nx]        per-column scalars
    gamma: np.ndarray
    db: np.ndarray
    a: np.ndarray

    def column(self, x) -> Lines:
        """The uniform-spectrum scalars of column x, as a `Lines`."""
        return Lines(self.n_bins, None, None, self.alpha, self.db[:, x], self.a[:, x], self.f[:, x], self.gamma[:, x])


def block_weights(nx, n_blocks):
    """(a): block b covers columns [b nx/n_blocks, (b+1) nx/n_blocks) (nx divisible by n_blocks), centre
    c_b = (b + ½) nx/n_blocks − ½ in pixel-centre coordinates; hat-function weights, clamped at both ends."""
    assert nx % n_blocks == 0
    wb = nx // n_blocks
    c = (np.arange(n_blocks) + 0.5) * wb - 0.5
    x = np.arange(nx, dtype=np.float64)
    w = np.zeros((n_blocks, nx))
    if n_blocks == 1:
        w[0] = 1.0
        return w
    t = np.clip((x - c[0]) / wb, 0.0, n_blocks - 1.0)       # position in units of blocks
    b0 = np.minimum(np.floor(t).astype(int), n_blocks - 2)
    fr = t - b0
    w[b0, np.arange(nx)] = 1.0 - fr
    w[b0 + 1, np.arange(nx)] += fr
    return w


def derive_profiles(pixel_m, L_m, energy_keV, nx, weight_blk, db_blk, mu_rel_blk=None) -> Profiles:
    """Per-block scalars like `derive_lines` (weight_blk, db_blk, mu_rel_blk: [n_blocks][n_bins]) and their per-column
    interpolation.  γ keeps ONE normalisation for the whole detector, so that τ is one thickness field: with
    g_s^{(b)} = 1/(E_s db_s^{(b)}) (R11) or mu_rel, γ_s^{(b)} = g_s^{(b)}/G, G = mean_b Σ_s f_s^{(b)} g_s^{(b)};
    uniform profiles reduce to R11."""
    E = np.atleast_1d(np.asarray(energy_keV, dtype=np.float64))
    wt = np.atleast_2d(np.asarray(weight_blk, dtype=np.float64))
    db = np.atleast_2d(np.asarray(db_blk, dtype=np.float64))
    nblk, n = wt.shape
    assert db.shape == (nblk, n) and E.size == n
    k = 2.0 * np.pi * E / HC_KEV_M
    alpha = L_m / (k * pixel_m * pixel_m)
    f_blk = wt / wt.sum(axis=1, keepdims=True)
    g = (1.0 / (E[None, :] * db)) if mu_rel_blk is None else np.atleast_2d(np.asarray(mu_rel_blk, dtype=np.float64))
    G = np.mean(np.sum(f_blk * g, axis=1))
    gamma_blk = g / G
    a_blk = alpha[None, :] * db / 2.0
    w = block_weights(nx, nblk)
    col = lambda v: np.einsum("bx,bs->sx", w, v)            # noqa: E731  Σ_b wblk[b][x] v[b][s]
    dbx = col(db)
    return Profiles(n, nblk, nx, alpha, w, f_blk, gamma_blk, a_blk, np.sum(f_blk * a_blk, axis=1),
                    col(f_blk), col(gamma_blk), dbx, alpha[:, None] * dbx / 2.0)


def line_intensities_x(tau, prof: Profiles):
    """I_s = f_s(x) exp(−γ_s(x) τ)   Eq. (7) PAPER.md:227 with the x-dependent profiles."""
    tau = np.asarray(tau, dtype=np.float64)
    return [prof.f[s][None, :] * np.exp(-prof.gamma[s][None, :] * tau) for s in range(prof.n_bins)]


def closure_x(tau, prof: Profiles, s, order=2, wkb1=True):
    """(b): P_s(y, x) = closure(f_s(x) e^{−γ_s(x) τ}; a_s(x), α_s) evaluated AT column x — the Eq. (1) closure of the
    uniform case with the scalars of the centre column.  The stencil has radius 2, so for every column a strip of the
    five columns x−2 … x+2 (periodic, R7) is enough; the strips are stacked as [x][y][k] and the centre k = 2 is kept."""
    tau = np.asarray(tau, dtype=np.float64)
    strips = np.stack([np.roll(tau, -k, axis=1) for k in (-2, -1, 0, 1, 2)], axis=-1)      # [y][x][k] = τ[y][x+k]
    strips = np.transpose(strips, (1, 0, 2))                                                # [x][y][k]
    I = prof.f[s][:, None, None] * np.exp(-prof.gamma[s][:, None, None] * strips)
    P = closure(I, prof.a[s][:, None, None], prof.alpha[s], order=order, wkb1=wkb1)
    return P[:, :, 2].T


def ray_map_x(tau, prof: Profiles, s, S):
    """(b): u_s = a_s(x) D⁰ ln I_s with the scalars of the source's own column frozen, i.e. D⁰ ln I_s = −γ_s(x) D⁰τ
    (Eq. (2) PAPER.md:164-167 with Eq. (6), (7)); each component clamped to ±S (R6)."""
    tau = np.asarray(tau, dtype=np.float64)
    c = (prof.a[s] * prof.gamma[s])[None, :]
    return np.clip(-c * d0x(tau), -S, S), np.clip(-c * d0y(tau), -S, S)


def wkb1_term_x(tau, prof: Profiles, s):
    """(b): the WKB1 term of Eq. (1) PAPER.md:146 (`wkb1_term`, R3) evaluated AT column x on I = f_s(x) e^{−γ_s(x) τ} with
    the scalars of the centre column, on the same five-column strips as `closure_x` (the term has radius 2)."""
    tau = np.asarray(tau, dtype=np.float64)
    strips = np.stack([np.roll(tau, -k, axis=1) for k in (-2, -1, 0, 1, 2)], axis=-1)      # [y][x][k] = τ[y][x+k]
    strips = np.transpose(strips, (1, 0, 2))                                                # [x][y][k]
    I = prof.f[s][:, None, None] * np.exp(-prof.gamma[s][:, None, None] * strips)
    return wkb1_term(I, prof.alpha[s])[:, :, 2].T


def forward_x(tau, prof: Profiles, solver="local", order=2, wkb1=True, S=16.0, nonlocal_wkb1=False):
    """Eq. (5) PAPER.md:209-212 with the x-dependent spectrum: returns (P_sum, [P_s], [(ux_s, uy_s)] or None).
    nonlocal_wkb1: the variant of reading R4 (see `forward`), the local term taken at the detector pixel's column."""
    Is = line_intensities_x(tau, prof)
    P_bins, maps = [], []
    for s in range(prof.n_bins):
        if solver == "local":
            P_bins.append(closure_x(tau, prof, s, order=order, wkb1=wkb1))
        else:
            ux, uy = ray_map_x(tau, prof, s, S)
            maps.append((ux, uy))
            P_s = splat(Is[s], ux, uy)
            if nonlocal_wkb1:
                P_s = P_s - wkb1_term_x(tau, prof, s)
            P_bins.append(P_s)
    return np.sum(P_bins, axis=0), P_bins, (maps if solver != "local" else None)


def max_shift_x(tau, prof: Profiles):
    """`max_shift` with the x-dependent spectrum: the largest component of the unclamped shift of `ray_map_x` over pixels
    and lines (regime indicator of PAPER.md:53-55 in the sup norm)."""
    m = 0.0
    for s in range(prof.n_bins):
        ux, uy = ray_map_x(tau, prof, s, np.inf)
        m = max(m, float(np.max(np.abs(ux))), float(np.max(np.abs(uy))))
    return m


def split_weights_x(P_bins, prof: Profiles):
    """R8 with the fallback f_s(x) of the detector pixel's column."""
    Pp = [np.maximum(P, 0.0) for P in P_bins]
    den = np.sum(Pp, axis=0)
    ok = den > 0.0
    safe = np.where(ok, den, 1.0)
    return [np.where(ok, Pp[s] / safe, prof.f[s][None, :]) for s in range(prof.n_bins)]


def precondition_x(r, a_blk, wblk, symbol=0):
    """(c) blockwise interpolation of the FFT-diagonal inverse: q = Σ_b wblk[b][x] ·
    IFFT2(FFT2(r)/(1 + a^{(b)} λ)); a_blk: [n_blocks] coefficients of ONE line (or the ā of the initial guess)."""
    r = np.asarray(r, dtype=np.float64)
    q = np.zeros_like(r)
    for b in range(len(a_blk)):
        q += wblk[b][None, :] * precondition(r, a_blk[b], symbol)
    return q


def project_x(T, prof: Profiles, tol=1e-14, max_iter=200):
    """Solve Σ_s f_s(x) exp(−γ_s(x) τ) = T per pixel (R10 with the column's scalars); Newton as in `project`."""
    T = np.asarray(T, dtype=np.float64)
    f = prof.f[:, None, :]
    g = prof.gamma[:, None, :]
    if prof.n_bins == 1:
        return -np.log(T / f[0]) / g[0]
    gbar = np.sum(f * g, axis=0) / np.sum(f, axis=0)
    tau = -np.log(T / np.sum(f, axis=0)) / gbar
    for _ in range(max_iter):
        Es = f * np.exp(-g * tau[None])
        step = (np.sum(Es, axis=0) - T) / (-np.sum(g * Es, axis=0))
        tau = tau - step
        if np.max(np.abs(step)) < tol:
            break
    return tau


def paganin_init_x(d, prof: Profiles, symbol=0, i_min=1e-6):
    """R9 with (c): the linear Paganin solve with the weighted-mean coefficient ā^{(b)} of every block, blended."""
    T0 = np.maximum(precondition_x(d, prof.abar_blk, prof.wblk, symbol), i_min)
    return project_x(T0, prof)


def retrieve_x(d, prof: Profiles, solver="local", iterations=10, step=1.0, order=2, wkb1=True, symbol=0, S=16.0,
               i_min=1e-6, tau0=None, history=None, shift_history=None, nonlocal_wkb1=False):
    """The correction loop of PAPER.md:231-233 with the x-dependent effective spectrum of Eq. (6)/(7) (reading R17):
    the same steps as `retrieve`, every per-line scalar taken at the pixel's column, the filter blockwise."""
    d = np.asarray(d, dtype=np.float64)
    tau = paganin_init_x(d, prof, symbol, i_min) if tau0 is None else np.asarray(tau0, np.float64).copy()
    n = prof.n_bins
    for _ in range(iterations):
        Is = line_intensities_x(tau, prof)
        P, P_bins, maps = forward_x(tau, prof, solver, order, wkb1, S, nonlocal_wkb1)
        e = d - P
        if history is not None:
            history.append(float(np.sqrt(np.mean(e * e))))
        if shift_history is not None:
            shift_history.append(max_shift_x(tau, prof))
        w = split_weights_x(P_bins, prof)
        for s in range(n):
            r = w[s] * e
            if solver != "local":
                r = gather(r, maps[s][0], maps[s][1])
            Is[s] = Is[s] + step * precondition_x(r, prof.a_blk[:, s], prof.wblk, symbol)
        T = np.maximum(np.sum(Is, axis=0), i_min)
        tau = project_x(T, prof)
    return tau


# --------------------------------------------------------------------------------------
# regime diagnostic: per-line distribution of the eikonal shift (Fig. 6)
# --------------------------------------------------------------------------------------
def shift_histogram(tau, lines: Lines, n_hist, bin_px):
    """"the distribution of estimated WKB0 transverse shifts (in detector-pixel units) for each sampling energy (spectral
    line) on a representative radiograph": for every line the histogram of η(r) = ‖Δ_s(r)‖/p =
    ‖a_s D⁰ ln I_s‖ (Eq. (2), Euclidean norm, NOT clamped) over the pixels, bins [k·bin_px, (k+1)·bin_px),
    the last bin open-ended.  Returns integer counts [n_bins][n_hist] (each row sums to the number of pixels)."""
    Is = line_intensities(tau, lines)
    out = np.zeros((lines.n_bins, n_hist), dtype=np.int64)
    for s in range(lines.n_bins):
        ux, uy = ray_map(Is[s], lines.a[s], np.inf)
        eta = np.sqrt(ux * ux + uy * uy)
        k = np.minimum(np.floor(eta / bin_px).astype(np.int64), n_hist - 1)
        out[s] = np.bincount(k.ravel(), minlength=n_hist)
    return out
