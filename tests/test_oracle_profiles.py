"""Pins for the oracle's x-dependent effective spectrum (Eq. (6), 227-229 Eq. (7), 431-441 §9.2; reading
R17 of DESIGN.md): hand-computed interpolation weights, reduction to the uniform spectrum ("single block"), brute force
from the definition for the frozen-coefficient closure and transport, closed forms for the blockwise filter and for one
whole iteration.  CPU only."""
import numpy as np
import pytest

from oracle import epr_oracle as O

E3 = np.array([70.0, 100.0, 130.0])
W3 = np.array([0.3, 0.45, 0.25])
DB3 = np.array([600.0, 1000.0, 1500.0])


def _smooth(ny, nx, seed):
    rng = np.random.default_rng(seed)
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    f = np.zeros((ny, nx))
    for _ in range(5):
        m, n = rng.integers(-2, 3, size=2)
        f += rng.normal() * np.cos(m * x + n * y + rng.uniform(0, 2 * np.pi))
    return f / np.max(np.abs(f))


def _varying(nx, n_blocks, L=3.0, mu=False):
    """Profiles whose weights, δ/β and (optionally) attenuation scaling all differ from block to block."""
    t = np.linspace(0.0, 1.0, n_blocks)[:, None]
    wt = W3[None, :] * (1.0 + t * np.array([0.8, 0.0, -0.6])[None, :])
    db = DB3[None, :] * (1.0 + 0.3 * t)
    mu_rel = None if not mu else (np.array([3.0, 1.0, 0.4])[None, :] * (1.0 + 0.2 * t))
    return O.derive_profiles(6.5e-6, L, E3, nx, wt, db, mu_rel), wt, db


def test_block_weights_hand_computed():
    """R17(a): 15 columns in 3 blocks of 5 → centres at columns 2, 7, 12; linear in between, constant outside."""
    w = O.block_weights(15, 3)
    want0 = [1, 1, 1, 0.8, 0.6, 0.4, 0.2, 0, 0, 0, 0, 0, 0, 0, 0]
    want1 = [0, 0, 0, 0.2, 0.4, 0.6, 0.8, 1, 0.8, 0.6, 0.4, 0.2, 0, 0, 0]
    want2 = [0, 0, 0, 0, 0, 0, 0, 0, 0.2, 0.4, 0.6, 0.8, 1, 1, 1]
    assert np.allclose(w, [want0, want1, want2], atol=1e-15)
    # even block width: centres fall between columns (8 columns, 2 blocks: centres 1.5 and 5.5)
    w = O.block_weights(8, 2)
    assert np.allclose(w[1], [0, 0, 0.125, 0.375, 0.625, 0.875, 1, 1], atol=1e-15) and np.allclose(w.sum(0), 1.0)
    assert np.array_equal(O.block_weights(6, 1), np.ones((1, 6)))


def test_derive_profiles_scalars():
    """Per-column scalars: a_s(x) = (L/(k_s p²)) db_s(x)/2 retyped from the physical constants, Σ_s f_s(x) = 1 in every
    column, one global γ normalisation; uniform profiles reduce to derive_lines (R11: Σ f γ = 1)."""
    prof, wt, db = _varying(20, 4)
    x = 7                                                    # between the centres of blocks 1 and 2 (2, 7, 12, 17)
    assert np.allclose(prof.wblk[:, x], [0, 1, 0, 0])
    k = 2 * np.pi * E3 / 1.2398419843e-9
    assert np.allclose(prof.a[:, x], 3.0 / (k * 6.5e-6 ** 2) * db[1] / 2.0, rtol=1e-14)
    x = 9                                                    # 0.6 of block 1, 0.4 of block 2
    assert np.allclose(prof.db[:, x], 0.6 * db[1] + 0.4 * db[2], rtol=1e-14)
    fb = wt / wt.sum(1, keepdims=True)
    assert np.allclose(prof.f[:, x], 0.6 * fb[1] + 0.4 * fb[2], rtol=1e-14)
    assert np.allclose(prof.f.sum(0), 1.0, atol=1e-15)
    g = 1.0 / (E3[None, :] * db)
    G = np.mean(np.sum(fb * g, axis=1))
    assert np.allclose(prof.gamma_blk, g / G, rtol=1e-14)
    uni = O.derive_profiles(6.5e-6, 3.0, E3, 12, [W3] * 3, [DB3] * 3)
    lines = O.derive_lines(6.5e-6, 3.0, E3, W3, DB3)
    for s in range(3):
        assert np.allclose(uni.f[s], lines.f[s], rtol=1e-15) and np.allclose(uni.gamma[s], lines.gamma[s], rtol=1e-15)
        assert np.allclose(uni.a[s], lines.a[s], rtol=1e-15)
    assert np.allclose(uni.abar_blk, lines.abar, rtol=1e-15)


@pytest.mark.parametrize("n_blocks", [1, 2, 4])
@pytest.mark.parametrize("solver,step", [("local", 1.0), ("nonlocal", 0.4)])
def test_uniform_profiles_reduce_to_uniform_spectrum(n_blocks, solver, step):
    """§9.2: "If such variations are negligible, the model reduces to a spatially uniform spectrum (single
    block)".  Identical blocks, any number of them, give the uniform-spectrum retrieval."""
    ny, nx, L = 24, 32, 20.0 if solver == "nonlocal" else 2.0
    prof = O.derive_profiles(6.5e-6, L, E3, nx, [W3] * n_blocks, [DB3] * n_blocks)
    lines = O.derive_lines(6.5e-6, L, E3, W3, DB3)
    d = 1.0 + 0.1 * _smooth(ny, nx, 3)
    t_x = O.retrieve_x(d, prof, solver, 3, step, S=8.0)
    t_u = O.retrieve(d, lines, solver, 3, step, S=8.0)
    assert np.max(np.abs(t_x - t_u)) < 1e-13
    if n_blocks == 1:
        assert np.max(np.abs(t_x - t_u)) < 2e-15             # the same arithmetic up to the last bits


def test_closure_x_brute_force_per_column():
    """R17(b) written out: column x of P_s is column x of the uniform-spectrum closure evaluated on the WHOLE plane
    with the scalars of column x."""
    ny, nx = 12, 20
    prof, _, _ = _varying(nx, 4, L=1.0)
    tau = 0.3 * (1.0 + 0.5 * _smooth(ny, nx, 5))
    for s in range(3):
        for order, wkb1 in ((2, True), (1, False)):
            got = O.closure_x(tau, prof, s, order=order, wkb1=wkb1)
            for x in range(nx):
                I = prof.f[s, x] * np.exp(-prof.gamma[s, x] * tau)
                want = O.closure(I, prof.a[s, x], prof.alpha[s], order=order, wkb1=wkb1)[:, x]
                assert np.max(np.abs(got[:, x] - want)) < 1e-13 * np.max(np.abs(want))


def test_empty_beam_stays_empty():
    """No derivative of the profiles is ever taken: τ = 0 predicts Σ_s f_s(x) = 1 in both solvers, whatever the
    profiles, and the retrieval of d = 1 is τ = 0."""
    prof, _, _ = _varying(20, 4, L=30.0, mu=True)
    z = np.zeros((8, 20))
    for solver in ("local", "nonlocal"):
        P, _, _ = O.forward_x(z, prof, solver)
        assert np.max(np.abs(P - 1.0)) < 1e-14
        assert np.max(np.abs(O.retrieve_x(np.ones((8, 20)), prof, solver, 2, 0.7))) < 1e-13


def test_nonlocal_forward_x_brute_force():
    """R17(b) for the ray map, from the definition PAPER.md:175-191 in plain Python loops: a source pixel carries the
    mass f_s(x) e^{−γ_s(x) τ} and the shift −a_s(x) γ_s(x) D⁰τ of ITS OWN column, clamped to ±S; targets wrap (R7)."""
    ny, nx, S = 6, 10, 2.5
    prof, _, _ = _varying(nx, 2, L=400.0)
    tau = 0.2 * (1.0 + 0.5 * _smooth(ny, nx, 8))
    _, P_bins, maps = O.forward_x(tau, prof, "nonlocal", S=S)
    clamped = False
    for s in range(3):
        want = np.zeros((ny, nx))
        for y in range(ny):
            for x in range(nx):
                c = prof.a[s, x] * prof.gamma[s, x]
                ux = -c * (tau[y, (x + 1) % nx] - tau[y, (x - 1) % nx]) / 2.0
                uy = -c * (tau[(y + 1) % ny, x] - tau[(y - 1) % ny, x]) / 2.0
                clamped |= abs(ux) > S or abs(uy) > S
                ux, uy = min(max(ux, -S), S), min(max(uy, -S), S)
                m = prof.f[s, x] * np.exp(-prof.gamma[s, x] * tau[y, x])
                x0, y0 = int(np.floor(x + ux)), int(np.floor(y + uy))
                dx, dy = x + ux - x0, y + uy - y0
                for b, a, wgt in ((0, 0, (1 - dx) * (1 - dy)), (0, 1, dx * (1 - dy)), (1, 0, (1 - dx) * dy), (1, 1, dx * dy)):
                    want[(y0 + b) % ny, (x0 + a) % nx] += m * wgt
        assert np.max(np.abs(P_bins[s] - want)) < 1e-14
    assert clamped and max(np.abs(m[0]).max() for m in maps) > 1.0


def test_blockwise_filter_closed_form():
    """R17(c): a single Fourier mode comes back multiplied by Σ_b wblk[b][x]/(1 + a^{(b)} λ(θ)); at a block centre that
    is exactly the block's own Paganin gain."""
    ny, nx, my, mx = 12, 15, 2, 3
    w = O.block_weights(nx, 3)
    a_blk = np.array([5.0, 20.0, 80.0])
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    mode = np.cos(2 * np.pi * (mx * x / nx + my * y / ny) + 0.4)
    lam = (2 - 2 * np.cos(2 * np.pi * mx / nx)) + (2 - 2 * np.cos(2 * np.pi * my / ny))
    gain = np.sum(w / (1.0 + a_blk[:, None] * lam), axis=0)
    q = O.precondition_x(mode, a_blk, w)
    assert np.max(np.abs(q - mode * gain[None, :])) < 1e-14
    for b, c in enumerate((2, 7, 12)):
        assert abs(gain[c] - 1.0 / (1.0 + a_blk[b] * lam)) < 1e-15
    assert gain[4] != gain[2]


@pytest.mark.parametrize("solver", ["local", "nonlocal"])
def test_one_iteration_closed_form_with_block_dependent_filter(solver):
    """PAPER.md:231 with R17(c).  f and γ uniform, δ/β different in every block: from a constant τ⁰ = c all predictions
    are constant, w_s = I_s/T⁰, and for d = T⁰ + ε cos(θ·r) one iteration gives
        Σ_s I_s = T⁰ + step ε cos(θ·r) Σ_s w_s Σ_b wblk[b][x]/(1 + a_s^{(b)} λ(θ))
    — line s is filtered with ITS coefficient of EVERY block, blended by the interpolation weights."""
    ny, nx, my, mx, c, eps, step, nblk = 16, 24, 1, 2, 0.6, 1e-3, 0.7, 3
    db = DB3[None, :] * np.array([1.0, 1.5, 0.7])[:, None]
    g = 1.0 / (E3 * DB3)
    prof = O.derive_profiles(6.5e-6, 3.0, E3, nx, [W3] * nblk, db, mu_rel_blk=[g] * nblk)
    assert np.ptp(prof.gamma, axis=1).max() < 1e-15 and np.ptp(prof.a_blk, axis=0).min() > 1.0
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    mode = np.cos(2 * np.pi * (mx * x / nx + my * y / ny))
    lam = (2 - 2 * np.cos(2 * np.pi * mx / nx)) + (2 - 2 * np.cos(2 * np.pi * my / ny))
    I0 = prof.f[:, 0] * np.exp(-prof.gamma[:, 0] * c)
    T0 = I0.sum()
    tau = O.retrieve_x(T0 + eps * mode, prof, solver, iterations=1, step=step, tau0=np.full((ny, nx), c))
    got = np.sum(O.line_intensities_x(tau, prof), axis=0)
    gain = np.zeros(nx)
    for s in range(3):
        gain += (I0[s] / T0) * np.sum(prof.wblk / (1.0 + prof.a_blk[:, s][:, None] * lam), axis=0)
    assert np.max(np.abs(got - (T0 + step * eps * mode * gain[None, :]))) < 1e-12
    wrong = sum((I0[s] / T0) * np.sum(prof.wblk / (1.0 + prof.abar_blk[:, None] * lam), axis=0) for s in range(3))
    assert np.max(np.abs(wrong - gain)) * step * eps > 1e-7


def test_identity_filter_puts_data_on_the_manifold_column_by_column():
    """With a vanishing propagation distance the filter and both forward models are the identity, so one iteration with
    step 1 gives Σ_s f_s(x) e^{−γ_s(x) τ} = d pixel by pixel (the weights sum to one, the projection uses the scalars
    of the pixel's column), and the start (R9) is the same; checked per pixel with scipy's bracketing root finder."""
    from scipy.optimize import brentq
    ny, nx = 6, 20
    prof, _, _ = _varying(nx, 4, L=1e-12, mu=True)
    d = 0.8 + 0.15 * _smooth(ny, nx, 4)
    for tau in (O.paganin_init_x(d, prof), O.retrieve_x(d, prof, "local", 1, 1.0, tau0=np.full((ny, nx), 0.1)),
                O.retrieve_x(d, prof, "nonlocal", 1, 1.0, tau0=np.full((ny, nx), 0.1))):
        for y in range(0, ny, 2):
            for x in range(nx):
                root = brentq(lambda t: np.sum(prof.f[:, x] * np.exp(-prof.gamma[:, x] * t)) - d[y, x], -5.0, 50.0, xtol=1e-14)
                assert abs(tau[y, x] - root) < 1e-9                  # a_s ~ 1e-10 px² is not exactly zero


def test_split_fallback_uses_the_columns_fraction():
    prof, _, _ = _varying(8, 2)
    P = [np.array([[0.3, -0.2, -0.1, 0.0] * 2]), np.array([[0.1, 0.5, -0.3, 0.0] * 2]), np.array([[0.0, 0.5, -1.0, 0.0] * 2])]
    w = O.split_weights_x(P, prof)
    assert np.allclose([w[s][0, 0] for s in range(3)], [0.75, 0.25, 0.0], atol=1e-15)
    assert np.allclose([w[s][0, 1] for s in range(3)], [0.0, 0.5, 0.5], atol=1e-15)
    for x in (2, 3, 6, 7):
        assert np.allclose([w[s][0, x] for s in range(3)], prof.f[:, x], atol=1e-15)
    assert abs(prof.f[0, 2] - prof.f[0, 6]) > 0.01


def test_nonlocal_wkb1_x_brute_force_and_uniform_reduction():
    """Variant of R4 with the x-dependent spectrum: column x of the subtracted term is column x of the uniform-spectrum
    `wkb1_term` evaluated on the WHOLE plane with the scalars of column x; the term is exactly what the frozen-coefficient
    local closure subtracts; identical blocks give the uniform-spectrum variant."""
    ny, nx = 12, 20
    en, wt, db = np.array([80.0, 120.0]), np.array([0.4, 0.6]), np.array([8.0, 12.0])   # small δ/β: α²/4 is not small
    t = np.linspace(0.0, 1.0, 4)[:, None]
    # line-dependent tilts of the weights: after the per-block normalisation f_s(x) really varies with x
    prof = O.derive_profiles(6.5e-6, 8.0, en, nx, wt[None, :] * (1.0 + t * np.array([0.8, -0.5])[None, :]),
                             db[None, :] * (1.0 + 0.3 * t))
    assert np.ptp(prof.f[0]) > 0.1 and np.ptp(prof.gamma[0]) > 0.01
    tau = 0.3 * (1.0 + 0.5 * _smooth(ny, nx, 21))
    P0, b0, _ = O.forward_x(tau, prof, "nonlocal", S=8.0)
    P1, b1, _ = O.forward_x(tau, prof, "nonlocal", S=8.0, nonlocal_wkb1=True)
    assert np.linalg.norm(P1 - P0) > 1e-4 * np.linalg.norm(P0 - 1.0)                    # the variant does something
    for s in range(2):
        for x in range(nx):
            I = prof.f[s, x] * np.exp(-prof.gamma[s, x] * tau)
            want = O.wkb1_term(I, prof.alpha[s])[:, x]
            assert np.max(np.abs((b0[s] - b1[s])[:, x] - want)) < 1e-15          # a difference of O(1) planes; term ~ 3e-4
        loc = O.closure_x(tau, prof, s, 2, False) - O.closure_x(tau, prof, s, 2, True)
        assert np.max(np.abs((b0[s] - b1[s]) - loc)) < 1e-13
    uni = O.derive_profiles(6.5e-6, 8.0, en, nx, [wt] * 4, [db] * 4)
    lines = O.derive_lines(6.5e-6, 8.0, en, wt, db)
    d = 1.0 + 0.1 * _smooth(ny, nx, 3)
    t_x = O.retrieve_x(d, uni, "nonlocal", 3, 0.4, S=8.0, nonlocal_wkb1=True)
    t_u = O.retrieve(d, lines, "nonlocal", 3, 0.4, S=8.0, nonlocal_wkb1=True)
    assert np.max(np.abs(t_x - t_u)) < 1e-13
    assert np.max(np.abs(t_u - O.retrieve(d, lines, "nonlocal", 3, 0.4, S=8.0))) > 1e-6


def test_max_shift_x_plain_loops_and_histories():
    """Regime indicator with the x-dependent spectrum: the largest |a_s(x) γ_s(x) D⁰τ| over pixels, lines and the two
    axes, written out in plain loops; `retrieve_x` records it and the residual RMS once per iteration, and identical
    blocks give the uniform-spectrum histories."""
    ny, nx = 10, 16
    prof, _, _ = _varying(nx, 4, L=300.0, mu=True)
    tau = 0.2 * (1.0 + 0.5 * _smooth(ny, nx, 17))
    want = 0.0
    for s in range(3):
        for y in range(ny):
            for x in range(nx):
                c = prof.a[s, x] * prof.gamma[s, x]
                want = max(want, c * abs(tau[y, (x + 1) % nx] - tau[y, (x - 1) % nx]) / 2.0,
                           c * abs(tau[(y + 1) % ny, x] - tau[(y - 1) % ny, x]) / 2.0)
    assert abs(O.max_shift_x(tau, prof) - want) < 1e-14 * want and want > 0.1
    uni = O.derive_profiles(6.5e-6, 20.0, E3, nx, [W3] * 2, [DB3] * 2)
    lines = O.derive_lines(6.5e-6, 20.0, E3, W3, DB3)
    d = 1.0 + 0.1 * _smooth(ny, nx, 4)
    hx, sx, hu, su = [], [], [], []
    O.retrieve_x(d, uni, "nonlocal", 3, 0.4, S=8.0, history=hx, shift_history=sx)
    O.retrieve(d, lines, "nonlocal", 3, 0.4, S=8.0, history=hu, shift_history=su)
    assert len(hx) == 3 and len(sx) == 3
    assert np.allclose(hx, hu, rtol=1e-11, atol=0) and np.allclose(sx, su, rtol=1e-11, atol=0)
    assert abs(sx[0] - O.max_shift(O.paganin_init(d, lines), lines)) < 1e-12 * sx[0]


def test_positivity_floor_with_profiles():
    """PAPER.md:225 "nonnegative spectral components", Eq. (7) PAPER.md:227 with the column's scalars: the total intensity
    is floored at i_min before it is put back on the manifold, in the start (R9) and in the loop.  Vanishing propagation
    distance: every filter is the identity (the block weights sum to one), so step = 1 from a constant start gives
    Σ_s I_s = d pixel by pixel; a pixel of d forced to −1 must come back at the τ with Σ_s f_s(x) e^{−γ_s(x) τ} = i_min for
    ITS column, found here by bracketing (brentq) on the column's scalars."""
    from scipy.optimize import brentq
    ny, nx, i_min = 8, 12, 1e-3
    prof, _, _ = _varying(nx, 4, L=1e-12, mu=True)
    assert np.max(prof.a) < 1e-9 and np.ptp(prof.gamma[0]) > 0.05
    d = np.full((ny, nx), 0.9)
    d[3, 5] = -1.0
    f5, g5 = prof.f[:, 5], prof.gamma[:, 5]
    want = brentq(lambda t: float(np.sum(f5 * np.exp(-g5 * t))) - i_min, 0.0, 1e3, xtol=1e-14, rtol=1e-14)
    for tau in (O.paganin_init_x(d, prof, i_min=i_min),
                O.retrieve_x(d, prof, "local", iterations=1, step=1.0, i_min=i_min, tau0=np.full(d.shape, 0.2)),
                O.retrieve_x(d, prof, "nonlocal", iterations=1, step=1.0, i_min=i_min, tau0=np.full(d.shape, 0.2))):
        assert np.all(np.isfinite(tau))
        assert abs(tau[3, 5] - want) < 1e-10 * want
        T = np.sum(O.line_intensities_x(tau, prof), axis=0)
        assert np.max(np.abs(np.delete(T.ravel(), 3 * nx + 5) - 0.9)) < 1e-9


@pytest.mark.parametrize("solver", ["local", "nonlocal"])
def test_residual_history_with_profiles_is_the_rms(solver):
    """`retrieve_x(history=…)`: root mean square of e = d − Σ_s P_s.  Constant start τ⁰: Σ_s P_s is the
    column's T⁰(x) = Σ_s f_s(x) e^{−γ_s(x) τ⁰}; d = T⁰(x) + ε cos(θ·r) over whole periods gives ε/√2 first."""
    ny, nx, eps, tau0 = 16, 24, 0.03, 0.2
    prof, _, _ = _varying(nx, 4, L=1.0, mu=True)
    T0 = np.sum(prof.f * np.exp(-prof.gamma * tau0), axis=0)[None, :]
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    d = T0 + eps * np.cos(2 * np.pi * (3 * x / nx + 2 * y / ny))
    h = []
    O.retrieve_x(d, prof, solver, iterations=2, step=0.5, tau0=np.full((ny, nx), tau0), history=h)
    assert len(h) == 2 and abs(h[0] - eps / np.sqrt(2.0)) < 1e-12 and abs(h[0] - 2 * eps / np.pi) > 1e-3
