"""Pins for the fp64 oracle's iteration (CPU only): special cases, limits, self-consistency."""
import numpy as np
import pytest

from oracle import epr_oracle as O

RNG = np.random.default_rng(777)


def _smooth(ny, nx, seed, scale=1.0):
    """Smooth periodic random field in [-scale, scale] (few low Fourier modes)."""
    rng = np.random.default_rng(seed)
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    f = np.zeros((ny, nx))
    for _ in range(6):
        m, n = rng.integers(-3, 4, size=2)
        f += rng.normal() * np.cos(m * x + n * y + rng.uniform(0, 2 * np.pi))
    return scale * f / np.max(np.abs(f))


def _mono(a_target=60.0):
    p, E, db = 6.5e-6, 100.0, 1000.0
    k = 2 * np.pi * E / O.HC_KEV_M
    L = a_target * 2.0 / db * k * p * p
    return O.derive_lines(p, L, [E], [1.0], [db])


def test_L1_mono_one_iteration_equals_paganin():
    """L1 mono is the Paganin single-distance retrieval.  With order=1, step=1 one
    iteration from ANY start gives IFFT(FFT(d)/(1+a lambda)) (discrete symbol, R5)."""
    lines = _mono()
    d = 1.0 + 0.2 * _smooth(32, 48, 1)
    tau0 = 0.3 * RNG.uniform(size=d.shape)
    tau = O.retrieve(d, lines, "local", iterations=1, step=1.0, order=1, tau0=tau0)
    pag = O.precondition(d, lines.a[0], 0)
    assert np.max(np.abs(np.exp(-tau) - pag)) < 1e-13
    # and iterations=0 returns exactly that Paganin result (R9)
    tau_init = O.retrieve(d, lines, "local", iterations=0)
    assert np.max(np.abs(np.exp(-tau_init) - pag)) < 1e-14


def test_weak_phase_limit_converges_to_paganin_linearly():
    """north_star pin: in the weak-phase limit the local-closure solution tends to the linear Paganin
    retrieval; the relative difference is proportional to the object strength eps."""
    lines = _mono(40.0)
    b = _smooth(48, 48, 2)
    ratios = []
    for eps in (1e-2, 1e-3, 1e-4):
        truth = eps * (1.0 + 0.5 * b)
        d, _, _ = O.forward(truth, lines, "local")
        tau = O.retrieve(d, lines, "local", iterations=12, step=1.0)
        pag = O.retrieve(d, lines, "local", iterations=0)
        assert np.max(np.abs(tau - truth)) < 1e-9 * max(1.0, eps / 1e-4)     # recovers its own data
        ratios.append(np.linalg.norm(tau - pag) / np.linalg.norm(pag - pag.mean()))
    assert ratios[0] < 5e-2
    assert 8.0 < ratios[0] / ratios[1] < 12.0
    assert 8.0 < ratios[1] / ratios[2] < 12.0


@pytest.mark.parametrize("solver,step,iters,bound", [("local", 1.0, 12, 1e-4), ("nonlocal", 0.4, 12, 0.15)])
def test_self_consistent_data_drive_residual_down(solver, step, iters, bound):
    """Noise-free data made by the same operator: the residual history falls monotonically over the
    first dozen iterations and the largest gain is at the first one.  (The non-local
    iteration is only slowly contractive: its residual stalls near 10 % — the bilinear "quantisation
    effect" of PAPER.md:79 — which is why the bound differs.)"""
    lines = _mono(50.0)
    truth = 0.05 * (1.0 + 0.8 * _smooth(64, 64, 3))
    d, _, _ = O.forward(truth, lines, solver)
    hist = []
    tau = O.retrieve(d, lines, solver, iterations=iters, step=step, history=hist)
    assert all(h1 < h0 for h0, h1 in zip(hist, hist[1:]))
    assert hist[-1] < bound * hist[0]
    drops = [h0 - h1 for h0, h1 in zip(hist, hist[1:])]
    assert drops[0] == max(drops)
    assert np.linalg.norm(tau - truth) < np.linalg.norm(O.retrieve(d, lines, solver, iterations=0) - truth)


def test_poly_with_identical_lines_reduces_to_mono():
    """Eq. (5)/(7): N_s copies of the same line (equal gamma, db, E) must reproduce the mono result."""
    p, E, db, L = 6.5e-6, 100.0, 1000.0, 2.0
    mono = O.derive_lines(p, L, [E], [1.0], [db])
    poly = O.derive_lines(p, L, [E, E, E], [0.2, 0.5, 0.3], [db, db, db])
    assert np.allclose(poly.gamma, 1.0)
    d = 1.0 + 0.1 * _smooth(32, 32, 4)
    for solver, step in (("local", 1.0), ("nonlocal", 0.4)):
        t1 = O.retrieve(d, mono, solver, iterations=4, step=step)
        t3 = O.retrieve(d, poly, solver, iterations=4, step=step)
        assert np.max(np.abs(t1 - t3)) < 1e-12


def test_fourier_sum_identity_R10():
    """R10 consequence: only the SUM of the per-line updates enters the projection, so summing the
    filtered residuals in Fourier space and inverse-transforming once changes nothing."""
    E = np.array([70.0, 100.0, 130.0])
    lines = O.derive_lines(6.5e-6, 3.0, E, [0.3, 0.4, 0.3], [900.0, 1000.0, 1100.0])
    assert np.ptp(lines.a) > 1.0                                   # unequal a_s
    r = [RNG.normal(size=(16, 20)) for _ in range(3)]
    per_line = sum(O.precondition(r[s], lines.a[s]) for s in range(3))
    lam = O.symbol_lambda(16, 20, 0)
    fused = np.real(np.fft.ifft2(sum(np.fft.fft2(r[s]) / (1 + lines.a[s] * lam) for s in range(3))))
    assert np.max(np.abs(per_line - fused)) < 1e-13


def test_split_weights_sum_to_one_and_fallback():
    lines = O.derive_lines(6.5e-6, 3.0, [80.0, 120.0], [0.4, 0.6], [800.0, 1200.0])
    P = [RNG.uniform(-0.2, 1.0, size=(8, 8)), RNG.uniform(-0.2, 1.0, size=(8, 8))]
    P[0][0, 0] = P[1][0, 0] = -1.0                                 # both negative: fallback to f_s
    w = O.split_weights(P, lines)
    assert np.max(np.abs(w[0] + w[1] - 1.0)) < 1e-15
    assert w[0][0, 0] == lines.f[0] and w[1][0, 0] == lines.f[1]
    assert (w[0] >= 0).all() and (w[1] >= 0).all()


def test_local_solver_degrades_beyond_one_pixel_nonlocal_stays_stable():
    """PAPER.md:97 (qualitative): with multi-pixel shifts the local closure diverges while the
    non-local solver with relaxation 0.4 stays stable."""
    lines = _mono(400.0)
    truth = 0.15 * (1.0 + _smooth(64, 64, 5))
    ux, _ = O.ray_map(np.exp(-truth), lines.a[0], 16.0)
    assert np.max(np.abs(ux)) > 1.5
    d, _, _ = O.forward(truth, lines, "nonlocal")
    h_loc, h_non = [], []
    with np.errstate(all="ignore"):
        O.retrieve(d, lines, "local", iterations=8, step=1.0, history=h_loc)
    O.retrieve(d, lines, "nonlocal", iterations=8, step=0.4, history=h_non)
    assert h_non[-1] < h_non[0]
    assert not (h_loc[-1] < h_non[-1])


def test_max_shift_closed_form_and_history():
    """I = exp(c x) (one line): u_x = a c exactly wherever the central difference does not straddle the periodic seam,
    u_y = 0; the indicator is not clamped.  The histories have one entry per iteration."""
    lines = _mono(50.0)
    ny, nx, c = 8, 64, 0.03
    tau = -c * np.tile(np.arange(nx, dtype=np.float64), (ny, 1))          # I = exp(c x)
    ux, uy = O.ray_map(np.exp(-tau), lines.a[0], np.inf)
    assert np.max(np.abs(ux[:, 1:-1] - lines.a[0] * c)) < 1e-10 and np.max(np.abs(uy)) == 0.0
    seam = lines.a[0] * c * (nx - 2) / 2.0                                 # |D0| across the wrap: (x_0 - x_{n-2}) / 2
    assert abs(O.max_shift(tau, lines) - seam) < 1e-9 * seam
    d = 1.0 + 0.01 * _smooth(32, 32, 3)
    h, sh = [], []
    O.retrieve(d, lines, "local", iterations=3, step=1.0, history=h, shift_history=sh)
    assert len(h) == len(sh) == 3 and all(v > 0 for v in sh)
    E = np.array([80.0, 120.0])
    l2 = O.derive_lines(6.5e-6, 2.0, E, [0.5, 0.5], [800.0, 1200.0])
    t2 = 0.1 * (1.0 + _smooth(16, 16, 9))
    per_line = [max(np.max(np.abs(l2.a[s] * l2.gamma[s] * O.d0x(t2))), np.max(np.abs(l2.a[s] * l2.gamma[s] * O.d0y(t2))))
                for s in range(2)]
    assert abs(O.max_shift(t2, l2) - max(per_line)) < 1e-12             # D0 ln I_s = −γ_s D0 τ (Eq. (7))


def test_nonlocal_wkb1_variant_keeps_mass_and_vanishes_for_exponentials():
    """Variant of R4: the WKB1 term of Eq. (1) added to the ray-map prediction.  It is a discrete
    divergence, so the total intensity is still conserved; for I = exp(cx + dy) the quantum potential Q is constant
    (interior) and the term vanishes; and it is exactly the term the local closure subtracts."""
    E = np.array([80.0, 120.0])
    lines = O.derive_lines(6.5e-6, 8.0, E, [0.4, 0.6], [8.0, 12.0])          # small δ/β: α²/4 = (a/db)² is not small
    tau = 0.3 * (1.0 + _smooth(24, 32, 11))
    P0, b0, _ = O.forward(tau, lines, "nonlocal", S=8.0)
    P1, b1, _ = O.forward(tau, lines, "nonlocal", S=8.0, nonlocal_wkb1=True)
    Is = O.line_intensities(tau, lines)
    assert np.linalg.norm(P1 - P0) > 1e-4 * np.linalg.norm(P0 - np.sum(Is, axis=0))   # the variant does something
    for s in range(2):
        assert abs(b1[s].sum() - Is[s].sum()) < 1e-12 * Is[s].sum()
        loc = O.closure(Is[s], lines.a[s], lines.alpha[s], 2, False) - O.closure(Is[s], lines.a[s], lines.alpha[s], 2, True)
        assert np.max(np.abs((b0[s] - b1[s]) - loc)) < 1e-13
    y, x = np.meshgrid(np.arange(16.0), np.arange(16.0), indexing="ij")
    W = O.wkb1_term(np.exp(0.03 * x - 0.02 * y), 3.0)
    assert np.max(np.abs(W[3:-3, 3:-3])) < 1e-12


# --------------------------------------------------------------------------------------------------------------------
# Closed-form pins of the polychromatic loop body: per-line filter coefficient, positivity-weighted
# split, weighted-mean Paganin start, positivity floor.  Each of them is a number worked out by hand from the paper's
# statement of the step, not a second call of the routine under test.
# --------------------------------------------------------------------------------------------------------------------
def _three_unequal_lines(L=3.0):
    E = np.array([70.0, 100.0, 130.0])
    lines = O.derive_lines(6.5e-6, L, E, [0.3, 0.45, 0.25], [600.0, 1000.0, 1500.0])
    assert np.ptp(lines.a) > 0.2 * lines.a.mean() and np.ptp(lines.gamma) > 0.3          # unequal a_s and γ_s
    return lines


def _lam(ny, nx, my, mx):
    """Discrete 5-point symbol of the mode cos(2π(mx x/nx + my y/ny)), written out (R5)."""
    return (2.0 - 2.0 * np.cos(2 * np.pi * mx / nx)) + (2.0 - 2.0 * np.cos(2 * np.pi * my / ny))


@pytest.mark.parametrize("solver", ["local", "nonlocal"])
def test_one_iteration_from_constant_start_closed_form(solver):
    """PAPER.md:231 "split [the residual] across spectral lines with positivity-weighted weights … apply a per-line
    FFT-diagonal inverse".  Start from a CONSTANT τ⁰ = c: every P_s = I_s = f_s e^{−γ_s c} is constant (all differences
    vanish, zero shift = identity transport), so w_s = I_s/T⁰ with T⁰ = Σ_s I_s, and for d = T⁰ + ε cos(θ·r) one
    iteration gives   Σ_s I_s = T⁰ + step·ε·cos(θ·r)·Σ_s w_s/(1 + a_s λ(θ))   — each line filtered with ITS OWN a_s."""
    lines = _three_unequal_lines()
    ny, nx, my, mx, c, eps, step = 24, 32, 2, 3, 0.8, 1e-3, 0.7
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    mode = np.cos(2 * np.pi * (mx * x / nx + my * y / ny))
    I0 = lines.f * np.exp(-lines.gamma * c)
    T0 = I0.sum()
    d = T0 + eps * mode
    tau = O.retrieve(d, lines, solver, iterations=1, step=step, tau0=np.full((ny, nx), c))
    got = np.sum(O.line_intensities(tau, lines), axis=0)
    w = I0 / T0
    gain = float(np.sum(w / (1.0 + lines.a * _lam(ny, nx, my, mx))))
    want = T0 + step * eps * mode * gain
    assert np.max(np.abs(got - want)) < 1e-12
    # the pin has teeth: the weighted-mean coefficient, or weights f_s, would be off by far more than the tolerance
    wrong_a = float(np.sum(w / (1.0 + lines.abar * _lam(ny, nx, my, mx))))
    wrong_w = float(np.sum(lines.f / (1.0 + lines.a * _lam(ny, nx, my, mx))))
    assert abs(wrong_a - gain) * step * eps > 1e-7 and abs(wrong_w - gain) * step * eps > 1e-7


def test_paganin_init_several_lines_uses_weighted_mean_coefficient():
    """R9 with PAPER.md:51: the start is ONE linear Paganin solve with ā = Σ_s f_s a_s, so for d = 1 + ε cos(θ·r) the
    total intensity of the start is 1 + ε cos(θ·r)/(1 + ā λ(θ)), ā worked out here from the physical constants."""
    lines = _three_unequal_lines()
    ny, nx, my, mx, eps = 20, 28, 1, 4, 2e-3
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    mode = np.cos(2 * np.pi * (mx * x / nx + my * y / ny))
    E, wgt, db = np.array([70.0, 100.0, 130.0]), np.array([0.3, 0.45, 0.25]), np.array([600.0, 1000.0, 1500.0])
    a_s = 3.0 * O.HC_KEV_M / (2 * np.pi * E) / (6.5e-6) ** 2 * db / 2.0          # (L/k_s p²)·db_s/2
    abar = float(np.sum(wgt / wgt.sum() * a_s))
    tau = O.paganin_init(1.0 + eps * mode, lines)
    got = np.sum(O.line_intensities(tau, lines), axis=0)
    assert np.max(np.abs(got - (1.0 + eps * mode / (1.0 + abar * _lam(ny, nx, my, mx))))) < 1e-13
    assert abs(1.0 / (1.0 + a_s[0] * _lam(ny, nx, my, mx)) - 1.0 / (1.0 + abar * _lam(ny, nx, my, mx))) * eps > 1e-6


def test_split_weights_hand_computed():
    """R8 ("positivity-weighted"): w_s = P_s⁺/Σ_t P_t⁺.  (0.3, 0.1) → (0.75, 0.25); a negative prediction
    gets no share: (−0.2, 0.5) → (0, 1); both non-positive → the spectral fractions f_s."""
    lines = O.derive_lines(6.5e-6, 3.0, [80.0, 120.0], [0.4, 0.6], [800.0, 1200.0])
    P = [np.array([[0.3, -0.2, -0.1, 0.0]]), np.array([[0.1, 0.5, -0.3, 0.0]])]
    w = O.split_weights(P, lines)
    assert np.allclose(w[0][0, :2], [0.75, 0.0], atol=1e-15) and np.allclose(w[1][0, :2], [0.25, 1.0], atol=1e-15)
    assert np.allclose(w[0][0, 2:], 0.4, atol=1e-15) and np.allclose(w[1][0, 2:], 0.6, atol=1e-15)


@pytest.mark.parametrize("n_lines", [1, 3])
def test_positivity_floor_returns_tau_of_i_min(n_lines):
    """PAPER.md:225 "nonnegative spectral components": the total intensity is floored at i_min before it is put back on
    the manifold Eq. (7).  With a vanishing propagation distance the filter is the identity, so step = 1 from a constant
    start gives Σ_s I_s = d pixel by pixel; a pixel of d forced to −1 must come back at exactly the τ with
    Σ_s f_s e^{−γ_s τ} = i_min (one line: τ = −ln i_min), in the start (R9) and in the loop."""
    if n_lines == 1:
        lines = O.derive_lines(6.5e-6, 1e-12, [100.0], [1.0], [1000.0])
    else:
        lines = _three_unequal_lines(L=1e-12)
    assert np.max(lines.a) < 1e-9
    i_min = 1e-3
    d = np.full((8, 12), 0.9)
    d[3, 5] = -1.0
    for tau in (O.paganin_init(d, lines, i_min=i_min),
                O.retrieve(d, lines, "local", iterations=1, step=1.0, i_min=i_min, tau0=np.full(d.shape, 0.2)),
                O.retrieve(d, lines, "nonlocal", iterations=1, step=1.0, i_min=i_min, tau0=np.full(d.shape, 0.2))):
        assert np.all(np.isfinite(tau))
        T = np.sum(O.line_intensities(tau, lines), axis=0)
        assert abs(T[3, 5] - i_min) < 1e-12 * i_min * 1e3
        assert np.max(np.abs(np.delete(T.ravel(), 3 * 12 + 5) - 0.9)) < 1e-9
        if n_lines == 1:
            assert abs(tau[3, 5] + np.log(i_min)) < 1e-12


def test_shift_histogram_closed_form():
    """η = ‖Δ‖/p per line.  τ = −(c x + e y) (I_s = f_s exp(γ_s (c x + e y))) gives the same shift
    a_s γ_s √(c² + e²) at every pixel whose central differences do not straddle the periodic seam, so each line's
    histogram is one spike of (nx − 2)(ny − 2) pixels in a bin known in closed form; the seam pixels (larger differences)
    land in higher bins; every row sums to the number of pixels."""
    E = np.array([80.0, 120.0])
    lines = O.derive_lines(6.5e-6, 2.0, E, [0.5, 0.5], [800.0, 1200.0])
    ny, nx, c, e = 12, 20, 0.003, 0.004
    y, x = np.meshgrid(np.arange(ny, dtype=np.float64), np.arange(nx, dtype=np.float64), indexing="ij")
    tau = -(c * x + e * y) + 1.0
    n_hist, bin_px = 40, 0.05
    h = O.shift_histogram(tau, lines, n_hist, bin_px)
    assert h.shape == (2, n_hist) and np.all(h.sum(axis=1) == nx * ny)
    for s in range(2):
        eta = lines.a[s] * lines.gamma[s] * np.hypot(c, e)
        k = int(np.floor(eta / bin_px))
        assert 0 < k < n_hist - 1
        assert h[s, k] == (nx - 2) * (ny - 2)
        assert h[s, :k].sum() == 0 and h[s, k + 1:].sum() == nx * ny - (nx - 2) * (ny - 2)   # seam pixels: larger shifts
    assert int(np.argmax(h[0])) != int(np.argmax(h[1]))              # the lines differ (Fig. 6: one curve per line)


def test_phase_is_eq6_written_out():
    """Eq. (6) PAPER.md:216 with Eq. (7): φ_s = (db_s/2) ln(I_s / f_s) = (db_s/2)(ln I_s − ln f_s), db_s = δ_s/β_s
    retyped here, I_s from `line_intensities`.  One line (γ = 1, f = 1): φ = (δ/2β) ln e^{−τ}.  A thicker object gives a more
    NEGATIVE phase (δ > 0: the wave is advanced in matter), which fixes the sign."""
    db = [800.0, 1200.0]
    lines = O.derive_lines(6.5e-6, 2.0, [80.0, 120.0], [0.4, 0.6], db)
    tau = 0.3 * (1.2 + _smooth(16, 24, 31))
    Is = O.line_intensities(tau, lines)
    for s in range(2):
        want = (db[s] / 2.0) * (np.log(Is[s]) - np.log(lines.f[s]))
        assert np.max(np.abs(O.phase(tau, lines, s) - want)) < 1e-12 * np.max(np.abs(want))
    one = O.derive_lines(6.5e-6, 2.0, [100.0], [1.0], [1000.0])
    assert np.max(np.abs(O.phase(tau, one) - 500.0 * np.log(np.exp(-tau)))) < 1e-11
    assert np.all(O.phase(tau, one) < 0.0) and np.all(O.phase(2.0 * tau, one) < O.phase(tau, one))


@pytest.mark.parametrize("solver", ["local", "nonlocal"])
def test_residual_history_is_the_rms(solver):
    """PAPER.md:231 "form the detector residual", PAPER.md:95 (convergence history): `history[n]` is the root mean square of
    e = d − Σ_s P_s over the pixels.  From a CONSTANT start τ⁰ every operator leaves the constant planes I_s alone, so
    Σ_s P_s = T⁰ = Σ_s f_s e^{−γ_s τ⁰} exactly; with d = T⁰ + ε cos(θ·r) over whole periods the first entry is ε/√2
    (a mean of |e| would give 2ε/π)."""
    lines = _three_unequal_lines(L=1.0)
    ny, nx, eps, tau0 = 16, 24, 0.03, 0.2
    T0 = float(np.sum(lines.f * np.exp(-lines.gamma * tau0)))
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    d = T0 + eps * np.cos(2 * np.pi * (3 * x / nx + 2 * y / ny))
    h = []
    O.retrieve(d, lines, solver, iterations=2, step=0.5, tau0=np.full((ny, nx), tau0), history=h)
    assert len(h) == 2
    assert abs(h[0] - eps / np.sqrt(2.0)) < 1e-13
    assert abs(h[0] - 2 * eps / np.pi) > 1e-3
