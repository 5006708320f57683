"""Pins for the oracle's oversampled-grid functions (reading R16; CPU only)."""
import numpy as np
import pytest

from oracle import epr_oracle as O

RNG = np.random.default_rng(4242)


@pytest.mark.parametrize("m", [1, 2, 3, 4])
def test_up_and_down_against_their_definitions(m):
    """Brute force from the definitions: fine[Y][X] = d[Y // m][X // m]; coarse = mean over the m x m block."""
    d = RNG.normal(size=(5, 6))
    up = O.upsample(d, m)
    assert up.shape == (5 * m, 6 * m)
    for Y in range(5 * m):
        for X in range(6 * m):
            assert up[Y, X] == d[Y // m, X // m]
    t = RNG.normal(size=(4 * m, 3 * m))
    down = O.downsample(t, m)
    for y in range(4):
        for x in range(3):
            acc = 0.0
            for j in range(m):
                for i in range(m):
                    acc += t[m * y + j, m * x + i]
            assert abs(down[y, x] - acc / (m * m)) < 1e-15


@pytest.mark.parametrize("m", [2, 4])
def test_down_is_the_left_inverse_of_up_and_both_keep_the_mean(m):
    d = RNG.uniform(0.5, 1.5, size=(8, 12))
    assert np.array_equal(O.downsample(O.upsample(d, m), m), d)           # exact for m a power of two
    assert abs(O.upsample(d, m).mean() - d.mean()) < 1e-15
    t = RNG.normal(size=(8 * m, 12 * m))
    assert abs(O.downsample(t, m).mean() - t.mean()) < 1e-15


@pytest.mark.parametrize("m", [2, 4])
@pytest.mark.parametrize("k", [1, 3, 7])
def test_replicate_filter_average_acts_on_a_detector_mode_by_its_closed_form_gain(m, k):
    """down ∘ (fine-grid Paganin filter) ∘ up is shift-invariant on the detector grid.  Replication spreads the
    detector mode k over the fine modes k + j n (j < m) with the box weights B_j = (1/m) Σ_{i<m} e^{−2πi (k + j n) i/(m n)},
    the filter scales each by 1/(1 + a λ_f), the block mean folds them back with conj(B_j):
        gain(k) = Σ_j |B_j|² / (1 + a (2 − 2 cos(2π (k + j n)/(m n)))),   Σ_j |B_j|² = 1.
    A misplaced block (an off-by-one in // or in the block mean) turns the gain complex and fails this."""
    n, a = 16, 7.3
    x = np.arange(n)
    d = np.tile(np.cos(2 * np.pi * k * x / n + 0.4), (4, 1))              # varies along x only
    got = O.downsample(O.precondition(O.upsample(d, m), a), m)
    gain = 0.0
    for j in range(m):
        kk = k + j * n
        B = np.mean(np.exp(-2j * np.pi * kk * np.arange(m) / (m * n)))
        gain += abs(B) ** 2 / (1.0 + a * (2.0 - 2.0 * np.cos(2 * np.pi * kk / (m * n))))
    assert np.max(np.abs(got - gain * d)) < 1e-13
    wsum = sum(abs(np.mean(np.exp(-2j * np.pi * (k + j * n) * np.arange(m) / (m * n)))) ** 2 for j in range(m))
    assert abs(wsum - 1.0) < 1e-14


def _lines(pixel, n_lines=1):
    E = np.linspace(80.0, 120.0, n_lines) if n_lines > 1 else np.array([100.0])
    return O.derive_lines(pixel, 0.8, E, np.ones(n_lines), 1000.0 * E / 100.0)


def test_factor_one_is_the_plain_loop():
    d = 1.0 + 0.05 * RNG.normal(size=(16, 16))
    lines = _lines(6.5e-6)
    assert np.array_equal(O.retrieve_oversampled(d, lines, 1, "local", 3, 1.0), O.retrieve(d, lines, "local", 3, 1.0))


@pytest.mark.parametrize("solver,n_lines", [("local", 1), ("nonlocal", 1), ("nonlocal", 3)])
def test_uniform_image_gives_the_closed_form_thickness(solver, n_lines):
    """d = c everywhere: every operator leaves a constant alone, so τ solves Σ_s f_s e^{−γ_s τ} = c at any factor
    (one line: τ = −ln c)."""
    c = 0.8
    d = np.full((8, 8), c)
    for m in (2, 4):
        lines = _lines(6.5e-6 / m, n_lines)
        tau = O.retrieve_oversampled(d, lines, m, solver, 2, 0.4 if solver == "nonlocal" else 1.0)
        assert tau.shape == (8, 8)
        T = sum(lines.f[s] * np.exp(-lines.gamma[s] * tau) for s in range(n_lines))
        assert np.max(np.abs(T - c)) < 1e-12
        if n_lines == 1:
            assert np.max(np.abs(tau + np.log(c))) < 1e-12


def test_fine_pixel_scalars_scale_as_the_square_of_the_factor():
    """shifts are counted in pixels of the internal grid, so α_s and a_s grow by m² on a grid refined
    m times (ε_s = L/k_s is a length²)."""
    l1, l2 = _lines(6.5e-6, 3), _lines(6.5e-6 / 2, 3)
    assert np.allclose(l2.alpha, 4.0 * l1.alpha, rtol=1e-14) and np.allclose(l2.a, 4.0 * l1.a, rtol=1e-14)
    assert np.allclose(l2.gamma, l1.gamma, rtol=1e-14)


def test_factor_one_nonlocal_hands_the_clamp_through():
    """PAPER.md:167 ("the internal pixel size on the oversampled grid"): S counts pixels of the grid the loop runs on and is
    handed to it unchanged.  With a clamp that BINDS (largest shift of the start > S) factor 1 must be the plain
    non-local loop with the same S — and not the loop with 2 S."""
    ny, nx, S = 16, 24, 0.1
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    d = 1.0 + 0.3 * np.cos(2 * x + y) + 0.2 * np.sin(3 * y - x)
    lines = O.derive_lines(6.5e-6, 30.0, [100.0], [1.0], [1000.0])
    tau0 = O.paganin_init(d, lines)
    assert 2 * S < O.max_shift(tau0, lines)                                # the clamp binds at S and still at 2 S
    plain = O.retrieve(d, lines, "nonlocal", 3, 0.4, S=S)
    assert np.array_equal(O.retrieve_oversampled(d, lines, 1, "nonlocal", 3, 0.4, S=S), plain)
    assert np.max(np.abs(O.retrieve(d, lines, "nonlocal", 3, 0.4, S=2 * S) - plain)) > 1e-6
    # and at factor 2: the fine loop written out with the same S
    fine = O.derive_lines(6.5e-6 / 2, 30.0, [100.0], [1.0], [1000.0])
    want = O.downsample(O.retrieve(O.upsample(d, 2), fine, "nonlocal", 2, 0.4, S=S), 2)
    assert np.array_equal(O.retrieve_oversampled(d, fine, 2, "nonlocal", 2, 0.4, S=S), want)
