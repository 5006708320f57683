"""GPU parity: the CUDA path (through the C-ABI binding) against the fp64 oracle, element by element, on the
same seeded inputs.  Tolerances are north_star's: per-operator relative L2 <= 1e-5, retrieved phase <= 1e-4,
splat mass conservation <= 1e-6 relative."""
import numpy as np
import pytest

from epr_inputs import make_workload
from oracle import epr_oracle as O

pytestmark = pytest.mark.gpu

TOL_OP = 1e-5
TOL_PHASE = 1e-4
TOL_MASS = 1e-6


K_MAX = 10.0      # element-wise bound: max|got − ref| <= K_MAX · tol · max|ref| (DESIGN.md §8 "Element-wise bound")


def rel_l2(got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    return float(np.linalg.norm(got - ref) / np.linalg.norm(ref))


def max_rel(got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    return float(np.max(np.abs(got - ref)) / np.max(np.abs(ref)))


def assert_close(got, ref, tol, what=""):
    """Both views of the same comparison: the relative L2 norm north_star states, and an element-wise bound so that a
    single wrong row, tile seam or pixel cannot hide in the norm of a multi-megapixel plane."""
    r, m = rel_l2(got, ref), max_rel(got, ref)
    assert r < tol, f"{what}: rel L2 {r:.3e} >= {tol:g}"
    assert m <= K_MAX * tol, f"{what}: max|got - ref| / max|ref| = {m:.3e} > {K_MAX:g} x {tol:g} (rel L2 {r:.3e})"


@pytest.fixture(scope="module")
def E():
    import torch
    import paper_2601_22793_b200 as epr
    assert torch.cuda.is_available()
    epr.load_library()
    return epr


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def _tau_field(ny, nx, seed, amp=0.05):
    """Smooth + rough thickness-like field (fp32-representable)."""
    rng = np.random.default_rng(seed)
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    t = amp * (1.2 + np.cos(2 * x + 0.3) * np.sin(3 * y) + 0.5 * np.cos(5 * x - 4 * y))
    t += 0.02 * amp * rng.normal(size=(ny, nx))
    return t.astype(np.float32)


POLY = dict(energy=np.linspace(60.0, 140.0, 8), weight=np.exp(-0.5 * ((np.linspace(60.0, 140.0, 8) - 100.0) / 20.0) ** 2))
SPECTRA = {
    "mono": (np.array([100.0]), np.array([1.0]), np.array([1000.0])),
    "poly8": (POLY["energy"], POLY["weight"], 200.0 * POLY["energy"] / 100.0),
    "poly3_unequal_a": (np.array([70.0, 100.0, 130.0]), np.array([0.3, 0.4, 0.3]), np.array([900.0, 1000.0, 1100.0])),
}
# (ny, nx): powers of two and radix-3/5 lengths; ny = 256 … 2048 with nx % 8 == 0 take the TMA-staged column kernel
# 2160 = 16·15·9, 2560 = 16·16·10, 1080 = 8·15·9 exercise the composite radices
SIZES = [(256, 256), (48, 80), (160, 96), (320, 512), (512, 128), (1024, 64), (2048, 32), (2160, 32), (32, 2160),
         (2560, 16), (16, 2560)]


@pytest.mark.parametrize("ny,nx", SIZES)
@pytest.mark.parametrize("spec", ["mono", "poly3_unequal_a"])
@pytest.mark.parametrize("symbol", [0, 1])
def test_precondition(E, ny, nx, spec, symbol):
    import torch
    en, w, db = SPECTRA[spec]
    L = 3.0
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "local", max_batch=2, symbol=symbol)
    lines = O.derive_lines(6.5e-6, L, en, w, db)
    rng = np.random.default_rng(5)
    r = rng.normal(size=(2, len(en), ny, nx)).astype(np.float32)
    q = torch.empty_like(_dev(r))
    E.epr_precondition(plan, _dev(r), q)
    q = q.cpu().numpy()
    for b in range(2):
        for s in range(len(en)):
            ref = O.precondition(r[b, s].astype(np.float64), lines.a[s], symbol)
            assert_close(q[b, s], ref, TOL_OP)
    plan.destroy()


@pytest.mark.parametrize("ny,nx", [(256, 256), (160, 96)])
@pytest.mark.parametrize("spec", ["mono", "poly8"])
@pytest.mark.parametrize("order,wkb1", [(2, 1), (2, 0), (1, 0)])
def test_forward_local(E, ny, nx, spec, order, wkb1):
    import torch
    en, w, db = SPECTRA[spec]
    L = 2.0
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "local", max_batch=2, order=order, wkb1=wkb1)
    lines = O.derive_lines(6.5e-6, L, en, w, db)
    tau = np.stack([_tau_field(ny, nx, 1), _tau_field(ny, nx, 2, amp=0.3)])
    P = torch.empty((2, ny, nx), device="cuda")
    Pb = torch.empty((2, len(en), ny, nx), device="cuda")
    E.epr_forward(plan, _dev(tau), P, Pb)
    P, Pb = P.cpu().numpy(), Pb.cpu().numpy()
    for b in range(2):
        ref, ref_bins, _ = O.forward(tau[b].astype(np.float64), lines, "local", order=order, wkb1=bool(wkb1))
        assert_close(P[b], ref, TOL_OP)
        assert rel_l2(P[b] - 1.0, ref - 1.0) < 20 * TOL_OP       # the propagation signal itself
        for s in range(len(en)):
            assert_close(Pb[b, s], ref_bins[s], TOL_OP)
    plan.destroy()


@pytest.mark.parametrize("ny,nx", [(256, 256), (160, 96)])
@pytest.mark.parametrize("spec,L", [("mono", 30.0), ("poly8", 60.0)])
def test_forward_nonlocal_splat_mass_and_adjoint(E, ny, nx, spec, L):
    import torch
    en, w, db = SPECTRA[spec]
    nb = len(en)
    S = 12.0
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "nonlocal", max_batch=2, max_shift_px=S)
    lines = O.derive_lines(6.5e-6, L, en, w, db)
    tau = np.stack([_tau_field(ny, nx, 3, amp=0.2), _tau_field(ny, nx, 4, amp=0.6)])
    P = torch.empty((2, ny, nx), device="cuda")
    Pb = torch.empty((2, nb, ny, nx), device="cuda")
    E.epr_forward(plan, _dev(tau), P, Pb)
    Ph, Pbh = P.cpu().numpy(), Pb.cpu().numpy()
    rng = np.random.default_rng(9)
    e = rng.normal(size=(2, nb, ny, nx)).astype(np.float32)
    x = rng.uniform(0.0, 2.0, size=(2, nb, ny, nx)).astype(np.float32)
    r = torch.empty_like(Pb)
    E.epr_adjoint(plan, _dev(e), r)
    Mx = torch.empty_like(Pb)
    E.epr_transport(plan, _dev(x), Mx)
    rh, Mxh = r.cpu().numpy(), Mx.cpu().numpy()
    saw_multi_pixel = False
    for b in range(2):
        ref, ref_bins, maps = O.forward(tau[b].astype(np.float64), lines, "nonlocal", S=S)
        Is = O.line_intensities(tau[b].astype(np.float64), lines)
        assert_close(Ph[b], ref, TOL_OP)
        # the propagation signal itself, P − Σ_s f_s (Σ f_s = 1): 1e-5 of ‖P‖ would be ~1e-3 of it on a weak object
        assert rel_l2(Ph[b] - 1.0, ref - 1.0) < 20 * TOL_OP
        for s in range(nb):
            saw_multi_pixel |= max(np.abs(maps[s][0]).max(), np.abs(maps[s][1]).max()) > 2.0
            assert_close(Pbh[b, s], ref_bins[s], TOL_OP)
            # mass conservation of the GPU splat (north_star: <= 1e-6 relative)
            assert abs(Pbh[b, s].astype(np.float64).sum() - Is[s].sum()) <= TOL_MASS * Is[s].sum()
            assert_close(rh[b, s], O.gather(e[b, s].astype(np.float64), *maps[s]), TOL_OP)
            assert_close(Mxh[b, s], O.splat(x[b, s].astype(np.float64), *maps[s]), TOL_OP)
        # <Mx, y> = <x, M*y> on the device results
        lhs = float(np.sum(Mxh[b].astype(np.float64) * e[b]))
        rhs = float(np.sum(x[b].astype(np.float64) * rh[b]))
        assert abs(lhs - rhs) <= 1e-5 * np.sqrt(np.sum(Mxh[b].astype(np.float64) ** 2) * np.sum(e[b].astype(np.float64) ** 2))
    assert saw_multi_pixel
    plan.destroy()


def test_forward_nonlocal_uniform_large_shift_several_lines(E):
    """Several lines share one list of ring candidates per detector tile (k_splat_tile); a triangle-wave τ gives a
    constant 14-pixel shift on both axes at the strongest line, so that about 2900 ring sources reach every 128x64
    tile — more than the list holds (2048) — and the kernel has to fall back to walking the ring line by line.
    The weaker lines (unequal a_s) reach the tile from a narrower ring.  Result against the oracle, mass included."""
    import torch
    ny = nx = 256
    en, w, db = SPECTRA["poly3_unequal_a"]
    S, c = 16.0, 0.002
    l0 = O.derive_lines(6.5e-6, 1.0, en, w, db)
    L = 14.0 / (c * float(np.max(l0.a * l0.gamma)))            # a_s is linear in L
    lines = O.derive_lines(6.5e-6, L, en, w, db)
    assert abs(float(np.max(lines.a * lines.gamma)) * c - 14.0) < 1e-9
    tri = np.abs(np.arange(nx) - nx / 2)
    tau = (c * (tri[None, :] + tri[:, None]) + 0.05).astype(np.float32)[None]
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "nonlocal", max_batch=1, max_shift_px=S)
    P = torch.empty((1, ny, nx), device="cuda")
    Pb = torch.empty((1, 3, ny, nx), device="cuda")
    E.epr_forward(plan, _dev(tau), P, Pb)
    ref, ref_bins, maps = O.forward(tau[0].astype(np.float64), lines, "nonlocal", S=S)
    Is = O.line_intensities(tau[0].astype(np.float64), lines)
    shifts = sorted(float(np.abs(maps[s][0]).max()) for s in range(3))
    assert shifts[-1] > 13.9 and shifts[0] < 0.8 * shifts[-1]
    assert_close(P.cpu().numpy()[0], ref, TOL_OP)
    for s in range(3):
        got = Pb.cpu().numpy()[0, s]
        assert_close(got, ref_bins[s], TOL_OP)
        assert abs(got.astype(np.float64).sum() - Is[s].sum()) <= TOL_MASS * Is[s].sum()
    plan.destroy()


def test_transport_signed_planes_and_wrap(E):
    """The linear splat accepts planes of either sign (fixed point is signed), and mass that leaves one side of a
    multi-tile grid enters the other (R7): compare with the oracle on a 320 x 320 grid (3 x 5 detector tiles, ragged in x)."""
    import torch
    en, w, db = SPECTRA["mono"]
    ny, nx, S = 320, 320, 9.0
    plan = E.epr_plan(nx, ny, 6.5e-6, 60.0, en, w, db, "nonlocal", max_batch=1, max_shift_px=S)
    lines = O.derive_lines(6.5e-6, 60.0, en, w, db)
    tau = _tau_field(ny, nx, 11, amp=0.8)[None]
    P = torch.empty((1, ny, nx), device="cuda")
    E.epr_forward(plan, _dev(tau), P)
    _, _, maps = O.forward(tau[0].astype(np.float64), lines, "nonlocal", S=S)
    assert max(np.abs(maps[0][0]).max(), np.abs(maps[0][1]).max()) > 4.0
    x = np.random.default_rng(3).normal(size=(1, 1, ny, nx)).astype(np.float32)
    Mx = torch.empty((1, 1, ny, nx), device="cuda")
    E.epr_transport(plan, _dev(x), Mx)
    got = Mx.cpu().numpy()[0, 0]
    ref = O.splat(x[0, 0].astype(np.float64), *maps[0])
    assert_close(got, ref, TOL_OP)
    assert abs(got.astype(np.float64).sum() - x.astype(np.float64).sum()) <= 1e-6 * np.abs(x).sum()
    plan.destroy()


def test_splat_is_deterministic(E):
    """Fixed-point accumulation: two runs give bit-identical planes regardless of atomic ordering."""
    import torch
    en, w, db = SPECTRA["mono"]
    plan = E.epr_plan(256, 256, 6.5e-6, 40.0, en, w, db, "nonlocal", max_batch=1)
    tau = _dev(_tau_field(256, 256, 8, amp=0.5)[None])
    P1 = torch.empty((1, 256, 256), device="cuda")
    P2 = torch.empty_like(P1)
    E.epr_forward(plan, tau, P1)
    E.epr_forward(plan, tau, P2)
    assert torch.equal(P1, P2)
    plan.destroy()


def _run_retrieve(E, w, iterations=None, batch_idx=(0,), **opts):
    import torch
    it = w.iterations if iterations is None else iterations
    plan = E.epr_plan(w.nx, w.ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver,
                      max_batch=len(batch_idx), max_shift_px=w.max_shift_px, **opts)
    d = _dev(w.d[list(batch_idx)])
    out = torch.empty_like(d)
    E.epr_retrieve(plan, d, out, it, w.step)
    torch.cuda.synchronize()
    plan.destroy()
    lines = O.derive_lines(w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    refs = [O.retrieve(w.d[j].astype(np.float64), lines, w.solver, it, w.step, S=w.max_shift_px) for j in batch_idx]
    return out.cpu().numpy(), refs


@pytest.mark.parametrize("name,n", [("C1", None), ("C2", 512), ("C3", 512), ("C4", 256), ("C5", (160, 320))])
def test_retrieve_parity(E, name, n):
    """Retrieved phase after the stated iteration count within 1e-4 relative L2 (phase ∝ τ, Eq. (6))."""
    w = make_workload(name, n=n, batch=2 if name == "C5" else 1)
    got, refs = _run_retrieve(E, w, batch_idx=tuple(range(w.batch)))
    for j, ref in enumerate(refs):
        assert_close(got[j], ref, TOL_PHASE)


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_full_size_periodic_tiling(E, name):
    """Full-size grids of BASELINE.json (2048 x 2048; C5: 2560 x 2160), in the launch configuration bench.py times
    (batched epr_retrieve, 20 iterations).  Every operator is periodic on the (nx, ny) grid (R7), so the retrieval of a
    k x k tiling of a small detector image is the k x k tiling of its small retrieval — which the oracle computes in
    seconds (C2-C4: 4 x 4 tiles of 512 x 512; C5: 8 x 8 tiles of 270 x 320 = 2160 rows x 2560 columns, 8 lines, S = 24).
    Checked on every pixel; the full-size transforms (2048 / 2160 / 2560 points), the TMA column kernels and the
    multi-tile splat all differ from the small path."""
    import torch
    tile, k = ((270, 320), 8) if name == "C5" else (512, 4)
    w = make_workload(name, n=tile, batch=1)
    lines = O.derive_lines(w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    ref = O.retrieve(w.d[0].astype(np.float64), lines, w.solver, w.iterations, w.step, S=w.max_shift_px)
    big = np.tile(w.d[0], (k, k))[None]
    ny, nx = big.shape[1:]
    assert (ny, nx) == ((2160, 2560) if name == "C5" else (2048, 2048))
    # one line: a batch of 8 selects the kernels bench.py's batch of 64 runs (128-row march, two-group column kernel:
    # both need a launch that fills the GPU); 8 lines: a batch of 2 already does
    nbatch = 8 if w.n_bins == 1 else 2
    d = _dev(np.concatenate([big] * nbatch))
    plan = E.epr_plan(nx, ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver,
                      max_batch=nbatch, max_shift_px=w.max_shift_px)
    out = torch.empty_like(d)
    E.epr_retrieve(plan, d, out, w.iterations, w.step)
    got = out.cpu().numpy()
    plan.destroy()
    assert_close(got[0], np.tile(ref, (k, k)), TOL_PHASE, f"{name} full size")
    for j in range(1, nbatch):
        assert np.array_equal(got[0], got[j])                  # batch entries are independent and deterministic


def test_retrieve_graph_replay_matches_eager(E):
    """On a non-default stream a launch-bound retrieval is captured into a CUDA graph (second call) and replayed
    (third call, with NEW data in the same buffers): all three must equal the eager result bit for bit."""
    import torch
    w = make_workload("C1")
    w2 = make_workload("C3", n=256)
    for wk in (w, w2):
        plan = E.epr_plan(wk.nx, wk.ny, wk.pixel_m, wk.L_m, wk.energy_keV, wk.weight, wk.delta_over_beta, wk.solver,
                          max_batch=1, max_shift_px=wk.max_shift_px)
        d = _dev(wk.d[:1])
        ref = torch.empty_like(d)
        E.epr_retrieve(plan, d, ref, wk.iterations, wk.step)            # default stream: eager
        d_alt = _dev(np.roll(wk.d[:1], 5, axis=2))
        ref_alt = torch.empty_like(d)
        E.epr_retrieve(plan, d_alt, ref_alt, wk.iterations, wk.step)
        torch.cuda.synchronize()
        side = torch.cuda.Stream()
        out = torch.empty_like(d)
        buf = d.clone()
        l0 = plan.launches
        with torch.cuda.stream(side):
            E.epr_retrieve(plan, buf, out, wk.iterations, wk.step)      # eager warm pass
            side.synchronize()
            per_call = plan.launches - l0
            assert torch.equal(out, ref)
            out.zero_()
            E.epr_retrieve(plan, buf, out, wk.iterations, wk.step)      # capture + launch
            side.synchronize()
            assert torch.equal(out, ref)
            buf.copy_(d_alt)
            E.epr_retrieve(plan, buf, out, wk.iterations, wk.step)      # replay on new contents
            side.synchronize()
            assert torch.equal(out, ref_alt)
        assert plan.launches - l0 == 3 * per_call
        plan.destroy()


def test_retrieve_zero_iterations_is_paganin(E):
    w = make_workload("C1")
    got, refs = _run_retrieve(E, w, iterations=0)
    assert_close(got[0], refs[0], TOL_OP)


def test_retrieve_unequal_a_lines(E):
    """The implementation must not rely on 'all a_s equal' (a coincidence of C4/C5): db_s constant here."""
    w = make_workload("C4", n=256)
    w.delta_over_beta = np.full(8, 200.0)
    got, refs = _run_retrieve(E, w, iterations=8)
    assert_close(got[0], refs[0], TOL_PHASE)


@pytest.mark.parametrize("n_lines", [3, 5, 10])
def test_retrieve_other_line_counts(E, n_lines):
    """Line counts other than 8: 5 and 10 lines (the paper's own runs) take the unrolled small-step
    projection, 3 lines the general routine; the gather tile kernel and the fused residual split serve all of them.
    The detector image is C4's; only the retrieval's spectral discretisation changes."""
    w = make_workload("C4", n=256)
    e = np.linspace(60.0, 140.0, n_lines)
    wt = np.exp(-0.5 * ((e - 100.0) / 20.0) ** 2)
    w.energy_keV, w.weight, w.delta_over_beta = e, wt / wt.sum(), 200.0 * e / 100.0
    got, refs = _run_retrieve(E, w, iterations=8)
    assert_close(got[0], refs[0], TOL_PHASE)


@pytest.mark.parametrize("name,n,m,S", [("C1", None, 2, 16.0), ("C2", 256, 2, 16.0), ("C3", 128, 4, 28.0), ("C4", 128, 2, 24.0)])
def test_retrieve_oversampled_parity(E, name, n, m, S):
    """PAPER.md:79 (reading R16): the loop on the grid refined m times (2 for the local solver, 4 for the non-local
    one), plan built for the fine pixel; replication in, block mean out.  S counts fine pixels."""
    import torch
    w = make_workload(name, n=n, batch=2)
    plan = E.epr_plan(m * w.nx, m * w.ny, w.pixel_m / m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver,
                      max_batch=2, max_shift_px=S)
    d = _dev(w.d)
    out = torch.empty_like(d)
    E.epr_retrieve_oversampled(plan, m, d, out, w.iterations, w.step)
    got = out.cpu().numpy()
    plan.destroy()
    lines = O.derive_lines(w.pixel_m / m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    for j in range(2):
        ref = O.retrieve_oversampled(w.d[j].astype(np.float64), lines, m, w.solver, w.iterations, w.step, S=S)
        assert got[j].shape == ref.shape == (w.ny, w.nx)
        assert_close(got[j], ref, TOL_PHASE)


def test_resampling_round_trip_is_exact(E):
    """Zero iterations of a plan whose filter is the identity (L -> 0): out = −ln(block mean … ) is not exact, so the
    round trip is checked on the intensity output instead: output = 2 returns T = e^{−τ}; with a vanishing propagation
    distance the Paganin solve is the identity and mean(replicate(d)) = d up to the fp32 rounding of exp/log."""
    import torch
    rng = np.random.default_rng(5)
    dn = (1.0 + 0.2 * rng.uniform(-1, 1, size=(2, 40, 64))).astype(np.float32)      # fine grids 80 x 128, 160 x 256
    for m in (2, 4):
        plan = E.epr_plan(m * 64, m * 40, 6.5e-6 / m, 1e-9, [100.0], [1.0], [1000.0], "local", max_batch=2, output=2)
        d = _dev(dn)
        out = torch.empty_like(d)
        E.epr_retrieve_oversampled(plan, m, d, out, 0, 1.0)
        plan.destroy()
        assert np.max(np.abs(out.cpu().numpy() - dn)) < 5e-7


@pytest.mark.parametrize("ny,nx,n_lines", [(2160, 32, 3), (2160, 64, 8), (320, 64, 5), (2560, 32, 3), (4096, 32, 3), (32, 4096, 1)])
def test_retrieve_non_power_of_two_columns_several_lines(E, ny, nx, n_lines):
    """The Fourier-space sum over lines (R10) on column lengths that are not powers of two: 2160 and 320 take the
    TMA-staged padded column kernel with two tiles in flight, 2560 (two tiles would not fit an SM) the direct one; 4096
    rows (the x2 oversampled grid of a 2048 detector) with several lines take the direct kernel as well, 4096 columns the
    2048-point row transforms."""
    import torch
    rng = np.random.default_rng(ny + nx + n_lines)
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    d = 1.0 + sum(0.02 * rng.normal() * np.cos(rng.integers(1, 9) * y + rng.integers(0, 4) * x + rng.uniform(0, 6.28))
                  for _ in range(8)) + 0.003 * rng.normal(size=(ny, nx))
    d = d.astype(np.float32)[None]
    e = np.linspace(60.0, 140.0, n_lines)
    wt = np.exp(-0.5 * ((e - 100.0) / 20.0) ** 2)
    db = 1000.0 * e / 100.0
    plan = E.epr_plan(nx, ny, 6.5e-6, 0.5, e, wt, db, "local", max_batch=1)
    dd = _dev(d)
    out = torch.empty_like(dd)
    E.epr_retrieve(plan, dd, out, 4, 1.0)
    got = out.cpu().numpy()[0]
    plan.destroy()
    lines = O.derive_lines(6.5e-6, 0.5, e, wt, db)
    ref = O.retrieve(d[0].astype(np.float64), lines, "local", 4, 1.0)
    assert_close(got, ref, TOL_PHASE)


@pytest.mark.parametrize("name,n", [("C1", None), ("C3", 256), ("C4", 128)])
def test_diagnostics_history(E, name, n):
    """epr_set_diagnostics: residual RMS and largest unclamped shift per iteration against the oracle's histories
    (PAPER.md:53-55, 231); switching it off restores the plain result bit for bit."""
    import torch
    w = make_workload(name, n=n, batch=2)
    plan = E.epr_plan(w.nx, w.ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver,
                      max_batch=2, max_shift_px=w.max_shift_px)
    d = _dev(w.d)
    out = torch.empty_like(d)
    diag = torch.zeros(2, w.iterations, 2, device="cuda")
    E.epr_set_diagnostics(plan, diag)
    E.epr_retrieve(plan, d, out, w.iterations, w.step)
    got = diag.cpu().numpy()
    # the host path works through the batch in chunks: every chunk must land in its own rows of the array
    diag_h = torch.zeros_like(diag)
    E.epr_set_diagnostics(plan, diag_h)
    dh = torch.from_numpy(w.d).pin_memory()
    oh = torch.empty_like(dh).pin_memory()
    E.epr_retrieve_host(plan, dh, oh, w.iterations, w.step)
    assert torch.equal(diag_h, diag) and torch.equal(oh.cuda(), out)
    E.epr_set_diagnostics(plan, None)
    out2 = torch.empty_like(d)
    E.epr_retrieve(plan, d, out2, w.iterations, w.step)
    assert torch.equal(out, out2)
    plan.destroy()
    lines = O.derive_lines(w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    for j in range(2):
        h, sh = [], []
        O.retrieve(w.d[j].astype(np.float64), lines, w.solver, w.iterations, w.step, S=w.max_shift_px, history=h,
                   shift_history=sh)
        h, sh = np.array(h), np.array(sh)
        assert np.max(np.abs(got[j, :, 0] - h)) < 2e-3 * h[0]          # e is a small difference of O(1) planes in fp32
        assert np.max(np.abs(got[j, :, 1] - sh) / sh) < 1e-3


@pytest.mark.parametrize("ny,nx,n_lines", [(16, 16, 1), (32, 48, 3), (48, 16, 8), (80, 160, 5)])
def test_retrieve_nonlocal_grids_smaller_than_a_tile(E, ny, nx, n_lines):
    """Grids smaller than one 128 x 64 detector tile, started (opt.init = 1) from a τ⁰ whose shifts span several pixels
    and hit the clamp: every source reaches the tile through several periodic images (R7), the block-maximum samples
    and the staged residual rows wrap more than once."""
    import torch
    rng = np.random.default_rng(100 * ny + nx)
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    d = (1.0 + 0.15 * np.cos(y + 0.3) * np.sin(2 * x) + 0.1 * np.cos(3 * y - x) + 0.01 * rng.normal(size=(ny, nx)))
    d = d.astype(np.float32)[None]
    tau0 = (0.12 * (1.0 + np.cos(y + 1.0) * np.cos(x)) + 0.05 * np.sin(2 * y + x)).astype(np.float32)[None]
    e = np.linspace(60.0, 140.0, n_lines) if n_lines > 1 else np.array([100.0])
    wt = np.exp(-0.5 * ((e - 100.0) / 20.0) ** 2)
    db = 200.0 * e / 100.0
    L_m, S, its = 40.0, 6.0, 2
    lines = O.derive_lines(6.5e-6, L_m, e, wt, db)
    assert O.max_shift(tau0[0].astype(np.float64), lines) > S        # several pixels, some clamped
    ref = O.retrieve(d[0].astype(np.float64), lines, "nonlocal", its, 0.4, S=S, tau0=tau0[0].astype(np.float64))
    plan = E.epr_plan(nx, ny, 6.5e-6, L_m, e, wt, db, "nonlocal", max_batch=1, max_shift_px=S, init=1)
    out = _dev(tau0.copy())
    E.epr_retrieve(plan, _dev(d), out, its, 0.4)
    got = out.cpu().numpy()[0]
    plan.destroy()
    assert_close(got, ref, TOL_PHASE)


def test_nonlocal_wkb1_variant(E):
    """opt.nonlocal_wkb1 (variant of R4): forward model and retrieval with the WKB1 term of Eq. (1) added
    to the ray-map prediction, at a δ/β small enough for the term to matter."""
    import torch
    ny, nx, S = 160, 96, 8.0
    en, wt, db = np.array([80.0, 100.0, 120.0]), np.array([0.3, 0.4, 0.3]), np.array([8.0, 10.0, 12.0])
    lines = O.derive_lines(6.5e-6, 20.0, en, wt, db)
    tau = _tau_field(ny, nx, 5, amp=0.3)[None]
    plan = E.epr_plan(nx, ny, 6.5e-6, 20.0, en, wt, db, "nonlocal", max_batch=1, max_shift_px=S, nonlocal_wkb1=1)
    P = torch.empty((1, ny, nx), device="cuda")
    Pb = torch.empty((1, 3, ny, nx), device="cuda")
    E.epr_forward(plan, _dev(tau), P, Pb)
    ref, ref_bins, _ = O.forward(tau[0].astype(np.float64), lines, "nonlocal", S=S, nonlocal_wkb1=True)
    plain, _, _ = O.forward(tau[0].astype(np.float64), lines, "nonlocal", S=S)
    assert rel_l2(ref, plain) > 100 * TOL_OP                         # the term is far above the tolerance here
    assert_close(P.cpu().numpy()[0], ref, TOL_OP)
    for s in range(3):
        assert_close(Pb.cpu().numpy()[0, s], ref_bins[s], TOL_OP)
    d = np.float32(ref + 0.002 * np.random.default_rng(3).normal(size=ref.shape))[None]
    out = torch.empty((1, ny, nx), device="cuda")
    E.epr_retrieve(plan, _dev(d), out, 5, 0.4)
    plan.destroy()
    want = O.retrieve(d[0].astype(np.float64), lines, "nonlocal", 5, 0.4, S=S, nonlocal_wkb1=True)
    assert_close(out.cpu().numpy()[0], want, TOL_PHASE)


def test_retrieve_outputs_and_host_path(E):
    import torch
    w = make_workload("C1")
    lines = O.derive_lines(w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    ref = O.retrieve(w.d[0].astype(np.float64), lines, w.solver, w.iterations, w.step)
    got_phi, _ = _run_retrieve(E, w, output=1)
    assert_close(got_phi[0], O.phase(ref, lines), TOL_PHASE)
    plan = E.epr_plan(w.nx, w.ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver, max_batch=2)
    d3 = np.concatenate([w.d, w.d, w.d]).astype(np.float32)          # batch 3 > max_batch 2: chunked + double buffered
    dh = torch.from_numpy(d3).pin_memory()
    oh = torch.empty_like(dh).pin_memory()
    E.epr_retrieve_host(plan, dh, oh, w.iterations, w.step)
    for j in range(3):
        assert_close(oh[j].numpy(), ref, TOL_PHASE)
    plan.destroy()


@pytest.mark.parametrize("name", ["C3", "C4"])
def test_retrieve_device_batch_larger_than_the_work_batch(E, name, monkeypatch):
    """epr_retrieve on DEVICE buffers with batch > the plan's work batch (what bench.py's C5 sub-result times: 64 projections
    in passes of 16): EPR_WORK_BATCH = 2 at plan time, batch 5 → passes of 2, 2, 1, each projection against the oracle."""
    import torch
    w = make_workload(name, n=128, batch=5)
    monkeypatch.setenv("EPR_WORK_BATCH", "2")
    plan = E.epr_plan(w.nx, w.ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver,
                      max_batch=5, max_shift_px=w.max_shift_px)
    monkeypatch.delenv("EPR_WORK_BATCH")
    d = _dev(w.d)
    out = torch.empty_like(d)
    E.epr_retrieve(plan, d, out, w.iterations, w.step)
    got = out.cpu().numpy()
    # the same call on a plan whose work batch holds everything: the passes change nothing, bit for bit
    whole = E.epr_plan(w.nx, w.ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver,
                       max_batch=5, max_shift_px=w.max_shift_px)
    out2 = torch.empty_like(d)
    E.epr_retrieve(whole, d, out2, w.iterations, w.step)
    assert torch.equal(out, out2)
    plan.destroy()
    whole.destroy()
    lines = O.derive_lines(w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    for j in range(5):
        ref = O.retrieve(w.d[j].astype(np.float64), lines, w.solver, w.iterations, w.step, S=w.max_shift_px)
        assert_close(got[j], ref, TOL_PHASE, f"{name} projection {j}")


@pytest.mark.parametrize("solver", ["local", "nonlocal"])
def test_retrieve_host_with_caller_supplied_start(E, solver):
    """epr_retrieve_host with opt.init = 1: out_host holds τ⁰ on entry and travels to the device beside d in every chunk
    (batch 5 > max_batch 2: three chunks)."""
    import torch
    w = make_workload("C3" if solver == "nonlocal" else "C1", n=128, batch=5)
    rng = np.random.default_rng(9)
    y, x = np.meshgrid(np.arange(w.ny) * 2 * np.pi / w.ny, np.arange(w.nx) * 2 * np.pi / w.nx, indexing="ij")
    tau0 = np.stack([(0.02 + 0.01 * j) * (1.0 + np.cos(x + j) * np.sin(2 * y)) + 0.001 * rng.normal(size=x.shape)
                     for j in range(5)]).astype(np.float32)
    its, step = 3, 0.3                                                    # under-relaxed: the start is still visible
    plan = E.epr_plan(w.nx, w.ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, solver, max_batch=2,
                      max_shift_px=w.max_shift_px, init=1)
    dh = torch.from_numpy(w.d).pin_memory()
    oh = torch.from_numpy(tau0.copy()).pin_memory()
    E.epr_retrieve_host(plan, dh, oh, its, step)
    plan.destroy()
    lines = O.derive_lines(w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    for j in range(5):
        ref = O.retrieve(w.d[j].astype(np.float64), lines, solver, its, step, S=w.max_shift_px,
                         tau0=tau0[j].astype(np.float64))
        start = O.retrieve(w.d[j].astype(np.float64), lines, solver, its, step, S=w.max_shift_px)
        assert rel_l2(ref, start) > 10 * TOL_PHASE                     # the start matters after 3 iterations
        assert_close(oh[j].numpy(), ref, TOL_PHASE, f"{solver} projection {j}")


@pytest.mark.parametrize("name", ["C1", "C3"])
def test_host_streaming_session_and_multi_plan(E, name):
    """epr_retrieve_host_async / epr_host_wait (the next chunk is prepared while the current one is processed):
    three batches of different sizes enqueued back to back, one wait — every result equals the plain epr_retrieve_host call
    bit for bit (same chunks, same kernels; only the waiting differs), and so does a plain call that follows an open session.
    epr_retrieve_host_multi: ONE host batch over two plans (here both on this GPU; one per device in production) — plan 0
    gets projections [0, 3), plan 1 [3, 5), the split of epr_inputs.shard_range — again the same bits."""
    import torch
    from epr_inputs import shard_range
    w = make_workload(name, n=128, batch=11)
    its = 4
    mk = lambda mb: E.epr_plan(w.nx, w.ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver,
                               max_batch=mb, max_shift_px=w.max_shift_px)
    plan = mk(2)
    dh = torch.from_numpy(w.d).pin_memory()
    want = torch.empty_like(dh).pin_memory()
    E.epr_retrieve_host(plan, dh, want, its, w.step)
    lines = O.derive_lines(w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    ref = O.retrieve(w.d[10].astype(np.float64), lines, w.solver, its, w.step, S=w.max_shift_px)
    assert_close(want[10].numpy(), ref, TOL_PHASE)
    got = torch.full_like(dh, float("nan")).pin_memory()
    for a, b in ((0, 5), (5, 6), (6, 11)):                              # 5, 1 and 5 projections: 3 + 1 + 3 chunks of <= 2
        E.epr_retrieve_host(plan, dh[a:b], got[a:b], its, w.step, wait=False)
    E.epr_host_wait(plan)
    assert torch.equal(got, want)
    got2 = torch.full_like(dh, float("nan")).pin_memory()
    E.epr_retrieve_host(plan, dh[:4], got2[:4], its, w.step, wait=False)   # session left open …
    E.epr_retrieve_host(plan, dh[4:], got2[4:], its, w.step)               # … a plain call closes it first
    assert torch.equal(got2, want)
    E.epr_host_wait(plan)                                                   # nothing open: returns at once
    other = mk(2)
    got3 = torch.full((5, w.ny, w.nx), float("nan")).pin_memory()
    E.epr_retrieve_host_multi([plan, other], dh[:5], got3, its, w.step)
    assert shard_range(5, 0, 2) == (0, 3) and shard_range(5, 1, 2) == (3, 5)
    assert torch.equal(got3, want[:5])
    got4 = torch.full((1, w.ny, w.nx), float("nan")).pin_memory()          # fewer projections than plans: plan 1 idles
    E.epr_retrieve_host_multi([plan, other], dh[7:8], got4, its, w.step)
    assert torch.equal(got4, want[7:8])
    plan.destroy()
    other.destroy()


def test_argument_errors(E):
    import torch
    en, w, db = SPECTRA["mono"]
    with pytest.raises(E.EprError) as ei:
        E.epr_plan(224, 256, 6.5e-6, 1.0, en, w, db)            # 224 = 2⁵·7: a prime factor outside {2, 3, 5}
    assert ei.value.status == 2
    with pytest.raises(E.EprError):
        E.epr_plan(256, 256, -1.0, 1.0, en, w, db)
    plan = E.epr_plan(256, 256, 6.5e-6, 1.0, en, w, db, max_batch=1)
    d = torch.ones((2, 256, 256), device="cuda")
    with pytest.raises(E.EprError):
        E.epr_retrieve(plan, d, torch.empty_like(d), 1, 1.0)   # batch > max_batch
    d = torch.ones((1, 256, 256), device="cuda")
    with pytest.raises(E.EprError):
        E.epr_retrieve(plan, d, torch.empty_like(d), 1, 0.0)   # step <= 0
    plan.destroy()


# ---------------------------------------------------------------------------------------------------------------------
# Branches and options no workload reaches by itself: split fallback (den <= 0), positivity floor, mu_rel, i_min,
# newton_iters, out_bin, chunked epr_forward, the ragged gather tile.
# ---------------------------------------------------------------------------------------------------------------------
def _fallback_floor_case():
    """Local solver, 3 unequal lines, started from a τ⁰ with isolated spikes (the closure undershoots there: every
    P_s < 0, so the split falls back to f_s) on data with two pixels forced to −3 (the update drives Σ_s I_s below
    i_min there: the floor binds)."""
    E_, wt, db = np.array([70.0, 100.0, 130.0]), np.array([0.3, 0.45, 0.25]), np.array([600.0, 1000.0, 1500.0])
    ny, nx, L = 96, 160, 0.02
    rng = np.random.default_rng(1)
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    tau0 = 0.3 + 0.1 * np.cos(2 * x) * np.sin(y)
    for yy, xx in ((10, 20), (50, 130), (95, 159), (0, 0)):
        tau0[yy, xx] += 1.5
    d = 1.0 + 0.05 * np.cos(x + y) + 0.01 * rng.normal(size=(ny, nx))
    d[30, 40] = d[31, 40] = -3.0
    return E_, wt, db, L, tau0.astype(np.float32), d.astype(np.float32)


def test_split_fallback_and_positivity_floor_local(E):
    import torch
    E_, wt, db, L, tau0, d = _fallback_floor_case()
    i_min = 1e-3
    lines = O.derive_lines(6.5e-6, L, E_, wt, db)
    _, Pb, _ = O.forward(tau0.astype(np.float64), lines, "local")
    den = np.sum([np.maximum(p, 0.0) for p in Pb], axis=0)
    assert (den <= 0).sum() >= 4                                    # the fallback w_s = f_s is taken (R8)
    for its in (1, 2):
        ref = O.retrieve(d.astype(np.float64), lines, "local", its, 1.0, i_min=i_min, tau0=tau0.astype(np.float64))
        T = np.sum(O.line_intensities(ref, lines), axis=0)
        assert (np.abs(T - i_min) < 1e-12).sum() >= 2               # the floor binds
        plan = E.epr_plan(160, 96, 6.5e-6, L, E_, wt, db, "local", max_batch=1, init=1, i_min=i_min, newton_iters=12)
        out = _dev(tau0[None].copy())
        E.epr_retrieve(plan, _dev(d[None]), out, its, 1.0)
        got = out.cpu().numpy()[0]
        plan.destroy()
        assert np.all(np.isfinite(got))
        assert_close(got, ref, TOL_PHASE, f"fallback/floor, {its} iteration(s)")
        floor_px = np.abs(T - i_min) < 1e-12
        assert np.max(np.abs(got[floor_px] - ref[floor_px])) < 1e-4 * np.max(ref[floor_px])


def test_split_fallback_in_detector_holes_nonlocal(E):
    """Non-local solver: where a caustic leaves detector pixels EMPTY (every P_s = 0 exactly) the split must take the
    fallback w_s = f_s on the device too — the decision 'P_s⁺ sums to zero' is taken on the integer accumulators, not on
    a float that rounding made ±1e-8.  Triangle-wave τ⁰: sources move apart at the ridge lines."""
    import torch
    en, w, db = SPECTRA["poly3_unequal_a"]
    ny = nx = 128
    S, c = 16.0, 0.002
    l0 = O.derive_lines(6.5e-6, 1.0, en, w, db)
    L = 6.0 / (c * float(np.max(l0.a * l0.gamma)))
    lines = O.derive_lines(6.5e-6, L, en, w, db)
    tri = np.abs(np.arange(nx) - nx / 2)
    tau0 = (c * (tri[None, :] + tri[:, None]) + 0.05).astype(np.float32)
    _, Pb, _ = O.forward(tau0.astype(np.float64), lines, "nonlocal", S=S)
    holes = np.sum([np.maximum(p, 0.0) for p in Pb], axis=0) <= 0
    assert holes.sum() > 100
    rng = np.random.default_rng(2)
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    d = (1 + 0.1 * np.cos(x) * np.cos(2 * y) + 0.01 * rng.normal(size=(ny, nx))).astype(np.float32)
    ref = O.retrieve(d.astype(np.float64), lines, "nonlocal", 2, 0.4, S=S, tau0=tau0.astype(np.float64))
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "nonlocal", max_batch=1, max_shift_px=S, init=1)
    out = _dev(tau0[None].copy())
    E.epr_retrieve(plan, _dev(d[None]), out, 2, 0.4)
    got = out.cpu().numpy()[0]
    plan.destroy()
    # the update is what the split decides; compare it, not τ (which it changes by a few per cent only)
    assert_close(got - tau0, ref - tau0, 10 * TOL_PHASE, "update over detector holes")
    assert_close(got, ref, TOL_PHASE)


@pytest.mark.parametrize("solver,step,L", [("local", 1.0, 0.3), ("nonlocal", 0.4, 8.0)])
def test_options_mu_rel_out_bin_i_min(E, solver, step, L):
    """opt.mu_rel overrides the derived γ_s (R11), opt.output = 1 with out_bin ≠ 0 returns the phase of THAT line
    (Eq. (6)), opt.i_min moves the floor (it binds on a tenth of the pixels of the local case): each
    against the oracle given the same values."""
    import torch
    en, wt, db = SPECTRA["poly3_unequal_a"]
    ny, nx, S, i_min, mu = 96, 160, 8.0, 0.7, [3.0, 1.0, 0.3]
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    rng = np.random.default_rng(3)
    d = (0.85 + 0.2 * np.cos(x) * np.sin(2 * y) + 0.08 * np.cos(3 * x - y) + 0.003 * rng.normal(size=(ny, nx))).astype(np.float32)
    lines = O.derive_lines(6.5e-6, L, en, wt, db, mu_rel=mu)
    ref = O.retrieve(d.astype(np.float64), lines, solver, 4, step, S=S, i_min=i_min)
    plain = O.retrieve(d.astype(np.float64), O.derive_lines(6.5e-6, L, en, wt, db), solver, 4, step, S=S, i_min=i_min)
    assert rel_l2(ref, plain) > 100 * TOL_PHASE            # mu_rel matters at this tolerance
    if solver == "local":
        T = np.sum(O.line_intensities(ref, lines), axis=0)
        assert (np.abs(T - i_min) < 1e-12).sum() > 500     # … and so does the floor
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, wt, db, solver, max_batch=1, max_shift_px=S, mu_rel=mu, i_min=i_min,
                      output=1, out_bin=2)
    assert np.allclose(plan.lines()["gamma"], lines.gamma, rtol=1e-12)
    dd = _dev(d[None])
    out = torch.empty_like(dd)
    E.epr_retrieve(plan, dd, out, 4, step)
    got = out.cpu().numpy()[0]
    plan.destroy()
    assert_close(got, O.phase(ref, lines, s=2), TOL_PHASE, "phase of line 2 with mu_rel and i_min")
    assert rel_l2(got, O.phase(ref, lines, s=0)) > 0.05    # not the phase of line 0


def test_option_newton_iters(E):
    """opt.newton_iters bounds the Newton steps of the single-thickness projection (R10).  On a start far from the
    data (thick object, init = 1 from τ⁰ = 0) the general routine is taken: many steps reproduce the oracle's converged
    projection; zero steps leave the first-order guess, which is measurably different."""
    import torch
    en, wt, db = SPECTRA["poly3_unequal_a"]
    ny, nx, L = 64, 96, 0.5
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    d = (0.45 + 0.35 * np.cos(x) * np.sin(2 * y)).astype(np.float32)            # transmission down to 0.1
    lines = O.derive_lines(6.5e-6, L, en, wt, db, mu_rel=[3.0, 1.0, 0.3])
    ref = O.retrieve(d.astype(np.float64), lines, "local", 1, 1.0, tau0=np.zeros((ny, nx)))
    res = {}
    for ni in (0, 16):
        plan = E.epr_plan(nx, ny, 6.5e-6, L, en, wt, db, "local", max_batch=1, init=1, newton_iters=ni, mu_rel=[3.0, 1.0, 0.3])
        out = torch.zeros((1, ny, nx), device="cuda")
        E.epr_retrieve(plan, _dev(d[None]), out, 1, 1.0)
        res[ni] = out.cpu().numpy()[0]
        plan.destroy()
    assert_close(res[16], ref, TOL_PHASE, "newton_iters = 16")
    assert rel_l2(res[0], ref) > 10 * TOL_PHASE


def test_forward_chunked_over_work_batch(E, monkeypatch):
    """epr_forward / epr_adjoint / epr_transport accept any batch <= max_batch even when the plan's workspaces hold
    fewer projections (EPR_WORK_BATCH = 2 here, batch 5): chunked inside the call, ray map kept for the whole batch."""
    import torch
    monkeypatch.setenv("EPR_WORK_BATCH", "2")
    en, w, db = SPECTRA["poly3_unequal_a"]
    ny, nx, S, L = 64, 160, 8.0, 40.0
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "nonlocal", max_batch=5, max_shift_px=S)
    monkeypatch.delenv("EPR_WORK_BATCH")
    lines = O.derive_lines(6.5e-6, L, en, w, db)
    tau = np.stack([_tau_field(ny, nx, 20 + j, amp=0.1 * (j + 1)) for j in range(5)])
    P = torch.empty((5, ny, nx), device="cuda")
    Pb = torch.empty((5, 3, ny, nx), device="cuda")
    E.epr_forward(plan, _dev(tau), P, Pb)
    e = np.random.default_rng(1).normal(size=(5, 3, ny, nx)).astype(np.float32)
    r = torch.empty_like(Pb)
    E.epr_adjoint(plan, _dev(e), r)
    Ph, rh = P.cpu().numpy(), r.cpu().numpy()
    plan.destroy()
    for b in range(5):
        ref, _, maps = O.forward(tau[b].astype(np.float64), lines, "nonlocal", S=S)
        assert_close(Ph[b], ref, TOL_OP)
        for s in range(3):
            assert_close(rh[b, s], O.gather(e[b, s].astype(np.float64), *maps[s]), TOL_OP)


def test_gather_ragged_tile_with_large_shift_at_column_zero(E):
    """nx = 160: the second 128-column gather tile is ragged (32 live columns).  Column 0 alone carries a period-4
    pattern in y: its y-shift reaches ±12 px at the strongest line while the ragged tile only sees the ±6 px x-shift
    of column 159 (halo 7 <= 8: served from the staged tile).  The ragged tile's idle threads must not pick up column
    0's shift — they would address 12 rows outside the staged tile.  (compute-sanitizer is closed on this pool, so the out-of-range
    read cannot be shown by the tool; the kernel zeroes the shifts of out-of-image pixels and this case pins the result.)"""
    import torch
    en, w, db = SPECTRA["poly3_unequal_a"]
    ny, nx, S, eps = 128, 160, 16.0, 0.01
    tau = np.full((ny, nx), 0.05, dtype=np.float32)
    tau[:, 0] += eps * np.array([0.0, 1.0, 0.0, -1.0], dtype=np.float32)[np.arange(ny) % 4]
    l0 = O.derive_lines(6.5e-6, 1.0, en, w, db)
    L = 12.0 / (eps * float(np.max(l0.a * l0.gamma)))
    lines = O.derive_lines(6.5e-6, L, en, w, db)
    yy = np.arange(ny)[:, None]
    xx = np.arange(nx)[None, :]
    d = (1.0 + 0.05 * np.cos(2 * np.pi * xx / nx * 3) * np.sin(2 * np.pi * yy / ny)).astype(np.float32)
    _, _, maps = O.forward(tau.astype(np.float64), lines, "nonlocal", S=S)
    uy0 = max(np.max(np.abs(m[1][:, 0])) for m in maps)
    ux_ragged = max(np.max(np.abs(m[0][:, 128:])) for m in maps)
    assert 11.9 < uy0 < 12.1 and 5.9 < ux_ragged < 6.1
    ref = O.retrieve(d.astype(np.float64), lines, "nonlocal", 1, 0.4, S=S, tau0=tau.astype(np.float64))
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "nonlocal", max_batch=1, max_shift_px=S, init=1)
    out = _dev(tau[None].copy())
    E.epr_retrieve(plan, _dev(d[None]), out, 1, 0.4)
    got = out.cpu().numpy()[0]
    plan.destroy()
    assert_close(got, ref, TOL_PHASE)


def test_splat_overflow_flag(E):
    """The splat's fixed-point accumulators (u32, 1.0 = 2^26) hold up to 32x the flat field per detector pixel and line.
    A cylindrical lens τ = (x − xc)²/(2c) sends 41 source columns onto ONE detector column (u_x = −(x − xc) exactly):
    ≈ 40x the flat field, which must raise EPR_FLAG_SPLAT_OVERFLOW; an ordinary forward must not."""
    import torch
    from paper_2601_22793_b200.binding import EPR_FLAG_SPLAT_OVERFLOW
    en, w, db = SPECTRA["mono"]
    ny, nx, S, xc = 64, 256, 24.0, 100
    l0 = O.derive_lines(6.5e-6, 1.0, en, w, db)
    c = 4000.0
    L = c / float(l0.a[0] * l0.gamma[0])
    xx = np.arange(nx, dtype=np.float64)
    prof = np.where(np.abs(xx - xc) <= 21, (xx - xc) ** 2 / (2 * c), 21.0 ** 2 / (2 * c))
    tau = np.tile(prof, (ny, 1)).astype(np.float32)[None]
    lines = O.derive_lines(6.5e-6, L, en, w, db)
    ref, _, maps = O.forward(tau[0].astype(np.float64), lines, "nonlocal", S=S)
    assert 33.0 < ref.max() < 63.0
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "nonlocal", max_batch=1, max_shift_px=S)
    P = torch.empty((1, ny, nx), device="cuda")
    assert plan.read_flags() == 0
    E.epr_forward(plan, _dev(0.1 * tau), P)                # a tenth of the lens: 5 columns per pixel at most
    assert plan.read_flags() == 0
    E.epr_forward(plan, _dev(tau), P)
    assert plan.read_flags(clear=False) & EPR_FLAG_SPLAT_OVERFLOW
    assert plan.read_flags() & EPR_FLAG_SPLAT_OVERFLOW and plan.read_flags() == 0      # cleared by the read
    plan.destroy()


def test_shift_histogram_largest_documented_shape(E):
    """epr_shift_histogram at the largest shape include/epr.h documents, 16 lines x 1024 bins (64 KB of per-CTA counters: the
    launcher takes the lines in passes that fit 48 KB of shared memory), and at 13 x 1024 and 16 x 800, against the
    oracle's histogram with the same near-edge allowance as below."""
    n = 16
    en = np.linspace(50.0, 150.0, n)
    wt = np.exp(-0.5 * ((en - 100.0) / 30.0) ** 2)
    db = 300.0 * en / 100.0
    ny, nx = 96, 160
    tau = np.stack([_tau_field(ny, nx, 21, amp=0.2), _tau_field(ny, nx, 22, amp=0.1)])
    for n_lines, n_hist in ((16, 1024), (13, 1024), (16, 800)):
        plan = E.epr_plan(nx, ny, 6.5e-6, 8.0, en[:n_lines], wt[:n_lines], db[:n_lines], "nonlocal", max_batch=2)
        lines = O.derive_lines(6.5e-6, 8.0, en[:n_lines], wt[:n_lines], db[:n_lines])
        bin_px = float(1.05 * O.max_shift(tau[0].astype(np.float64), lines) * np.sqrt(2.0) / n_hist)
        hist = E.epr_shift_histogram(plan, _dev(tau), n_hist, bin_px).cpu().numpy()
        plan.destroy()
        assert hist.shape == (2, n_lines, n_hist)
        for j in range(2):
            t64 = tau[j].astype(np.float64)
            ref = O.shift_histogram(t64, lines, n_hist, bin_px)
            assert np.all(hist[j].sum(axis=1) == nx * ny)
            assert np.count_nonzero(ref[0]) > n_hist // 8                   # the counts really spread over the bins
            for s in range(n_lines):
                ux, uy = O.ray_map(O.line_intensities(t64, lines)[s], lines.a[s], np.inf)
                eta = np.sqrt(ux * ux + uy * uy) / bin_px
                near_edge = int(np.sum(np.abs(eta - np.rint(eta)) < 1e-4 * np.maximum(eta, 1.0)))
                assert np.sum(np.abs(hist[j, s].astype(np.int64) - ref[s])) <= 2 * near_edge, (n_lines, n_hist, j, s)


def test_oversampled_host_path_and_shift_histogram(E):
    """epr_retrieve_oversampled_host (detector-grid host buffers, chunked: batch 5 > max_batch 2) equals the device call bit
    for bit; epr_shift_histogram of the result against the oracle's per-line histogram (Fig. 6): the bin of a
    pixel is decided by a float, so the counts may differ by the pixels whose fp64 value lies within 1e-4 of a bin edge."""
    import torch
    w = make_workload("C4", n=64, batch=5)
    m = 2
    plan = E.epr_plan(m * w.nx, m * w.ny, w.pixel_m / m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver,
                      max_batch=2, max_shift_px=24.0)
    dh = torch.from_numpy(w.d).pin_memory()
    oh = torch.empty_like(dh).pin_memory()
    E.epr_retrieve_host(plan, dh, oh, 3, w.step, factor=m)
    for j0 in (0, 2, 4):
        d = _dev(w.d[j0:j0 + 2])
        out = torch.empty_like(d)
        E.epr_retrieve_oversampled(plan, m, d, out, 3, w.step)
        assert torch.equal(out.cpu(), oh[j0:j0 + 2])
    plan.destroy()
    # histogram on a plan of the detector grid, from the retrieved τ
    plan = E.epr_plan(w.nx, w.ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver, max_batch=5)
    tau = oh.cuda()
    n_hist, bin_px = 64, 0.25
    hist = E.epr_shift_histogram(plan, tau, n_hist, bin_px).cpu().numpy()
    plan.destroy()
    lines = O.derive_lines(w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    for j in range(5):
        t64 = oh[j].numpy().astype(np.float64)
        ref = O.shift_histogram(t64, lines, n_hist, bin_px)
        assert np.all(hist[j].sum(axis=1) == w.nx * w.ny)
        for s in range(w.n_bins):
            ux, uy = O.ray_map(O.line_intensities(t64, lines)[s], lines.a[s], np.inf)
            eta = np.sqrt(ux * ux + uy * uy) / bin_px
            near_edge = int(np.sum(np.abs(eta - np.rint(eta)) < 1e-4 * np.maximum(eta, 1.0)))
            assert np.sum(np.abs(hist[j, s].astype(np.int64) - ref[s])) <= 2 * near_edge
        assert ref[0].argmax() != ref[-1].argmax() or ref[0].max() != ref[-1].max()


def test_two_plans_on_two_devices(E):
    """A plan belongs to the device that was current in epr_plan; launcher state (function attributes, occupancy) is kept
    per device.  Runs when two GPUs are visible: one plan each, interleaved calls from the OTHER device's context, results
    equal to the one-device result."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two visible GPUs")
    w = make_workload("C3", n=256)
    outs = []
    plans = []
    for dev in (0, 1):
        with torch.cuda.device(dev):
            plans.append(E.epr_plan(w.nx, w.ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver,
                                    max_batch=1, max_shift_px=w.max_shift_px))
    for dev in (0, 1):
        d = torch.from_numpy(w.d[:1]).to(f"cuda:{dev}")
        out = torch.empty_like(d)
        with torch.cuda.device(1 - dev):                           # the caller's current device is the OTHER one; the
            E.epr_retrieve(plans[dev], d, out, w.iterations, w.step)   # default stream handle (0) means the plan's device
        torch.cuda.synchronize(dev)
        outs.append(out.cpu())
    for p in plans:
        p.destroy()
    assert torch.equal(outs[0], outs[1])


@pytest.mark.parametrize("n_lines", [2, 16])
def test_retrieve_fewest_and_most_lines(E, n_lines):
    """2 lines and the maximum the plan accepts (16: every per-line array of the kernels' parameter block in use), non-local."""
    w = make_workload("C4", n=128)
    e = np.linspace(60.0, 140.0, n_lines)
    wt = np.exp(-0.5 * ((e - 100.0) / 20.0) ** 2)
    w.energy_keV, w.weight, w.delta_over_beta = e, wt / wt.sum(), 200.0 * e / 100.0
    got, refs = _run_retrieve(E, w, iterations=6)
    assert_close(got[0], refs[0], TOL_PHASE)


@pytest.mark.parametrize("S", [0.0, 30.0])
def test_shift_clamp_extremes(E, S):
    """max_shift_px = 0 (every shift clamped to zero: the transport degenerates to the identity, R6) and 30 (the largest the
    library accepts: one 1024-thread CTA per SM in the splat), against the oracle with the same clamp; one and three lines."""
    import torch
    for spec in ("mono", "poly3_unequal_a"):
        en, w, db = SPECTRA[spec]
        ny, nx, L = 128, 256, 200.0
        tau = _tau_field(ny, nx, 6, amp=0.5)[None]
        lines = O.derive_lines(6.5e-6, L, en, w, db)
        assert O.max_shift(tau[0].astype(np.float64), lines) > 31.0          # the clamp binds at either extreme
        plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "nonlocal", max_batch=1, max_shift_px=S)
        P = torch.empty((1, ny, nx), device="cuda")
        Pb = torch.empty((1, len(en), ny, nx), device="cuda")
        E.epr_forward(plan, _dev(tau), P, Pb)
        ref, ref_bins, _ = O.forward(tau[0].astype(np.float64), lines, "nonlocal", S=S)
        assert_close(P.cpu().numpy()[0], ref, TOL_OP)
        if S == 0.0:
            Is = O.line_intensities(tau[0].astype(np.float64), lines)
            assert_close(Pb.cpu().numpy()[0, 0], Is[0], TOL_OP)               # identity transport
        d = np.float32(ref * (1.0 + 0.01 * np.cos(np.arange(nx) * 0.1))[None, :])[None]
        out = _dev(tau.copy())
        plan.destroy()
        plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "nonlocal", max_batch=1, max_shift_px=S, init=1)
        E.epr_retrieve(plan, _dev(d), out, 2, 0.4)
        plan.destroy()
        want = O.retrieve(d[0].astype(np.float64), lines, "nonlocal", 2, 0.4, S=S, tau0=tau[0].astype(np.float64))
        assert_close(out.cpu().numpy()[0], want, TOL_PHASE)


def test_argument_errors_more(E):
    import torch
    en, w, db = SPECTRA["mono"]
    e17 = np.linspace(60.0, 140.0, 17)
    for kw in (dict(max_shift_px=31.0), dict(newton_iters=-1), dict(order=3), dict(output=3), dict(out_bin=1), dict(i_min=0.0)):
        with pytest.raises(E.EprError) as ei:
            E.epr_plan(64, 64, 6.5e-6, 1.0, en, w, db, "nonlocal", **kw)
        assert ei.value.status == 1
    with pytest.raises(E.EprError):
        E.epr_plan(64, 64, 6.5e-6, 1.0, e17, np.ones(17), np.full(17, 1000.0))      # more than 16 lines
    with pytest.raises(E.EprError):
        E.epr_plan(64, 64, 6.5e-6, 1.0, en, [0.0], db)                              # non-positive weight
    plan = E.epr_plan(64, 64, 6.5e-6, 1.0, en, w, db, max_batch=2)
    empty = torch.ones((0, 64, 64), device="cuda")
    with pytest.raises(E.EprError):
        E.epr_retrieve(plan, empty, torch.empty_like(empty), 1, 1.0)                # empty batch
    d = torch.ones((1, 64, 64), device="cuda")
    with pytest.raises(E.EprError):
        E.epr_retrieve(plan, d, torch.empty_like(d), -1, 1.0)                       # negative iteration count
    with pytest.raises(E.EprError):
        E.epr_plan_profiles(plan, np.ones((3, 1)), np.full((3, 1), 1000.0))         # 3 blocks do not divide nx = 64
    with pytest.raises(E.EprError):
        E.epr_shift_histogram(plan, d, 1, 0.1)                                      # fewer than 2 bins
    plan.destroy()
