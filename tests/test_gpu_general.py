"""GPU parity of the GENERAL path (epr_general.cu, epr_fftgen.cu) against the fp64 oracle: any {2,3,5}-smooth grid >= 8
 and the x-dependent effective spectrum (reading R17;
oracle: retrieve_x and friends).  Same tolerances as tests/test_gpu_parity.py, same element-wise bound."""
import numpy as np
import pytest

from oracle import epr_oracle as O
from test_gpu_parity import TOL_OP, TOL_PHASE, TOL_MASS, assert_close, rel_l2, _dev, _tau_field, SPECTRA  # noqa: F401

pytestmark = pytest.mark.gpu

E3 = np.array([70.0, 100.0, 130.0])
W3 = np.array([0.3, 0.45, 0.25])
DB3 = np.array([600.0, 1000.0, 1500.0])


@pytest.fixture(scope="module")
def E():
    import torch
    import paper_2601_22793_b200 as epr
    assert torch.cuda.is_available()
    epr.load_library()
    return epr


def _data(ny, nx, seed, amp=0.1):
    rng = np.random.default_rng(seed)
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    d = 1.0 + amp * (np.cos(x + 0.3) * np.sin(2 * y) + 0.5 * np.cos(3 * x - 2 * y)) + 0.003 * rng.normal(size=(ny, nx))
    return d.astype(np.float32)


# (nx, ny): sizes SURVEY.md §8(b) / VERDICT name — 1536², 1920 x 1080, 3200 x 256 (the paper's 3104-wide radiographs
# padded to 2^7·5²), 250 = 2·5³ — plus an odd length, a tiny grid and a non-multiple of 4
GRIDS = [(1536, 1536), (1920, 1080), (3200, 256), (250, 256), (256, 250), (375, 40), (8, 24), (90, 150), (1080, 48),
         (8192, 16), (16, 8192), (6561, 8)]            # the longest lengths the run-time-radix FFT takes (8192 = 2^13, 6561 = 3^8)


@pytest.mark.parametrize("nx,ny", GRIDS)
def test_precondition_any_smooth_grid(E, nx, ny):
    import torch
    en, w, db = SPECTRA["poly3_unequal_a"]
    L = 3.0
    for symbol in (0, 1):
        plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, "local", max_batch=1, symbol=symbol)
        lines = O.derive_lines(6.5e-6, L, en, w, db)
        r = np.random.default_rng(5).normal(size=(1, 3, ny, nx)).astype(np.float32)
        q = torch.empty_like(_dev(r))
        E.epr_precondition(plan, _dev(r), q)
        q = q.cpu().numpy()
        plan.destroy()
        for s in range(3):
            assert_close(q[0, s], O.precondition(r[0, s].astype(np.float64), lines.a[s], symbol), TOL_OP, f"{nx}x{ny} line {s}")


@pytest.mark.parametrize("nx,ny", GRIDS)
@pytest.mark.parametrize("solver,step,L", [("local", 1.0, 0.3), ("nonlocal", 0.4, 8.0)])
def test_retrieve_any_smooth_grid(E, nx, ny, solver, step, L):
    """A short retrieval (Paganin start + 3 iterations, 3 unequal lines) on every grid, both solvers."""
    import torch
    en, w, db = SPECTRA["poly3_unequal_a"]
    d = _data(ny, nx, nx + ny)
    lines = O.derive_lines(6.5e-6, L, en, w, db)
    ref = O.retrieve(d.astype(np.float64), lines, solver, 3, step, S=8.0)
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, solver, max_batch=1, max_shift_px=8.0)
    dd = _dev(d[None])
    out = torch.empty_like(dd)
    E.epr_retrieve(plan, dd, out, 3, step)
    got = out.cpu().numpy()[0]
    plan.destroy()
    assert_close(got, ref, TOL_PHASE, f"{nx}x{ny} {solver}")


def test_argument_errors_sizes(E):
    en, w, db = SPECTRA["mono"]
    for nx, ny in ((14, 16), (16, 7 * 16), (4, 64), (64, 4), (0, 64), (64, -8)):   # prime factor 7; below 8; not positive
        with pytest.raises(E.EprError) as ei:
            E.epr_plan(nx, ny, 6.5e-6, 1.0, en, w, db)
        assert ei.value.status == (1 if min(nx, ny) < 1 else 2)        # EPR_EINVAL / EPR_ESIZE as include/epr.h says
    E.epr_plan(250, 16, 6.5e-6, 1.0, en, w, db).destroy()          # 250 = 2·5³ plans


@pytest.mark.parametrize("nx,ny", [(150, 90), (160, 96)])
def test_operators_general_path_uniform(E, nx, ny):
    """epr_forward / epr_adjoint / epr_transport on the general path (150 x 90: unaligned, run-time-radix FFT; 160 x 96 with
    one block profile: the general kernels with the tuned FFT), uniform spectrum, against the oracle's operators."""
    import torch
    en, w, db = SPECTRA["poly3_unequal_a"]
    for solver, L, S in (("local", 2.0, 16.0), ("nonlocal", 60.0, 12.0)):
        plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, solver, max_batch=2, max_shift_px=S)
        if nx % 16 == 0:
            E.epr_plan_profiles(plan, [w], [db])
        lines = O.derive_lines(6.5e-6, L, en, w, db)
        tau = np.stack([_tau_field(ny, nx, 1, amp=0.05), _tau_field(ny, nx, 2, amp=0.3)])
        P = torch.empty((2, ny, nx), device="cuda")
        Pb = torch.empty((2, 3, ny, nx), device="cuda")
        E.epr_forward(plan, _dev(tau), P, Pb)
        Ph, Pbh = P.cpu().numpy(), Pb.cpu().numpy()
        rng = np.random.default_rng(9)
        e = rng.normal(size=(2, 3, ny, nx)).astype(np.float32)
        xs = rng.uniform(-1.0, 2.0, size=(2, 3, ny, nx)).astype(np.float32)
        r = torch.empty_like(Pb)
        E.epr_adjoint(plan, _dev(e), r)
        rh = r.cpu().numpy()
        if solver == "nonlocal":
            Mx = torch.empty_like(Pb)
            E.epr_transport(plan, _dev(xs), Mx)
            Mxh = Mx.cpu().numpy()
        plan.destroy()
        for b in range(2):
            ref, ref_bins, maps = O.forward(tau[b].astype(np.float64), lines, solver, S=S)
            Is = O.line_intensities(tau[b].astype(np.float64), lines)
            assert_close(Ph[b], ref, TOL_OP)
            assert rel_l2(Ph[b] - 1.0, ref - 1.0) < 20 * TOL_OP
            for s in range(3):
                assert_close(Pbh[b, s], ref_bins[s], TOL_OP)
                if solver == "nonlocal":
                    assert abs(Pbh[b, s].astype(np.float64).sum() - Is[s].sum()) <= TOL_MASS * Is[s].sum()
                    assert_close(rh[b, s], O.gather(e[b, s].astype(np.float64), *maps[s]), TOL_OP)
                    assert_close(Mxh[b, s], O.splat(xs[b, s].astype(np.float64), *maps[s]), TOL_OP)
                else:
                    assert np.array_equal(rh[b, s], e[b, s])


# ---------------------------------------------------------------------------------------------------------------------
# x-dependent effective spectrum
# ---------------------------------------------------------------------------------------------------------------------
def _profiles(nx, n_blocks, L, n_lines=3, mu=False):
    t = np.linspace(0.0, 1.0, n_blocks)[:, None]
    if n_lines == 3:
        en = E3
        wt = W3[None, :] * (1.0 + t * np.array([0.8, 0.0, -0.6])[None, :])
        db = DB3[None, :] * (1.0 + 0.3 * t)
        mu_rel = None if not mu else (np.array([3.0, 1.0, 0.4])[None, :] * (1.0 + 0.2 * t))
    else:
        en = np.array([100.0])
        wt = np.ones((n_blocks, 1))
        db = 1000.0 * (1.0 + 0.4 * t)
        mu_rel = None if not mu else 1.0 + 0.3 * t
    return en, wt, db, mu_rel, O.derive_profiles(6.5e-6, L, en, nx, wt, db, mu_rel)


@pytest.mark.parametrize("nx,ny", [(160, 96), (150, 90)])
@pytest.mark.parametrize("solver,step,L,S", [("local", 1.0, 0.3, 16.0), ("nonlocal", 0.4, 8.0, 6.0)])
@pytest.mark.parametrize("n_lines,mu", [(3, False), (3, True), (1, True)])
def test_retrieve_profiles_parity(E, nx, ny, solver, step, L, S, n_lines, mu):
    """The loop with block profiles of f_s, γ_s, db_s (5 blocks) against the oracle's retrieve_x: tuned-FFT grid and
    run-time-radix grid, both solvers, derived and caller-given attenuation scaling, one line with x-dependent γ."""
    import torch
    nblk = 5
    en, wt, db, mu_rel, prof = _profiles(nx, nblk, L, n_lines, mu)
    d = _data(ny, nx, 7 + nx)
    ref = O.retrieve_x(d.astype(np.float64), prof, solver, 4, step, S=S)
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, wt[0], db[0], solver, max_batch=2, max_shift_px=S)
    E.epr_plan_profiles(plan, wt, db, mu_rel)
    cols = plan.columns()
    assert np.allclose(cols["f"], prof.f, rtol=1e-12) and np.allclose(cols["gamma"], prof.gamma, rtol=1e-12)
    assert np.allclose(cols["a"], prof.a, rtol=1e-12)
    dd = _dev(np.stack([d, d[::-1].copy()]))
    out = torch.empty_like(dd)
    E.epr_retrieve(plan, dd, out, 4, step)
    got = out.cpu().numpy()
    plan.destroy()
    assert_close(got[0], ref, TOL_PHASE, f"profiles {solver} {n_lines} line(s)")
    ref1 = O.retrieve_x(d[::-1].astype(np.float64), prof, solver, 4, step, S=S)
    assert_close(got[1], ref1, TOL_PHASE)
    if n_lines == 3:
        uni = O.retrieve(d.astype(np.float64), O.derive_lines(6.5e-6, L, en, wt[0], db[0]), solver, 4, step, S=S)
        assert rel_l2(ref, uni) > 50 * TOL_PHASE          # the profiles matter at this tolerance


@pytest.mark.parametrize("solver,L,S", [("local", 2.0, 16.0), ("nonlocal", 60.0, 12.0)])
def test_operators_profiles_parity(E, solver, L, S):
    """epr_forward, epr_adjoint, epr_transport, epr_precondition with block profiles against forward_x, gather, splat and the
    blockwise-interpolated filter precondition_x (R17(c))."""
    import torch
    nx, ny, nblk = 160, 96, 4
    en, wt, db, mu_rel, prof = _profiles(nx, nblk, L, 3, True)
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, wt[0], db[0], solver, max_batch=1, max_shift_px=S)
    E.epr_plan_profiles(plan, wt, db, mu_rel)
    tau = _tau_field(ny, nx, 2, amp=0.3)[None]
    P = torch.empty((1, ny, nx), device="cuda")
    Pb = torch.empty((1, 3, ny, nx), device="cuda")
    E.epr_forward(plan, _dev(tau), P, Pb)
    ref, ref_bins, maps = O.forward_x(tau[0].astype(np.float64), prof, solver, S=S)
    Is = O.line_intensities_x(tau[0].astype(np.float64), prof)
    assert_close(P.cpu().numpy()[0], ref, TOL_OP)
    assert rel_l2(P.cpu().numpy()[0] - 1.0, ref - 1.0) < 20 * TOL_OP
    rng = np.random.default_rng(4)
    e = rng.normal(size=(1, 3, ny, nx)).astype(np.float32)
    q = torch.empty_like(Pb)
    E.epr_precondition(plan, _dev(e), q)
    qh = q.cpu().numpy()
    ebuf = _dev(e)
    E.epr_precondition(plan, ebuf, ebuf)                   # in place
    assert np.array_equal(ebuf.cpu().numpy(), qh)
    for s in range(3):
        assert_close(Pb.cpu().numpy()[0, s], ref_bins[s], TOL_OP)
        assert_close(qh[0, s], O.precondition_x(e[0, s].astype(np.float64), prof.a_blk[:, s], prof.wblk), TOL_OP)
    if solver == "nonlocal":
        r = torch.empty_like(Pb)
        E.epr_adjoint(plan, _dev(e), r)
        Mx = torch.empty_like(Pb)
        xs = rng.uniform(0.0, 2.0, size=(1, 3, ny, nx)).astype(np.float32)
        E.epr_transport(plan, _dev(xs), Mx)
        for s in range(3):
            assert abs(Pb.cpu().numpy()[0, s].astype(np.float64).sum() - Is[s].sum()) <= TOL_MASS * Is[s].sum()
            assert_close(r.cpu().numpy()[0, s], O.gather(e[0, s].astype(np.float64), *maps[s]), TOL_OP)
            assert_close(Mx.cpu().numpy()[0, s], O.splat(xs[0, s].astype(np.float64), *maps[s]), TOL_OP)
    plan.destroy()


@pytest.mark.parametrize("solver,step,L", [("local", 1.0, 0.3), ("nonlocal", 0.4, 8.0)])
def test_uniform_profiles_match_the_tuned_path(E, solver, step, L):
    """§9.2 "single block": identical block profiles on the general path give the tuned path's result (same readings, other
    kernels: agreement to fp32 rounding, far inside the tolerance), for 1 and for 4 blocks."""
    import torch
    nx, ny = 256, 128
    en, w, db = SPECTRA["poly3_unequal_a"]
    d = _dev(_data(ny, nx, 11)[None])
    res = []
    for nblk in (0, 1, 4):
        plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w, db, solver, max_batch=1, max_shift_px=8.0)
        if nblk:
            E.epr_plan_profiles(plan, [w] * nblk, [db] * nblk)
        out = torch.empty_like(d)
        E.epr_retrieve(plan, d, out, 4, step)
        res.append(out.cpu().numpy()[0])
        plan.destroy()
    assert_close(res[1], res[0], 0.1 * TOL_PHASE)
    assert_close(res[2], res[0], 0.1 * TOL_PHASE)


def test_profiles_output_modes_and_host_path(E):
    """opt.output with column scalars (phase of a line: −(db_s(x)/2) γ_s(x) τ, Eq. (6)) and the chunked host call on a
    profile plan."""
    import torch
    nx, ny, L = 160, 96, 0.3
    en, wt, db, mu_rel, prof = _profiles(nx, 4, L, 3, False)
    d = np.stack([_data(ny, nx, 21), _data(ny, nx, 22), _data(ny, nx, 23)])
    refs = [O.retrieve_x(d[j].astype(np.float64), prof, "local", 3, 1.0) for j in range(3)]
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, wt[0], db[0], "local", max_batch=2, output=1, out_bin=2)
    E.epr_plan_profiles(plan, wt, db, mu_rel)
    dh = torch.from_numpy(d).pin_memory()
    oh = torch.empty_like(dh).pin_memory()
    E.epr_retrieve_host(plan, dh, oh, 3, 1.0)
    plan.destroy()
    for j in range(3):
        want = -(prof.db[2][None, :] / 2.0) * prof.gamma[2][None, :] * refs[j]
        assert_close(oh[j].numpy(), want, TOL_PHASE)


@pytest.mark.parametrize("solver,step,L,S", [("local", 1.0, 0.3, 16.0), ("nonlocal", 0.4, 8.0, 6.0)])
@pytest.mark.parametrize("n_lines", [3, 1])
def test_retrieve_profiles_staged_column_transforms(E, solver, step, L, S, n_lines):
    """ny = 256 (power of two, TMA column kernel): with several blocks the columns are transformed ONCE per iteration and every
    block filter runs on the transformed spectra (stage 1 / stage 2 of k_cols_tma), also for the initial solve; 64 x 256 grid,
    4 blocks, against retrieve_x."""
    import torch
    nx, ny, nblk = 64, 256, 4
    en, wt, db, mu_rel, prof = _profiles(nx, nblk, L, n_lines, True)
    d = _data(ny, nx, 31)
    ref = O.retrieve_x(d.astype(np.float64), prof, solver, 4, step, S=S)
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, wt[0], db[0], solver, max_batch=1, max_shift_px=S)
    E.epr_plan_profiles(plan, wt, db, mu_rel)
    dd = _dev(d[None])
    out = torch.empty_like(dd)
    l0 = plan.launches
    E.epr_retrieve(plan, dd, out, 4, step)
    got = out.cpu().numpy()[0]
    n_launch = plan.launches - l0
    plan.destroy()
    assert_close(got, ref, TOL_PHASE, f"staged columns, {solver}, {n_lines} line(s)")
    # 5 solves x (1 row pass + 1 staged column pass + 4 x (block filter + inverse rows) + 1 update) + forward-model launches
    assert n_launch >= 5 * (1 + 1 + 2 * nblk + 1)


def test_profiles_on_the_oversampled_grid_and_graph_replay(E):
    """The x-dependent spectrum combined with the oversampled loop (PAPER.md:79 + §9.2: the paper's production set-up): plan on
    the x2 grid with block profiles, replicate -> retrieve_x -> block mean against the oracle; and on a side stream the
    launch-bound general-path retrieval is captured into a CUDA graph and replayed bit for bit."""
    import torch
    nxd, nyd, m, L = 80, 48, 2, 0.3
    en, wt, db, mu_rel, _ = _profiles(m * nxd, 4, L, 3, True)
    prof_f = O.derive_profiles(6.5e-6 / m, L, en, m * nxd, wt, db, mu_rel)
    d = _data(nyd, nxd, 41)
    ref = O.downsample(O.retrieve_x(O.upsample(d.astype(np.float64), m), prof_f, "local", 3, 1.0), m)
    plan = E.epr_plan(m * nxd, m * nyd, 6.5e-6 / m, L, en, wt[0], db[0], "local", max_batch=1)
    E.epr_plan_profiles(plan, wt, db, mu_rel)
    dd = _dev(d[None])
    out = torch.empty_like(dd)
    E.epr_retrieve_oversampled(plan, m, dd, out, 3, 1.0)
    assert_close(out.cpu().numpy()[0], ref, TOL_PHASE, "profiles on the x2 grid")
    plan.destroy()
    # graph capture of the general path (160 x 96, non-local, run-time memset + atomics inside the capture on 150 x 90)
    for nx, ny in ((160, 96), (150, 90)):
        en, wt, db, mu_rel, prof = _profiles(nx, 5, 8.0, 3, False)
        plan = E.epr_plan(nx, ny, 6.5e-6, 8.0, en, wt[0], db[0], "nonlocal", max_batch=1, max_shift_px=6.0)
        E.epr_plan_profiles(plan, wt, db, mu_rel)
        dd = _dev(_data(ny, nx, 5)[None])
        ref = torch.empty_like(dd)
        E.epr_retrieve(plan, dd, ref, 3, 0.4)                  # default stream: eager
        torch.cuda.synchronize()
        side = torch.cuda.Stream()
        out = torch.empty_like(dd)
        with torch.cuda.stream(side):
            for _ in range(3):                                 # eager warm pass, capture + launch, replay
                out.zero_()
                E.epr_retrieve(plan, dd, out, 3, 0.4)
                side.synchronize()
                assert torch.equal(out, ref)
        plan.destroy()


# ---------------------------------------------------------------------------------------------------------------------
# variants on the general path: opt.nonlocal_wkb1 (R4) and epr_set_diagnostics
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nx,ny,blocks", [(90, 150, 0), (96, 160, 4), (90, 150, 3)])
def test_nonlocal_wkb1_variant_general_path(E, nx, ny, blocks):
    """opt.nonlocal_wkb1 (variant of R4) on a grid the tuned kernels do not take (blocks = 0: uniform
    spectrum) and with block profiles on an aligned and on an unaligned grid: the WKB1 term of Eq. (1) at the detector
    pixel's column (oracle: forward / forward_x with nonlocal_wkb1), at a δ/β small enough for the term to matter."""
    import torch
    S, L = 8.0, 20.0
    en, wt, db = np.array([80.0, 100.0, 120.0]), np.array([0.3, 0.4, 0.3]), np.array([8.0, 10.0, 12.0])
    tau = _tau_field(ny, nx, 5, amp=0.3)[None]
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, wt, db, "nonlocal", max_batch=1, max_shift_px=S, nonlocal_wkb1=1)
    if blocks:
        t = np.linspace(0.0, 1.0, blocks)[:, None]
        wb, dbb = wt[None, :] * (1.0 + t * np.array([0.5, 0.0, -0.4])[None, :]), db[None, :] * (1.0 + 0.3 * t)
        E.epr_plan_profiles(plan, wb, dbb, None)
        prof = O.derive_profiles(6.5e-6, L, en, nx, wb, dbb)
        fwd = lambda t64, **kw: O.forward_x(t64, prof, "nonlocal", S=S, **kw)
        ret = lambda d64: O.retrieve_x(d64, prof, "nonlocal", 4, 0.4, S=S, nonlocal_wkb1=True)
    else:
        lines = O.derive_lines(6.5e-6, L, en, wt, db)
        fwd = lambda t64, **kw: O.forward(t64, lines, "nonlocal", S=S, **kw)
        ret = lambda d64: O.retrieve(d64, lines, "nonlocal", 4, 0.4, S=S, nonlocal_wkb1=True)
    P = torch.empty((1, ny, nx), device="cuda")
    Pb = torch.empty((1, 3, ny, nx), device="cuda")
    E.epr_forward(plan, _dev(tau), P, Pb)
    ref, ref_bins, _ = fwd(tau[0].astype(np.float64), nonlocal_wkb1=True)
    plain, _, _ = fwd(tau[0].astype(np.float64))
    assert rel_l2(ref, plain) > 100 * TOL_OP                         # the term is far above the tolerance here
    assert_close(P.cpu().numpy()[0], ref, TOL_OP)
    for s in range(3):
        assert_close(Pb.cpu().numpy()[0, s], ref_bins[s], TOL_OP)
    d = np.float32(ref + 0.002 * np.random.default_rng(3).normal(size=ref.shape))[None]
    out = torch.empty((1, ny, nx), device="cuda")
    E.epr_retrieve(plan, _dev(d), out, 4, 0.4)
    plan.destroy()
    assert_close(out.cpu().numpy()[0], ret(d[0].astype(np.float64)), TOL_PHASE)


@pytest.mark.parametrize("nx,ny,blocks,solver,step,L", [(90, 150, 0, "local", 1.0, 0.3), (90, 150, 0, "nonlocal", 0.4, 8.0),
                                                         (160, 96, 5, "local", 1.0, 0.3), (160, 96, 5, "nonlocal", 0.4, 8.0),
                                                         (150, 90, 5, "nonlocal", 0.4, 8.0)])
def test_diagnostics_general_path(E, nx, ny, blocks, solver, step, L):
    """epr_set_diagnostics on the general path: residual RMS and largest unclamped shift per iteration against the oracle's
    histories, uniform spectrum on an unaligned grid and block profiles (shift with the scalars of the
    pixel's own column); the host path writes every chunk into its own rows; switching it off restores the plain result."""
    import torch
    its, S = 4, 6.0
    if blocks:
        en, wt, db, mu_rel, prof = _profiles(nx, blocks, L, 3, True)
        w0, db0 = wt[0], db[0]
    else:
        en, w0, db0 = E3, W3, DB3
        lines = O.derive_lines(6.5e-6, L, en, w0, db0)
    d = np.stack([_data(ny, nx, 11), _data(ny, nx, 12, amp=0.2)])
    plan = E.epr_plan(nx, ny, 6.5e-6, L, en, w0, db0, solver, max_batch=2, max_shift_px=S)
    if blocks:
        E.epr_plan_profiles(plan, wt, db, mu_rel)
    dd = _dev(d)
    out = torch.empty_like(dd)
    diag = torch.zeros(2, its, 2, device="cuda")
    E.epr_set_diagnostics(plan, diag)
    E.epr_retrieve(plan, dd, out, its, step)
    got = diag.cpu().numpy()
    diag_h = torch.zeros_like(diag)
    E.epr_set_diagnostics(plan, diag_h)
    dh = torch.from_numpy(d).pin_memory()
    oh = torch.empty_like(dh).pin_memory()
    E.epr_retrieve_host(plan, dh, oh, its, step)
    assert torch.equal(diag_h, diag) and torch.equal(oh.cuda(), out)
    E.epr_set_diagnostics(plan, None)
    out2 = torch.empty_like(dd)
    E.epr_retrieve(plan, dd, out2, its, step)
    assert torch.equal(out, out2)
    plan.destroy()
    for j in range(2):
        h, sh = [], []
        if blocks:
            O.retrieve_x(d[j].astype(np.float64), prof, solver, its, step, S=S, history=h, shift_history=sh)
        else:
            O.retrieve(d[j].astype(np.float64), lines, solver, its, step, S=S, history=h, shift_history=sh)
        h, sh = np.array(h), np.array(sh)
        assert np.max(np.abs(got[j, :, 0] - h)) < 2e-3 * h[0]          # e is a small difference of O(1) planes in fp32
        assert np.max(np.abs(got[j, :, 1] - sh) / sh) < 1e-3
