"""epr_residual_rms_static — the entry point for callers that cannot allocate device memory.

Some users of this library run it inside a process whose GPU memory is already fully committed (the reconstruction
framework's pool, plans sized at start-up) or inside an acquisition-rate loop that cannot take the stall of a
cudaMalloc; the plan-based residual diagnostic (epr_set_diagnostics) takes its reduction scratch from cudaMalloc on first
use, so they get a variant whose scratch is a fixed array inside libepr.so (include/epr.h).  This file checks that the
variant returns what the existing path returns — on two calls in a row, because both calls share that array and the
second one starts from the first one's leftovers.

It is a file of its own, named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It holds no state from other tests (own plan, own tensors), so it passes alone in a
fresh process as well as at the end of the whole suite."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_DIAG = 2e-3      # test_diagnostics_history's tolerance for diag[..][0]: e is a small difference of O(1) planes in fp32
TOL_SUM = 1e-6       # against the same sum written out in fp64 on the same planes: only the fp32 line sum differs


@pytest.fixture(scope="module")
def E():
    import torch
    import paper_2601_22793_b200 as epr
    assert torch.cuda.is_available()
    epr.load_library()
    return epr


def _existing_path(E, solver, ny, nx, seed):
    """One correction iteration from a caller-supplied τ⁰ (opt.init = 1) with the plan-based diagnostic switched on: returns
    diag[b][0][0] — the existing path's residual RMS at τ⁰ — together with per-line residual planes of the same τ⁰
    (epr_forward, then e_s = f_s · (d − Σ_t P_t): any split whose sum is e) for the new entry point."""
    import torch
    rng = np.random.default_rng(seed)
    batch = 3
    en, wt, db = np.array([70.0, 100.0, 130.0]), np.array([0.3, 0.4, 0.3]), np.array([900.0, 1000.0, 1100.0])
    y, x = np.meshgrid(np.arange(ny) * 2 * np.pi / ny, np.arange(nx) * 2 * np.pi / nx, indexing="ij")
    tau0 = np.stack([(0.04 + 0.01 * b) * (1.2 + np.cos(2 * x + b) * np.sin(3 * y)) for b in range(batch)])
    d = 1.0 + 0.05 * np.cos(3 * x - y)[None] * np.linspace(0.5, 1.5, batch)[:, None, None] + 0.01 * rng.normal(size=tau0.shape)
    tau0_t = torch.from_numpy(tau0.astype(np.float32)).cuda()
    d_t = torch.from_numpy(d.astype(np.float32)).cuda()
    plan = E.epr_plan(nx, ny, 6.5e-6, 0.5, en, wt, db, solver, max_batch=batch, max_shift_px=8.0, init=1)
    diag = torch.zeros(batch, 1, 2, device="cuda")
    E.epr_set_diagnostics(plan, diag)
    out = tau0_t.clone()
    E.epr_retrieve(plan, d_t, out, 1, 0.5)
    E.epr_set_diagnostics(plan, None)
    P = torch.empty_like(d_t)
    E.epr_forward(plan, tau0_t, P)
    f = torch.from_numpy(plan.lines()["f"].astype(np.float32)).cuda()
    e_bins = (f[None, :, None, None] * (d_t - P)[:, None]).contiguous()
    torch.cuda.synchronize()
    plan.destroy()
    return diag[:, 0, 0].clone(), e_bins


def _fp64(e_bins):
    import torch
    return torch.sqrt((e_bins.double().sum(1) ** 2).mean((1, 2)))


@pytest.mark.parametrize("solver", ["local", "nonlocal"])
def test_static_scratch_matches_the_plan_based_diagnostic_twice_in_a_row(E, solver):
    import torch
    want_a, e_a = _existing_path(E, solver, 128, 256, 1)
    want_b, e_b = _existing_path(E, solver, 64, 48, 2)
    rms_a = torch.full((3,), -1.0, device="cuda")
    rms_b = torch.full((2,), -1.0, device="cuda")
    # two calls back to back on one stream; the second is smaller, with other data, and starts from the first one's scratch
    E.epr_residual_rms_static(e_a, rms_a)
    E.epr_residual_rms_static(e_b[:2].contiguous(), rms_b)
    torch.cuda.synchronize()
    for got, want, e in ((rms_a, want_a, e_a), (rms_b, want_b[:2], e_b[:2])):
        got, want = got.cpu().numpy().astype(np.float64), want.cpu().numpy().astype(np.float64)
        assert np.all(want > 1e-3)                                        # a real residual, not a converged one
        assert np.max(np.abs(got - want)) < TOL_DIAG * np.max(want), (got, want)
        ref = _fp64(e).cpu().numpy()
        assert np.max(np.abs(got - ref) / ref) < TOL_SUM, (got, ref)
    # and again, same inputs: the same bits (fixed summation order, nothing read that the call did not write)
    again = torch.empty_like(rms_a)
    E.epr_residual_rms_static(e_a, again)
    assert torch.equal(again, rms_a)


def test_static_scratch_shapes_and_limits(E):
    """Unaligned plane (nx · ny % 4 != 0), one line, and the stated maximum: one projection more than
    EPR_STATIC_MAX_BATCH is refused with a message that names the limit, and nothing is written."""
    import torch
    g = torch.Generator(device="cuda").manual_seed(7)
    e = torch.randn((5, 1, 7, 9), device="cuda", generator=g) * 0.1
    rms = torch.empty(5, device="cuda")
    E.epr_residual_rms_static(e, rms)
    ref = _fp64(e)
    assert float(((rms.double() - ref).abs() / ref).max()) < TOL_SUM
    nb = E.EPR_STATIC_MAX_BATCH
    e = torch.randn((nb + 1, 2, 4, 8), device="cuda", generator=g)
    rms = torch.full((nb + 1,), -1.0, device="cuda")
    E.epr_residual_rms_static(e[:nb].contiguous(), rms[:nb])              # the maximum itself is served
    ref = _fp64(e[:nb])
    assert float(((rms[:nb].double() - ref).abs() / ref).max()) < TOL_SUM
    rms.fill_(-1.0)
    with pytest.raises(E.EprError) as ei:
        E.epr_residual_rms_static(e, rms)
    assert ei.value.status == 2 and "EPR_STATIC_MAX_BATCH" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((rms == -1.0).all())
    with pytest.raises(E.EprError) as ei:                                  # 17 lines: outside 1..16, like every plan
        E.epr_residual_rms_static(torch.zeros((1, 17, 4, 4), device="cuda"), torch.empty(1, device="cuda"))
    assert ei.value.status == 1
