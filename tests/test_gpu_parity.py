"""GPU parity: libdg (CUDA, fp32, through the C ABI) against the fp64 oracle on the same seeded
inputs.  Tolerances are BASELINE.json's: rel-L2 <= 2e-6 per RHS, <= 1e-4 after the LSRK run."""
import numpy as np
import pytest

from paper_1602_07997_b200 import workloads as W

from gpu_common import RHS_TOL, RUN_TOL, Case, assert_close, describe, rel_l2

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def dg():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_1602_07997_b200 import dg as mod          # raises if libdg.so is missing: no fallback
    return mod


def _sweep_case(model, N, n=3):
    w = W.config(4, N=N, model=model, n=n)
    w.jitter, w.top, w.ic = 0.08, W.BC_FREE, "random"
    return w


# ---------------------------------------------------------------- per-RHS parity, every degree, both models
@pytest.mark.parametrize("N", range(1, 11))
@pytest.mark.parametrize("model", [W.ACOUSTIC, W.ELASTIC])
@pytest.mark.parametrize("variant", [1, 4])
def test_rhs_parity_all_degrees(dg, variant, model, N):
    """K = 162 elements (several CTAs / batches and a ragged last batch; for the elastic tensor-core
    kernel with odd Np also batches whose first value is not 16-byte aligned), random N(0,1) fields,
    random discontinuous materials, free top + rigid walls.  variant 1 = fused FP32 SIMT kernel,
    variant 4 = pipelined tcgen05 kernel (BF16x3 split, every degree)."""
    case = Case(dg, _sweep_case(model, N), variant=variant)
    # variant 1 = the SIMT family: element-per-thread kernel for acoustic N <= 2 / elastic N = 1, fused node-per-thread above
    epk = N == 1 or (N == 2 and model == W.ACOUSTIC)
    assert case.ctx.variant_name.startswith(("simt_elem_per_thread" if epk else "simt_fused") if variant == 1 else "tc_pipe")
    q32 = case.initial_fields32()
    got = case.gpu_rhs(torch, q32)
    want = case.oracle_rhs(q32.astype(np.float64))
    assert_close(got, want, RHS_TOL, case.ctx.variant_name)
    per_field = [rel_l2(got[:, f], want[:, f]) for f in range(got.shape[1])]
    assert max(per_field) <= 2 * RHS_TOL, (per_field, describe(got, want))


@pytest.mark.parametrize("N", range(1, 4))
@pytest.mark.parametrize("model", [W.ACOUSTIC, W.ELASTIC])
def test_rhs_parity_row_per_thread(dg, model, N):
    """Variant 5 (rpt_kernels.cuh: thread = (element, field) row, operators in constant memory), N = 1..3: the same case as
    above -- ragged last warp (K = 162 is no multiple of 8 or 3), boundary faces of both kinds -- against the oracle."""
    case = Case(dg, _sweep_case(model, N), variant=5)
    assert case.ctx.variant_name.startswith("simt_row_per_thread")
    q32 = case.initial_fields32()
    got = case.gpu_rhs(torch, q32)
    want = case.oracle_rhs(q32.astype(np.float64))
    assert_close(got, want, RHS_TOL, case.ctx.variant_name)
    per_field = [rel_l2(got[:, f], want[:, f]) for f in range(got.shape[1])]
    assert max(per_field) <= 2 * RHS_TOL, (per_field, describe(got, want))


@pytest.mark.parametrize("model,N,E,G", [(W.ACOUSTIC, 1, 1, 16), (W.ACOUSTIC, 2, 1, 5), (W.ACOUSTIC, 3, 8, 3), (W.ACOUSTIC, 4, 2, 1),
                                         (W.ELASTIC, 1, 2, 8), (W.ELASTIC, 2, 4, 7), (W.ELASTIC, 3, 1, 2), (W.ELASTIC, 5, 4, 1)])
def test_rhs_parity_other_launch_shapes(dg, model, N, E, G):
    """An explicit launch shape selects the fused node-per-thread kernel at every degree (also where auto would take the
    element-per-thread kernel)."""
    case = Case(dg, _sweep_case(model, N), variant=1, elems_per_thread=E, groups_per_cta=G)
    assert case.ctx.variant_name.startswith("simt_fused")
    q32 = case.initial_fields32()
    assert_close(case.gpu_rhs(torch, q32), case.oracle_rhs(q32.astype(np.float64)), RHS_TOL, case.ctx.variant_name)


@pytest.mark.parametrize("variant", [1, 4])
def test_rhs_smooth_fields_and_slip_walls(dg, variant):
    """Smooth data (strong cancellation in D q) and the test-only SLIP tag."""
    w = W.config(3, n=3)
    w.top = W.BC_SLIP
    case = Case(dg, w, variant=variant)
    q32 = case.initial_fields32()
    assert np.abs(q32).max() > 0.1
    assert_close(case.gpu_rhs(torch, q32), case.oracle_rhs(q32.astype(np.float64)), RHS_TOL, case.ctx.variant_name)


# ---------------------------------------------------------------- config 1 exactly
def test_config1_rhs_and_100_steps(dg):
    case = Case(dg, W.config(1))
    assert case.ctx.K == 384 and case.ctx.Np == 20
    q32 = case.initial_fields32()
    assert_close(case.gpu_rhs(torch, q32), case.oracle_rhs(q32.astype(np.float64)), RHS_TOL, "config 1 r(q)")
    dt = case.dt32()
    got = case.gpu_run(torch, q32, dt, 100)
    want = case.oracle_run(q32.astype(np.float64), dt, 100)
    assert_close(got, want, RUN_TOL, "config 1 after 100 steps")
    exact = W.standing_mode(case.mesh.x, 100 * dt)
    assert np.abs(got - exact).max() < 1e-2                     # and it is the right physics


# ---------------------------------------------------------------- reduced-size trajectories of configs 2, 3, 5
@pytest.mark.parametrize("variant", [1, 4])
@pytest.mark.parametrize("cfg,n", [(2, 6), (3, 4), (5, 2)])
def test_trajectory_parity_reduced_configs(dg, cfg, n, variant):
    w = W.config(cfg, n=n)
    case = Case(dg, w, variant=variant)
    q32 = case.initial_fields32()
    dt = case.dt32()
    got = case.gpu_run(torch, q32, dt, w.nsteps)
    want = case.oracle_run(q32.astype(np.float64), dt, w.nsteps)
    assert_close(got, want, RUN_TOL, f"{w.name} {case.ctx.variant_name} after {w.nsteps} steps")


# ---------------------------------------------------------------- full-size configs: sampled elements
@pytest.mark.parametrize("cfg", [2, 3, 5])
def test_full_size_sampled_rhs(dg, cfg):
    """BASELINE.json sizes in the launch configuration bench.py times; the oracle evaluates r_k on
    sampled elements (first/last batches, boundary and interior ones) from the same global q."""
    w = W.config(cfg)
    K = w.K
    rng = np.random.default_rng(cfg)
    sample = np.unique(np.concatenate([np.arange(8), np.arange(K - 8, K), rng.integers(0, K, 48)]))
    case = Case(dg, w, only_elems=sample)
    q32 = case.initial_fields32()
    if w.ic == "pulse":
        # the pulse is ~0 away from the centre, so the whole-mesh rel-L2 of BASELINE.json lives on its
        # support: take every element that carries more than 1e-3 of the peak amplitude as well
        amp = np.abs(q32).max(axis=(1, 2))
        sample = np.unique(np.concatenate([sample, np.flatnonzero(amp > 1e-3 * amp.max())]))
        case = Case(dg, w, only_elems=sample)
    got = case.gpu_rhs(torch, q32)[sample]
    want = case.oracle_rhs(q32.astype(np.float64), sample)
    assert_close(got, want, RHS_TOL, f"{w.name} {case.ctx.variant_name} on {len(sample)} sampled elements")
    # (stage mode at full size against the oracle: test_gpu_stage_parity.py.)  One whole LSRK step: the discrete energy
    # -- a property that holds at any size, BASELINE.json north_star -- does not grow
    from oracle import timestep
    dt = case.dt32()
    out = case.gpu_run(torch, q32, dt, 1)
    assert np.isfinite(out).all()
    if w.model == W.ACOUSTIC:
        energy = lambda q: timestep.energy_acoustic(case.ref, case.mesh, *case.mats, q)   # noqa: E731
    else:
        energy = lambda q: timestep.energy_elastic(case.ref, case.mesh, *case.mats, q)    # noqa: E731
    e0, e1 = energy(q32.astype(np.float64)), energy(out.astype(np.float64))
    assert 0 < e1 <= e0 * (1 + 1e-6), (e0, e1)


# ---------------------------------------------------------------- API behaviour and edge cases
@pytest.mark.parametrize("variant", [1, 4])
def test_edge_cases_and_api_contract(dg, variant):
    w = W.config(1, n=1)                                   # K = 6: less than one batch
    case = Case(dg, w, variant=variant)
    ctx = case.ctx
    q32 = case.initial_fields32()
    assert rel_l2(case.gpu_rhs(torch, q32), case.oracle_rhs(q32.astype(np.float64))) <= RHS_TOL
    d_q = torch.from_numpy(q32).cuda()
    with pytest.raises(dg.DGError):
        ctx.rhs(d_q.data_ptr(), d_q.data_ptr())
    with pytest.raises(dg.DGError):
        ctx.rhs(0, d_q.data_ptr())
    # nsteps = 0 is a no-op
    ctx.run(d_q.data_ptr(), 1e-3, 0)
    torch.cuda.synchronize()
    assert np.array_equal(d_q.cpu().numpy(), q32) and ctx.last_launch_count == 0
    # 2 x dg_step == dg_run(2), bit for bit; launch counts 5*n (+1 copy when odd)
    dt = case.dt32()
    a = case.gpu_run(torch, q32, dt, 2)
    assert ctx.last_launch_count == 10
    d_b = torch.from_numpy(q32).cuda()
    ctx.step(d_b.data_ptr(), dt)
    assert ctx.last_launch_count == 6
    ctx.step(d_b.data_ptr(), dt)
    torch.cuda.synchronize()
    assert np.array_equal(a, d_b.cpu().numpy())
    # dg_rhs does not modify q and works on a non-default stream
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        d_q2 = torch.from_numpy(q32).cuda()
        d_r = torch.empty_like(d_q2)
        ctx.rhs(d_q2.data_ptr(), d_r.data_ptr(), s.cuda_stream)
    s.synchronize()
    assert np.array_equal(d_q2.cpu().numpy(), q32)
    assert rel_l2(d_r.cpu().numpy(), case.oracle_rhs(q32.astype(np.float64))) <= RHS_TOL


def test_zero_field_gives_zero_rhs_and_energy_decays(dg):
    w = _sweep_case(W.ELASTIC, 4)
    case = Case(dg, w)
    z = np.zeros(case.ctx.shape, dtype=np.float32)
    assert np.all(case.gpu_rhs(torch, z) == 0)
    from oracle import timestep
    q32 = case.initial_fields32()
    dt = case.dt32()
    out = case.gpu_run(torch, q32, dt, 10).astype(np.float64)
    e0 = timestep.energy_elastic(case.ref, case.mesh, *case.mats, q32.astype(np.float64))
    e1 = timestep.energy_elastic(case.ref, case.mesh, *case.mats, out)
    assert 0 < e1 < e0


@pytest.mark.parametrize("model,N,opts", [(W.ACOUSTIC, 3, {}), (W.ELASTIC, 5, {"max_ctas": 2}), (W.ELASTIC, 8, {}), (W.ACOUSTIC, 2, {}),
                                          (W.ELASTIC, 1, {}), (W.ACOUSTIC, 4, {"variant": 1}), (W.ELASTIC, 10, {"max_ctas": 4}),
                                          (W.ACOUSTIC, 3, {"variant": 5}), (W.ELASTIC, 2, {"variant": 5})])
def test_ab3_matches_paper_eq4(dg, model, N, opts):
    """The paper's own integrator (eq. (4)) as a fused epilogue of every stage-kernel family: 24 steps
    (two start-up steps, reading Q21, then 22 fused AB3 kernels -- with `max_ctas` several batches per persistent
    CTA; N = 8, 10: padded rows, N = 10: two CTAs per batch) against oracle.timestep.ab3_step; dg_ab3_run in one call, in
    two calls and step by step give the same bits."""
    from oracle import timestep
    case = Case(dg, _sweep_case(model, N), **opts)
    ctx = case.ctx
    q32 = case.initial_fields32()
    dt = case.dt32(0.05)
    stream = torch.cuda.current_stream().cuda_stream
    d_q = torch.from_numpy(q32).cuda()
    ctx.ab3_reset()
    ctx.ab3_run(d_q.data_ptr(), dt, 24, stream)
    torch.cuda.synchronize()
    npad = 2 if "pitch=" in ctx.variant_name and f"pitch={ctx.Np}," not in ctx.variant_name else 0
    assert ctx.last_launch_count == 2 * 6 + 22 + (npad if npad else 0), ctx.last_launch_count      # even number of swaps: no copy back
    q = q32.astype(np.float64)
    hist = []
    for _ in range(24):
        timestep.ab3_step(q, hist, dt, case.oracle_rhs)
    got = d_q.cpu().numpy()
    assert_close(got, q, 1e-5, f"{ctx.variant_name}: 24 AB3 steps")
    inc = rel_l2(got.astype(np.float64) - q32, q - q32)
    assert inc <= 1e-4, (ctx.variant_name, inc)
    d_b = torch.from_numpy(q32).cuda()
    ctx.ab3_reset()
    ctx.ab3_run(d_b.data_ptr(), dt, 7, stream)
    for _ in range(17):
        ctx.ab3_step(d_b.data_ptr(), dt, stream)
    torch.cuda.synchronize()
    assert np.array_equal(d_b.cpu().numpy(), got)


def test_padded_private_layout_paths(dg):
    """Degrees with Np % 4 != 0 (N = 2, 4, 8, 10): the tensor-core kernel works on a private copy of the state with
    16-byte aligned rows; dg_rhs, dg_run and dg_ab3_step convert on entry / exit.  Elastic N = 4 (Np = 35)."""
    from oracle import timestep
    case = Case(dg, _sweep_case(W.ELASTIC, 4), variant=4)
    assert "pitch=36" in case.ctx.variant_name
    q32 = case.initial_fields32()
    dt = case.dt32()
    got = case.gpu_run(torch, q32, dt, 3)
    assert case.ctx.last_launch_count == 5 * 3 + 2                  # two layout conversions around the 15 stage kernels
    assert rel_l2(got, case.oracle_run(q32.astype(np.float64), dt, 3)) <= RUN_TOL
    # dg_rhs leaves q untouched and fills every entry of rhs (no pad column leaks into the caller's arrays)
    d_q = torch.from_numpy(q32).cuda()
    d_r = torch.full_like(d_q, float("nan"))
    case.ctx.rhs(d_q.data_ptr(), d_r.data_ptr())
    torch.cuda.synchronize()
    assert case.ctx.last_launch_count == 3
    assert np.array_equal(d_q.cpu().numpy(), q32) and np.isfinite(d_r.cpu().numpy()).all()
    # the paper's AB3 step through the same conversion (two start-up steps + three fused AB3 kernels)
    dta = case.dt32(0.05)
    case.ctx.ab3_reset()
    for _ in range(5):
        case.ctx.ab3_step(d_q.data_ptr(), dta)
    torch.cuda.synchronize()
    q = q32.astype(np.float64)
    hist = []
    for _ in range(5):
        timestep.ab3_step(q, hist, dta, case.oracle_rhs)
    assert rel_l2(d_q.cpu().numpy(), q) <= 1e-5


def test_variant_selection_and_errors(dg):
    """auto picks the element-per-thread SIMT kernel at N = 1, the row-per-thread one at N = 2, the tensor-core kernel
    elsewhere; unknown variants and misaligned device buffers are rejected."""
    names = {(m, N): Case(dg, _sweep_case(m, N, n=1)).ctx.variant_name for m in (W.ACOUSTIC, W.ELASTIC) for N in (1, 2, 3)}
    assert names[(W.ACOUSTIC, 1)].startswith("simt_elem_per_thread") and names[(W.ELASTIC, 1)].startswith("simt_elem_per_thread")
    assert names[(W.ACOUSTIC, 2)].startswith("simt_row_per_thread") and names[(W.ELASTIC, 2)].startswith("simt_row_per_thread")
    assert names[(W.ACOUSTIC, 3)].startswith("tc_pipe") and names[(W.ELASTIC, 3)].startswith("tc_pipe")
    with pytest.raises(dg.DGError):
        Case(dg, _sweep_case(W.ACOUSTIC, 3, n=1), variant=2)
    with pytest.raises(dg.DGError):                                  # the row-per-thread kernel stops at N = 3
        Case(dg, _sweep_case(W.ACOUSTIC, 4, n=1), variant=5)
    case = Case(dg, _sweep_case(W.ACOUSTIC, 3, n=1), variant=4)
    buf = torch.zeros(int(np.prod(case.ctx.shape)) + 1, dtype=torch.float32, device="cuda")
    out = torch.zeros_like(buf)
    with pytest.raises(dg.DGError):                                  # q not 16-byte aligned
        case.ctx.rhs(buf.data_ptr() + 4, out.data_ptr())


@pytest.mark.parametrize("model,N", [(W.ACOUSTIC, 1), (W.ACOUSTIC, 2), (W.ELASTIC, 1)])
def test_element_per_thread_kernel_many_ctas(dg, model, N):
    """The element-per-thread kernel (variant 1 at these degrees) on a mesh of K = 162 000 elements (1 266 CTAs, ragged last
    one): r_k on sampled elements against the oracle, and one LSRK step with non-increasing energy (its stage mode is
    compared with the oracle in test_gpu_stage_parity.py)."""
    from oracle import timestep
    w = W.config(4, N=N, model=model, n=30)
    w.ic = "random"
    K = w.K
    rng = np.random.default_rng(N)
    sample = np.unique(np.concatenate([np.arange(8), np.arange(K - 8, K), rng.integers(0, K, 48)]))
    case = Case(dg, w, only_elems=sample, variant=1)
    assert case.ctx.variant_name.startswith("simt_elem_per_thread")
    q32 = case.initial_fields32()
    got = case.gpu_rhs(torch, q32)[sample]
    want = case.oracle_rhs(q32.astype(np.float64), sample)
    assert_close(got, want, RHS_TOL, case.ctx.variant_name)
    out = case.gpu_run(torch, q32, case.dt32(), 1)
    assert np.isfinite(out).all()
    energy = timestep.energy_acoustic if model == W.ACOUSTIC else timestep.energy_elastic
    e0 = energy(case.ref, case.mesh, *case.mats, q32.astype(np.float64))
    e1 = energy(case.ref, case.mesh, *case.mats, out.astype(np.float64))
    assert 0 < e1 <= e0 * (1 + 1e-6), (e0, e1)
