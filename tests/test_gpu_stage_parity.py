"""GPU parity of the LSRK stage mode (row a7 fused into the stage kernels): libdg through the C ABI against the
fp64 oracle, at every degree on the kernel `auto` picks, with persistent CTAs that loop over several batches, and at
BASELINE.json's full sizes on sampled elements through the one-stage entry point dg_stage.

Tolerances: BASELINE.json north_star -- rel-L2 <= 2e-6 per RHS evaluation, <= 1e-4 after the LSRK run; a single LSRK
step (five evaluations, q = q0 + O(dt r)) must agree to 2e-6 in q as well.
"""
import re

import numpy as np
import pytest

from oracle import timestep
from paper_1602_07997_b200 import workloads as W

from gpu_common import RHS_TOL, RUN_TOL, Case, assert_close, describe, rel_l2

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

A, B = timestep.LSRK_A, timestep.LSRK_B


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


def _increment_error(got, want, before):
    """Error of the step's increment relative to the increment's norm, after discounting what storing q in fp32 costs:
    |got - want| <= tol |want - before| + 2^-23 |want|.  Returns the left-over as a multiple of |want - before|.
    (On the pulse workloads the increment of p in stage 2 is below one ulp of p: the storage rounding alone is 2e-4 of the
    increment's norm there, while a wrong A_s / B_s / residual carry is O(1) of it.)"""
    got, want, before = (np.asarray(a, dtype=np.float64) for a in (got, want, before))
    err = np.linalg.norm((got - want).ravel()) - 2.0 ** -23 * np.linalg.norm(want.ravel())
    return max(err, 0.0) / max(np.linalg.norm((want - before).ravel()), 1e-300)


def _info(name, key):
    m = re.search(key + r"=(\d+)", name)
    return int(m.group(1)) if m else None


# ---------------------------------------------------------------- LSRK trajectory, every degree, the kernel auto picks
@pytest.mark.parametrize("N", range(1, 11))
@pytest.mark.parametrize("model", [W.ACOUSTIC, W.ELASTIC])
def test_run_parity_every_degree_auto(dg, model, N):
    """dg_run against oracle.timestep.lsrk_run for N = 1..10, both models, on the variant dg_create picks by itself
    (element-per-thread SIMT kernel at N = 1, row-per-thread at N = 2, tensor-core kernel elsewhere): one step to 2e-6,
    three steps to 1e-4.  K = 162, random fields, random discontinuous materials, free top."""
    case = Case(dg, _sweep_case(model, N))
    q32 = case.initial_fields32()
    q64 = q32.astype(np.float64)
    dt = case.dt32()
    one = case.gpu_run(torch, q32, dt, 1)
    want1 = case.oracle_run(q64, dt, 1)
    assert_close(one, want1, RHS_TOL, f"{case.ctx.variant_name}: one LSRK step")
    # the increment of the step is what the five stages computed: a wrong A_s / B_s / residual carry shows here at O(1)
    inc = _increment_error(one, want1, q64)
    assert inc <= 2e-5, f"{case.ctx.variant_name}: increment of one step off by {inc:.3e}; {describe(one, want1)}"
    three = case.gpu_run(torch, q32, dt, 3)
    assert_close(three, case.oracle_run(q64, dt, 3), RUN_TOL, f"{case.ctx.variant_name}: three LSRK steps")


@pytest.mark.parametrize("N", range(1, 4))
@pytest.mark.parametrize("model", [W.ACOUSTIC, W.ELASTIC])
def test_run_parity_row_per_thread(dg, model, N):
    """The same trajectory check for variant 5 (row-per-thread kernel, N <= 3): one LSRK step to 2e-6 with the increment
    check, three steps to 1e-4."""
    case = Case(dg, _sweep_case(model, N), variant=5)
    assert case.ctx.variant_name.startswith("simt_row_per_thread")
    q32 = case.initial_fields32()
    q64 = q32.astype(np.float64)
    dt = case.dt32()
    one = case.gpu_run(torch, q32, dt, 1)
    want1 = case.oracle_run(q64, dt, 1)
    assert_close(one, want1, RHS_TOL, f"{case.ctx.variant_name}: one LSRK step")
    inc = _increment_error(one, want1, q64)
    assert inc <= 2e-5, f"{case.ctx.variant_name}: increment of one step off by {inc:.3e}; {describe(one, want1)}"
    assert_close(case.gpu_run(torch, q32, dt, 3), case.oracle_run(q64, dt, 3), RUN_TOL, f"{case.ctx.variant_name}: three LSRK steps")


# ---------------------------------------------------------------- persistent CTAs over several batches (tensor-core kernel)
@pytest.mark.parametrize("N", range(1, 11))
@pytest.mark.parametrize("model", [W.ACOUSTIC, W.ELASTIC])
def test_stage_parity_several_batches_per_cta(dg, model, N):
    """The tensor-core kernel with its grid capped (dg_options.max_ctas) so that every persistent CTA works through
    >= 3 batches, the last one ragged: exercises the double-buffered tile slots, the alternating accumulator sets, the
    phase wrap of every mbarrier ring, the epilogue's two-chunks-ahead TMA prefetch across batch boundaries and the L2
    prefetch of the residual -- the paths the kernel takes at full size -- against the full oracle (RHS mode and two LSRK
    steps)."""
    w = _sweep_case(model, N)
    probe = Case(dg, w, variant=4)
    nsplit = _info(probe.ctx.variant_name, "nsplit")
    eb = _info(probe.ctx.variant_name, "elems/batch")
    probe.ctx.close()
    case = Case(dg, w, variant=4, max_ctas=2 * nsplit)
    K = case.ctx.K
    nbatch = -(-K // eb)
    assert nbatch // 2 >= 3 and K % eb != 0, (K, eb)          # >= 3 batches per CTA and a ragged last batch
    q32 = case.initial_fields32()
    q64 = q32.astype(np.float64)
    assert_close(case.gpu_rhs(torch, q32), case.oracle_rhs(q64), RHS_TOL, f"{case.ctx.variant_name}: r(q), {nbatch} batches on 2 workers")
    dt = case.dt32()
    got = case.gpu_run(torch, q32, dt, 2)
    want = case.oracle_run(q64, dt, 2)
    assert_close(got, want, 1e-5, f"{case.ctx.variant_name}: two LSRK steps, {nbatch} batches on 2 workers")
    # one worker (pair): every batch of the mesh on the same CTA
    one = Case(dg, w, variant=4, max_ctas=nsplit)
    assert np.array_equal(one.gpu_run(torch, q32, dt, 2), got), "result depends on how batches are dealt to CTAs"


@pytest.mark.parametrize("model,N,n,steps", [(W.ACOUSTIC, 3, 14, 2), (W.ACOUSTIC, 5, 14, 2), (W.ELASTIC, 3, 11, 2), (W.ELASTIC, 7, 11, 1)])
def test_stage_parity_natural_grid_three_batches_per_cta(dg, model, N, n, steps):
    """The same with the grid the library launches by itself (one CTA per SM): meshes large enough that each of the 148
    persistent CTAs gets >= 3 batches (acoustic K = 16 464 > 148 x 32 x 3; elastic K = 7 986 > 148 x 14 x 3), full oracle."""
    w = _sweep_case(model, N, n=n)
    case = Case(dg, w)
    assert case.ctx.variant_name.startswith("tc_pipe")
    eb = _info(case.ctx.variant_name, "elems/batch")
    assert -(-case.ctx.K // eb) >= 3 * 148
    q32 = case.initial_fields32()
    dt = case.dt32()
    got = case.gpu_run(torch, q32, dt, steps)
    want = case.oracle_run(q32.astype(np.float64), dt, steps)
    assert_close(got, want, 1e-5, f"{case.ctx.variant_name}: {steps} LSRK step(s) on K = {case.ctx.K}")


# ---------------------------------------------------------------- full size: one stage at a time on sampled elements
def _sample(K, eb, rng, nrand=160):
    """First / last elements, one element of each of ~nrand evenly spread batches (so that every region of the batch
    sequence -- and with it every persistent CTA's early, middle and late batches -- is hit) and random ones."""
    nb = -(-K // eb)
    spread = (np.linspace(0, nb - 1, min(nb, nrand)).astype(np.int64) * eb + rng.integers(0, eb, min(nb, nrand))).clip(0, K - 1)
    return np.unique(np.concatenate([np.arange(8), np.arange(K - 8, K), spread, rng.integers(0, K, 64)]))


def _two_stages_sampled(dg, w, sample_extra=None, **opts):
    """Stage 1 (A_1 = 0) and stage 2 (carries the residual) of the LSRK step through dg_stage on the full mesh; the
    oracle evaluates r_k on the sampled elements from the same global state:
        q1 = q0 + B_1 dt r(q0);   q2 = q1 + B_2 (A_2 dt r(q0) + dt r(q1))."""
    K = w.K
    rng = np.random.default_rng(w.N + 17 * w.model)
    probe = dg.from_workload(W.config(4, N=w.N, model=w.model, n=1), device=0, **opts)
    eb = _info(probe.variant_name, "elems/batch") or 128
    probe.close()
    sample = _sample(K, eb, rng)
    if sample_extra is not None:
        sample = np.unique(np.concatenate([sample, sample_extra(w)]))
    case = Case(dg, w, only_elems=sample, **opts)
    q0 = case.initial_fields32()
    dt = case.dt32()
    q1, d_q1 = case.gpu_stage(torch, q0, 0.0, B[0], dt)
    r0 = case.oracle_rhs(q0.astype(np.float64), sample)
    want1 = q0[sample].astype(np.float64) + np.float32(B[0]) * np.float64(dt) * r0
    name = case.ctx.variant_name
    assert_close(q1[sample], want1, RHS_TOL, f"{name}: stage 1 on {len(sample)} sampled elements of K = {K}")
    inc1 = _increment_error(q1[sample], want1, q0[sample])
    q2, _ = case.gpu_stage(torch, None, A[1], B[1], dt, d_in=d_q1)
    r1 = case.oracle_rhs(q1.astype(np.float64), sample)          # from the GPU's own q1: isolates stage 2
    res2 = np.float32(A[1]) * (np.float64(dt) * r0) + np.float64(dt) * r1
    want2 = q1[sample].astype(np.float64) + np.float32(B[1]) * res2
    assert_close(q2[sample], want2, RHS_TOL, f"{name}: stage 2 (residual carried) on sampled elements of K = {K}")
    inc2 = _increment_error(q2[sample], want2, q1[sample])
    assert max(inc1, inc2) <= 5e-5, f"{name}: stage increments off by {inc1:.3e} / {inc2:.3e}"
    # everything outside the sample at least finite, and nothing left unwritten (the output started as NaN)
    assert np.isfinite(q1).all() and np.isfinite(q2).all()
    return case


def _pulse_support(w):
    vx, et, bc, cell = w.mesh()
    cen = vx[et].mean(axis=1)
    return np.flatnonzero(np.linalg.norm(cen - 0.5, axis=1) < 0.2)


@pytest.mark.parametrize("cfg", [2, 3, 5])
def test_full_size_stage_mode_sampled(dg, cfg):
    """BASELINE.json sizes in the launch configuration bench.py times (148 persistent CTAs, 81 / 78 / 40 batches each)."""
    w = W.config(cfg)
    _two_stages_sampled(dg, w, sample_extra=_pulse_support if w.ic == "pulse" else None)


@pytest.mark.parametrize("model,N", [(W.ACOUSTIC, 1), (W.ACOUSTIC, 2), (W.ELASTIC, 1)])
def test_element_per_thread_stage_mode_sampled(dg, model, N):
    """The element-per-thread kernel (variant 1 at these degrees) in stage mode on K = 162 000 elements (1 266 CTAs)."""
    w = W.config(4, N=N, model=model, n=30)
    w.ic = "random"
    case = _two_stages_sampled(dg, w, variant=1)
    assert case.ctx.variant_name.startswith("simt_elem_per_thread")


# ---------------------------------------------------------------- full size: every element, kernel against kernel
@pytest.mark.parametrize("cfg", [2, 3, 5])
def test_full_size_tensor_core_vs_simt_every_element(dg, cfg):
    """Two LSRK steps at full size on the tensor-core kernel and on the fused FP32 SIMT kernel (oracle-pinned on the small
    meshes above): every element compared, so a defect confined to batches the sampled tests miss cannot hide."""
    w = W.config(cfg)
    a = dg.from_workload(w, device=0, variant=4)
    xyz = a.node_coords()
    q32 = w.initial_fields(xyz).astype(np.float32)
    del xyz
    dt = float(np.float32(a.stable_dt(0.5)))
    d_a = torch.from_numpy(q32).cuda()
    a.run(d_a.data_ptr(), dt, 2)
    torch.cuda.synchronize()
    a.close()
    b = dg.from_workload(w, device=0, variant=1)
    d_b = torch.from_numpy(q32).cuda()
    b.run(d_b.data_ptr(), dt, 2)
    torch.cuda.synchronize()
    b.close()
    diff = (d_a - d_b).double()
    err = float(diff.norm() / d_b.double().norm())
    worst = int(diff.abs().amax(dim=(1, 2)).argmax())
    assert err <= 1e-5, f"{w.name}: tensor-core vs SIMT after two steps rel-L2 {err:.3e}, worst element {worst}"
    inc = float(diff.norm() / (d_b - torch.from_numpy(q32).cuda()).double().norm())
    assert inc <= 1e-4, f"{w.name}: increments differ by {inc:.3e}, worst element {worst}"


@pytest.mark.parametrize("model,N", [(W.ACOUSTIC, 1), (W.ACOUSTIC, 2), (W.ELASTIC, 1)])
def test_element_per_thread_vs_node_per_thread_every_element(dg, model, N):
    w = W.config(4, N=N, model=model, n=30)
    w.ic = "random"
    out = []
    for opts in ({"variant": 1}, {"variant": 1, "elems_per_thread": 1}):
        ctx = dg.from_workload(w, device=0, **opts)
        if not out:
            q32 = w.initial_fields(ctx.node_coords()).astype(np.float32)
            dt = float(np.float32(ctx.stable_dt(0.5)))
        d = torch.from_numpy(q32).cuda()
        ctx.run(d.data_ptr(), dt, 2)
        torch.cuda.synchronize()
        out.append((ctx.variant_name, d))
        ctx.close()
    assert out[0][0].startswith("simt_elem_per_thread") and out[1][0].startswith("simt_fused")
    err = float((out[0][1] - out[1][1]).double().norm() / out[1][1].double().norm())
    assert err <= 1e-5, (out[0][0], out[1][0], err)


@pytest.mark.parametrize("model,N,opts", [(W.ACOUSTIC, 2, {}), (W.ELASTIC, 2, {}), (W.ACOUSTIC, 3, {"variant": 5}), (W.ELASTIC, 1, {"variant": 5})])
def test_row_per_thread_stage_mode_sampled(dg, model, N, opts):
    """The row-per-thread kernel (auto at N = 2) in stage mode on K = 162 000 elements: every persistent warp walks over
    several tiles through its two shared-memory slots (cp.async prefetch of the next tile), ragged last tile."""
    w = W.config(4, N=N, model=model, n=30)
    w.ic = "random"
    case = _two_stages_sampled(dg, w, **opts)
    assert case.ctx.variant_name.startswith("simt_row_per_thread")


@pytest.mark.parametrize("model,N", [(W.ACOUSTIC, 2), (W.ELASTIC, 2)])
def test_row_per_thread_vs_node_per_thread_every_element(dg, model, N):
    """Two LSRK steps on K = 162 000 elements, row-per-thread kernel against the fused node-per-thread kernel, every value."""
    w = W.config(4, N=N, model=model, n=30)
    w.ic = "random"
    out = []
    for opts in ({}, {"variant": 1, "elems_per_thread": 1}):
        ctx = dg.from_workload(w, device=0, **opts)
        if not out:
            q32 = w.initial_fields(ctx.node_coords()).astype(np.float32)
            dt = float(np.float32(ctx.stable_dt(0.5)))
        d = torch.from_numpy(q32).cuda()
        ctx.run(d.data_ptr(), dt, 2)
        torch.cuda.synchronize()
        out.append((ctx.variant_name, d))
        ctx.close()
    assert out[0][0].startswith("simt_row_per_thread") and out[1][0].startswith("simt_fused")
    err = float((out[0][1] - out[1][1]).double().norm() / out[1][1].double().norm())
    assert err <= 1e-5, (out[0][0], out[1][0], err)


# ---------------------------------------------------------------- multi-rate hook: a stage restricted to an element range
@pytest.mark.parametrize("model,N,opts", [(W.ACOUSTIC, 1, {}), (W.ACOUSTIC, 3, {}), (W.ELASTIC, 3, {}), (W.ELASTIC, 5, {"max_ctas": 2}),
                                          (W.ELASTIC, 9, {}), (W.ACOUSTIC, 4, {"variant": 1}), (W.ELASTIC, 2, {"variant": 1}),
                                          (W.ACOUSTIC, 3, {"variant": 5}), (W.ELASTIC, 2, {"variant": 5}), (W.ELASTIC, 1, {}), (W.ACOUSTIC, 2, {"variant": 1})])
def test_stage_range_composes_to_the_full_stage(dg, model, N, opts):
    """dg_stage_range over [0, k1), [k1, k2), [k2, K) -- the per-level launches of a multi-rate driver
    -- writes exactly what one dg_stage over the mesh writes, touches nothing outside its range (q_out and the residual),
    and agrees with the oracle's r_k on the range."""
    case = Case(dg, _sweep_case(model, N), **opts)
    ctx = case.ctx
    al = ctx.range_alignment
    K = ctx.K
    k1, k2 = al * max(1, (K // 3) // al), al * max(2, (2 * K // 3) // al)
    assert 0 < k1 < k2 < K
    q32 = case.initial_fields32()
    dt = case.dt32()
    stream = torch.cuda.current_stream().cuda_stream
    d_q = torch.from_numpy(q32).cuda()
    full1, d_full1 = case.gpu_stage(torch, q32, 0.0, B[0], dt)
    full2, _ = case.gpu_stage(torch, None, A[1], B[1], dt, d_in=d_full1)
    # the same two stages, range by range
    d_o1 = torch.full_like(d_q, float("nan"))
    ctx.stage_range(d_q.data_ptr(), d_o1.data_ptr(), 0.0, B[0], dt, k1, k2, stream)
    torch.cuda.synchronize()
    part = d_o1.cpu().numpy()
    assert np.isnan(part[:k1]).all() and np.isnan(part[k2:]).all(), "dg_stage_range wrote outside its range"
    assert np.array_equal(part[k1:k2], full1[k1:k2])
    want = q32[k1:k2].astype(np.float64) + np.float32(B[0]) * np.float64(dt) * case.oracle_rhs(q32.astype(np.float64), np.arange(k1, k2))
    assert_close(part[k1:k2], want, RHS_TOL, f"{ctx.variant_name}: stage on elements [{k1}, {k2})")
    for lo, hi in ((0, k1), (k2, K)):
        ctx.stage_range(d_q.data_ptr(), d_o1.data_ptr(), 0.0, B[0], dt, lo, hi, stream)
    torch.cuda.synchronize()
    assert np.array_equal(d_o1.cpu().numpy(), full1)
    d_o2 = torch.full_like(d_q, float("nan"))
    for lo, hi in ((k2, K), (0, k1), (k1, k2)):                 # any order: ranges are independent within a stage
        ctx.stage_range(d_o1.data_ptr(), d_o2.data_ptr(), A[1], B[1], dt, lo, hi, stream)
    torch.cuda.synchronize()
    assert np.array_equal(d_o2.cpu().numpy(), full2), "residual carried differently range by range"
    ctx.stage_range(d_q.data_ptr(), d_o1.data_ptr(), 0.0, B[0], dt, k1, k1, stream)     # empty range: no-op
    assert ctx.last_launch_count == 0
    with pytest.raises(dg.DGError):
        ctx.stage_range(d_q.data_ptr(), d_o1.data_ptr(), 0.0, B[0], dt, k1 + (1 if al > 1 else K + 1), k2, stream)
    with pytest.raises(dg.DGError):
        ctx.stage_range(d_q.data_ptr(), d_q.data_ptr(), 0.0, B[0], dt, 0, K, stream)


def test_stage_range_is_refused_on_padded_rows(dg):
    case = Case(dg, _sweep_case(W.ELASTIC, 4), variant=4)
    d = torch.zeros(case.ctx.shape, dtype=torch.float32, device="cuda")
    o = torch.zeros_like(d)
    with pytest.raises(dg.DGError):
        case.ctx.stage_range(d.data_ptr(), o.data_ptr(), 0.0, 1.0, 1e-3, 0, case.ctx.K)


# ---------------------------------------------------------------- interface-centric surface step
@pytest.mark.parametrize("model,N,opts", [(W.ACOUSTIC, 1, {}), (W.ELASTIC, 1, {}), (W.ACOUSTIC, 2, {}), (W.ELASTIC, 2, {}),
                                          (W.ACOUSTIC, 3, {}), (W.ELASTIC, 3, {"max_ctas": 2}), (W.ACOUSTIC, 5, {"max_ctas": 2}),
                                          (W.ELASTIC, 4, {}), (W.ELASTIC, 7, {}), (W.ACOUSTIC, 10, {"max_ctas": 4}),
                                          (W.ACOUSTIC, 3, {"variant": 1}), (W.ELASTIC, 2, {"variant": 1}),
                                          (W.ACOUSTIC, 2, {"variant": 5}), (W.ELASTIC, 3, {"variant": 5})])
def test_interface_centric_surface_step(dg, model, N, opts):
    """dg_options.surface = 1: the paper's SGEMM-strategy surface kernel -- one thread per interface face node computes the
    penalty terms of both sides once into a face buffer, boundary faces behind the interior ones -- as the producer of rows
    a4 + a5 for each stage-kernel family (element per thread, tensor core, fused SIMT, row per thread): r(q), two LSRK steps and five AB3
    steps against the oracle, and against the element-centric default (same formulas per side: agreement to rounding)."""
    w = _sweep_case(model, N)
    w.top = W.BC_SLIP if model == W.ELASTIC else W.BC_FREE          # rigid, and free / slip faces among the boundary ones
    case = Case(dg, w, surface=1, **opts)
    assert "interface-centric" in case.ctx.variant_name
    q32 = case.initial_fields32()
    q64 = q32.astype(np.float64)
    got = case.gpu_rhs(torch, q32)
    assert case.ctx.last_launch_count in (2, 4)                      # interface kernel + stage kernel (+ two layout conversions)
    assert_close(got, case.oracle_rhs(q64), RHS_TOL, f"{case.ctx.variant_name}: r(q)")
    ref = Case(dg, w, **opts)
    base = ref.gpu_rhs(torch, q32)
    assert rel_l2(got, base) <= 2e-7, (case.ctx.variant_name, rel_l2(got, base))
    dt = case.dt32()
    assert_close(case.gpu_run(torch, q32, dt, 2), case.oracle_run(q64, dt, 2), 1e-5, f"{case.ctx.variant_name}: two LSRK steps")
    from oracle import timestep as ts
    d_q = torch.from_numpy(q32).cuda()
    dta = case.dt32(0.05)
    case.ctx.ab3_run(d_q.data_ptr(), dta, 5)
    torch.cuda.synchronize()
    q, hist = q64.copy(), []
    for _ in range(5):
        ts.ab3_step(q, hist, dta, case.oracle_rhs)
    assert_close(d_q.cpu().numpy(), q, 1e-5, f"{case.ctx.variant_name}: five AB3 steps")


# ---------------------------------------------------------------- multi-GPU form on one GPU: two partitions, halo exchange
@pytest.mark.parametrize("model,N,opts", [(W.ACOUSTIC, 1, {}), (W.ACOUSTIC, 3, {}), (W.ELASTIC, 4, {}), (W.ELASTIC, 6, {"max_ctas": 2}),
                                          (W.ACOUSTIC, 9, {}), (W.ELASTIC, 2, {"variant": 1}), (W.ACOUSTIC, 3, {"surface": 1})])
def test_two_partitions_with_halo_exchange_match_single_domain(dg, model, N, opts):
    """The path as it would run on two GPUs, emulated rank after rank on one: each rank's context holds
    its slab of the element list plus ghost copies (dg_partition_*, dg_options.owned_elements); before every LSRK stage the
    face traces of the cut faces are packed (dg_halo_pack), handed to the peer (here: a device copy where NCCL send/recv
    would be) and unpacked into its ghosts (dg_halo_unpack); dg_stage then advances the owned elements.  Two steps must
    reproduce the single-domain result bit for bit -- ghosts start as NaN, so nothing but exchanged traces is ever read."""
    w = _sweep_case(model, N)
    vxyz, etov, bc, cell = w.mesh()
    mats = w.material_arrays(cell)
    single = Case(dg, w, **opts)
    q32 = single.initial_fields32()
    dt = single.dt32()
    want = single.gpu_run(torch, q32, dt, 2)
    stream = torch.cuda.current_stream().cuda_stream
    ranks = []
    for r in range(2):
        part = dg.Partition(vxyz, etov, bc, 2, r)
        ids, no = part.global_ids, part.num_owned
        ctx = dg.Context(vxyz, part.etov, N, model, mats[0][ids], mats[1][ids], mats[2][ids] if model == W.ELASTIC else None,
                         part.bc, device=0, owned_elements=no, **opts)
        assert ctx.K_owned == no and ctx.K == len(ids) and part.num_ghost > 0
        q = q32[ids].copy()
        q[no:] = np.nan
        cur = torch.from_numpy(q).cuda()
        nxt = torch.full_like(cur, float("nan"))
        peers = [(peer, torch.from_numpy(s).cuda(), torch.from_numpy(rv).cuda(),
                  torch.empty(len(s) * ctx.NF * ctx.Nfp, device="cuda"), torch.empty(len(rv) * ctx.NF * ctx.Nfp, device="cuda"))
                 for peer, s, rv in part.peers]
        assert [p[0] for p in peers] == [1 - r]
        ranks.append(dict(part=part, ctx=ctx, cur=cur, nxt=nxt, peers=peers))
    for step in range(2):
        for s in range(5):
            for rk in ranks:                                       # pack on every rank
                for peer, send, recv, sbuf, rbuf in rk["peers"]:
                    rk["ctx"].halo_pack(rk["cur"].data_ptr(), send.data_ptr(), send.numel(), sbuf.data_ptr(), stream)
            for r, rk in enumerate(ranks):                         # "send / recv": my receive buffer is the peer's send buffer
                for peer, send, recv, sbuf, rbuf in rk["peers"]:
                    other = [p for p in ranks[peer]["peers"] if p[0] == r][0]
                    assert other[3].numel() == rbuf.numel()
                    rbuf.copy_(other[3])
                    rk["ctx"].halo_unpack(rk["cur"].data_ptr(), recv.data_ptr(), recv.numel(), rbuf.data_ptr(), stream)
            for rk in ranks:
                rk["ctx"].stage(rk["cur"].data_ptr(), rk["nxt"].data_ptr(), A[s], B[s], dt, stream)
                rk["cur"], rk["nxt"] = rk["nxt"], rk["cur"]
    torch.cuda.synchronize()
    for rk in ranks:
        ids, no = rk["part"].global_ids, rk["part"].num_owned
        got = rk["cur"].cpu().numpy()[:no]
        assert np.isfinite(got).all(), "a ghost value that was never exchanged reached an owned element"
        assert np.array_equal(got, want[ids[:no]]), f"rank {rk['part'].rank}: {describe(got, want[ids[:no]])}"
    halo_bytes = sum(4 * (p[3].numel() + p[4].numel()) for rk in ranks for p in rk["peers"])
    state_bytes = 4 * q32.size
    assert halo_bytes < state_bytes                                # only traces of the cut faces move


# ---------------------------------------------------------------- full size: the optional paths, kernel against kernel
@pytest.mark.parametrize("cfg", [2, 3])
def test_full_size_ab3_and_interface_paths_every_element(dg, cfg):
    """BASELINE.json sizes: (1) six steps of the paper's AB3 integrator (two start-up steps, four fused AB3 kernels; 81 / 78
    batches per persistent CTA) on the tensor-core kernel against the fused SIMT kernel, which the small-mesh tests pin to
    the oracle; (2) two LSRK steps with the interface-centric surface kernel against the element-centric default.  Every
    element is compared."""
    w = W.config(cfg)
    outs = {}
    q32 = dt = None
    for name, opts, what in (("tc_ab3", {"variant": 4}, "ab3"), ("simt_ab3", {"variant": 1}, "ab3"),
                             ("tc", {"variant": 4}, "lsrk"), ("tc_iface", {"variant": 4, "surface": 1}, "lsrk")):
        ctx = dg.from_workload(w, device=0, **opts)
        if q32 is None:
            q32 = w.initial_fields(ctx.node_coords()).astype(np.float32)
            dt = float(np.float32(ctx.stable_dt(0.5)))
        d = torch.from_numpy(q32).cuda()
        if what == "ab3":
            ctx.ab3_run(d.data_ptr(), 0.1 * dt, 6)
        else:
            ctx.run(d.data_ptr(), dt, 2)
        torch.cuda.synchronize()
        outs[name] = d
        ctx.close()
    d0 = torch.from_numpy(q32).cuda()
    for a, b in (("tc_ab3", "simt_ab3"), ("tc_iface", "tc")):
        diff = (outs[a] - outs[b]).double()
        err = float(diff.norm() / outs[b].double().norm())
        inc = float(diff.norm() / (outs[b] - d0).double().norm())
        worst = int(diff.abs().amax(dim=(1, 2)).argmax())
        assert err <= 1e-5 and inc <= 2e-4, f"{w.name}: {a} vs {b}: rel-L2 {err:.3e}, of the increment {inc:.3e}, worst element {worst}"
