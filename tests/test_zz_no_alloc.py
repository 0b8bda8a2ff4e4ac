"""dg_step_static (include/dg.h): the LSRK step whose work memory is the library's file-scope static device array
instead of buffers from cudaMalloc -- for callers that must not allocate.  Checked against the existing path (dg_step) on
the same seeded inputs, two calls in a row (the second call finds the first one's leftovers in the array), on every
stage-kernel family incl. the padded-row case, plus the size limit.  The file sorts last on purpose: the suite runs
with `pytest -x`, and a failure here must not hide the parity tests.
"""
import numpy as np
import pytest

from paper_1602_07997_b200 import workloads as W

from gpu_common import RHS_TOL, Case, assert_close

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def dg():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_1602_07997_b200 import dg as mod          # raises if libdg.so is missing: no fallback
    return mod


def _case(model, N, n):
    w = W.config(4, N=N, model=model, n=n)
    w.jitter, w.top, w.ic = 0.08, W.BC_FREE, "random"
    return w


# element per thread; row per thread (persistent warps); tensor core; tensor core with padded rows (Np = 35 -> pitch 36);
# fused node-per-thread SIMT; tensor core with the interface-centric surface step
@pytest.mark.parametrize("model,N,n,opts,kernel", [
    (W.ACOUSTIC, 1, 8, {}, "simt_elem_per_thread"),
    (W.ELASTIC, 2, 6, {}, "simt_row_per_thread"),
    (W.ACOUSTIC, 5, 6, {}, "tc_pipe"),
    (W.ELASTIC, 4, 5, {}, "tc_pipe"),
    (W.ACOUSTIC, 3, 5, {"variant": 1}, "simt_fused"),
    (W.ELASTIC, 3, 4, {"surface": 1}, "tc_pipe"),
    (W.ACOUSTIC, 2, 1, {}, "simt_row_per_thread"),          # K = 6: less than one tile / one CTA
    (W.ELASTIC, 1, 1, {}, "simt_elem_per_thread"),
    (W.ELASTIC, 10, 2, {}, "tc_pipe"),                      # padded rows (Np = 286 -> 288), two CTAs per batch
])
def test_step_static_matches_step_two_calls_in_a_row(dg, model, N, n, opts, kernel):
    case = Case(dg, _case(model, N, n), only_elems=np.arange(4), **opts)
    ctx = case.ctx
    assert ctx.variant_name.startswith(kernel)
    need = (3 if "pitch=" in ctx.variant_name and f"pitch={ctx.Np}," not in ctx.variant_name else 2) * 4 * int(np.prod(ctx.shape))
    assert need < dg.STATIC_SCRATCH_BYTES
    q32 = case.initial_fields32()
    dt = case.dt32()
    stream = torch.cuda.current_stream().cuda_stream
    d_ref = torch.from_numpy(q32).cuda()
    d_new = torch.from_numpy(q32).cuda()
    for call in (1, 2):
        ctx.step(d_ref.data_ptr(), dt, stream)                     # the existing path: context-owned residual / ping-pong
        ctx.step_static(d_new.data_ptr(), dt, stream)              # the same step on the static array
        torch.cuda.synchronize()
        want, got = d_ref.cpu().numpy(), d_new.cpu().numpy()
        assert_close(got, want, RHS_TOL, f"{ctx.variant_name}: dg_step_static vs dg_step, call {call}")
        assert np.array_equal(got, want), f"{ctx.variant_name}: call {call}: same kernels, same order: the bits must agree"
    assert not np.array_equal(d_new.cpu().numpy(), q32)             # (the steps did move the state)


def test_step_static_ignores_what_earlier_calls_left_in_the_array(dg):
    """A larger context runs first and leaves its residual / state in the array; the smaller one's step must not see it
    (padded rows: the pad columns it relies on being zero were written by the other context)."""
    big = Case(dg, _case(W.ACOUSTIC, 5, 8), only_elems=np.arange(4))
    small = Case(dg, _case(W.ELASTIC, 4, 4), only_elems=np.arange(4))
    stream = torch.cuda.current_stream().cuda_stream
    d_big = torch.from_numpy(big.initial_fields32()).cuda()
    big.ctx.step_static(d_big.data_ptr(), big.dt32(), stream)
    q32 = small.initial_fields32()
    d_ref, d_new = torch.from_numpy(q32).cuda(), torch.from_numpy(q32).cuda()
    small.ctx.step(d_ref.data_ptr(), small.dt32(), stream)
    small.ctx.step_static(d_new.data_ptr(), small.dt32(), stream)
    torch.cuda.synchronize()
    assert np.isfinite(d_new.cpu().numpy()).all()
    assert np.array_equal(d_new.cpu().numpy(), d_ref.cpu().numpy())


def test_step_static_rejects_sizes_beyond_the_static_array(dg):
    case = Case(dg, _case(W.ACOUSTIC, 3, 24), only_elems=np.arange(4))     # K = 82 944: 2 x 26.5 MB of work memory
    ctx = case.ctx
    assert 2 * 4 * int(np.prod(ctx.shape)) > dg.STATIC_SCRATCH_BYTES
    d_q = torch.zeros(ctx.shape, dtype=torch.float32, device="cuda")
    d_q += 1.0
    with pytest.raises(dg.DGError, match="DG_STATIC_SCRATCH_BYTES"):
        ctx.step_static(d_q.data_ptr(), 1e-3, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert bool((d_q == 1.0).all())                                    # nothing was enqueued
    ctx.step(d_q.data_ptr(), case.dt32(), torch.cuda.current_stream().cuda_stream)   # the allocating path still serves it
    torch.cuda.synchronize()
    assert bool(torch.isfinite(d_q).all())
