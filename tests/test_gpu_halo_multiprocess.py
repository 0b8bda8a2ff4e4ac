"""The multi-GPU form of the path across real processes: two ranks (here both on cuda:0, as only one GPU is at hand; on a
multi-GPU node each takes its own device and the backend is NCCL), torch.distributed for the exchange (gloo, staged through
host memory), libdg for everything else -- partition, pack, unpack, stage.  Two LSRK steps of halo.HaloExchanger.run_lsrk
must reproduce the single-process, single-domain dg_run bit for bit.  The ranks never wait on one another on the device
(every exchange is a host-side send / recv after a stream synchronise), so sharing one GPU is safe."""
import os
import sys

import numpy as np
import pytest

from paper_1602_07997_b200 import workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _case(model, N):
    w = W.config(4, N=N, model=model, n=3)
    w.jitter, w.top, w.ic = 0.08, W.BC_FREE, "random"
    return w


def _rank_main(rank, world, port, model, N, dt, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from paper_1602_07997_b200 import dg, halo
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = _case(model, N)
    vxyz, etov, bc, cell = w.mesh()
    mats = w.material_arrays(cell)
    part = dg.Partition(vxyz, etov, bc, world, rank)
    ids, no = part.global_ids, part.num_owned
    ctx = dg.Context(vxyz, part.etov, N, model, mats[0][ids], mats[1][ids], mats[2][ids] if model == W.ELASTIC else None, part.bc,
                     device=0, owned_elements=no)
    q = w.initial_fields(None).astype(np.float32)[ids]            # random fields: node coordinates are not needed
    q[no:] = np.nan
    d_q = torch.from_numpy(q).cuda()
    hx = halo.HaloExchanger(part, ctx, torch.device("cuda", 0))
    hx.run_lsrk(d_q, dt, 2)
    torch.cuda.synchronize()
    out.put((rank, ids[:no].copy(), d_q.cpu().numpy()[:no], hx.bytes_per_exchange()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("model,N", [(W.ACOUSTIC, 3), (W.ELASTIC, 2), (W.ACOUSTIC, 1)])
def test_two_processes_halo_exchange_match_single_domain(model, N):
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_1602_07997_b200 import dg
    import torch.multiprocessing as mp
    w = _case(model, N)
    ctx = dg.from_workload(w, device=0)
    q32 = w.initial_fields(None).astype(np.float32)
    dt = float(np.float32(ctx.stable_dt(0.5)))
    d = torch.from_numpy(q32).cuda()
    ctx.run(d.data_ptr(), dt, 2)
    torch.cuda.synchronize()
    want = d.cpu().numpy()
    ctx.close()
    mpc = mp.get_context("spawn")
    out = mpc.Queue()
    port = 29700 + (os.getpid() + 13 * N + model) % 2000
    procs = [mpc.Process(target=_rank_main, args=(r, 2, port, model, N, dt, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = [out.get(timeout=600) for _ in procs]
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    seen = np.zeros(len(want), dtype=bool)
    for rank, ids, q, nbytes in got:
        assert nbytes > 0 and np.isfinite(q).all()
        assert np.array_equal(q, want[ids]), f"rank {rank} differs from the single-domain run"
        seen[ids] = True
    assert seen.all()
