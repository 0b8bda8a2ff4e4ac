"""Multi-GPU groundwork on the CPU: the slab partition of the
element list, the ghost elements and the per-peer halo face lists that libdg builds (dg_partition_*), and the exchange
itself over torch.distributed with two gloo ranks -- each rank evaluates the oracle's r_k on its own elements from its
local mesh and the traces it received, and reproduces the single-domain oracle result."""
import os
import sys

import numpy as np
import pytest

from oracle import mesh as omesh
from oracle import physics, refelem
from paper_1602_07997_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def dg():
    from paper_1602_07997_b200 import build
    build.build()
    from paper_1602_07997_b200 import dg as mod
    return mod


def _mesh(n=3):
    vxyz, etov, _ = W.kuhn_cube(n, 0.06, seed=1)
    rng = np.random.default_rng(2)
    et = etov.copy()
    for k in range(len(et)):                      # any vertex order / orientation: the lists are in the library's face numbering
        et[k] = et[k][rng.permutation(4)]
    return vxyz, et


@pytest.mark.parametrize("nranks", [2, 3, 5])
def test_partition_slabs_ghosts_and_matching_halo_lists(dg, nranks):
    vxyz, etov = _mesh()
    K = len(etov)
    glob = dg.Context(vxyz, etov, 2, dg.ACOUSTIC, np.ones(K), np.ones(K), None, None, device=-1)
    gcon = glob.connectivity()
    parts = [dg.Partition(vxyz, etov, None, nranks, r) for r in range(nranks)]
    owned = np.concatenate([p.global_ids[:p.num_owned] for p in parts])
    assert np.array_equal(owned, np.arange(K))                                     # contiguous slabs tile the element list
    assert max(p.num_owned for p in parts) - min(p.num_owned for p in parts) <= 1
    Nfp = glob.Nfp
    for p in parts:
        gh = p.global_ids[p.num_owned:]
        assert np.all(np.diff(gh) > 0) and not np.intersect1d(gh, p.global_ids[:p.num_owned]).size
        # the local mesh is a valid mesh for dg_create; owned elements see the same neighbours as in the global mesh
        loc = dg.Context(vxyz, p.etov, 2, dg.ACOUSTIC, np.ones(len(p.etov)), np.ones(len(p.etov)), None, p.bc, device=-1,
                         owned_elements=p.num_owned)
        assert loc.K_owned == p.num_owned and loc.K == p.num_owned + p.num_ghost
        lcon = loc.connectivity()
        no = p.num_owned
        assert np.array_equal(p.global_ids[lcon["elemP"][:no]], gcon["elemP"][p.global_ids[:no]])
        assert np.array_equal(lcon["nodeP"][:no], gcon["nodeP"][p.global_ids[:no]])
        assert np.array_equal(lcon["bctag"][:no], gcon["bctag"][p.global_ids[:no]])
        assert np.abs(loc.node_coords()[:no] - glob.node_coords()[p.global_ids[:no]]).max() == 0.0
        # every ghost is the neighbour of an owned element, and only their faces towards owned elements are received
        assert set(gh) == set(np.unique(p.global_ids[lcon["elemP"][:no]])) - set(p.global_ids[:no])
        for rank, send, recv in p.peers:
            assert rank != p.rank and np.all(send >> 2 < no) and np.all(recv >> 2 >= no)
            q = parts[rank]
            back = [x for x in q.peers if x[0] == p.rank]
            assert len(back) == 1
            # what I send is, entry by entry, what the peer expects: same global element, same face
            assert np.array_equal(p.global_ids[send >> 2], q.global_ids[back[0][2] >> 2]) and np.array_equal(send & 3, back[0][2] & 3)
            # and each received face is the far side of one of my owned elements' faces
            nbr_of_owned = set(zip(p.global_ids[lcon["elemP"][:no, ::Nfp]].ravel().tolist(),
                                   np.repeat(p.global_ids[:no], 4).tolist()))
            assert all((int(p.global_ids[f >> 2]), g) in nbr_of_owned for f, g in
                       zip(recv, p.global_ids[lcon["elemP"][recv >> 2, (recv & 3) * Nfp]]))
        loc.close()
    with pytest.raises(dg.DGError):
        dg.Partition(vxyz, etov, None, 2, 2)
    with pytest.raises(dg.DGError):
        dg.Partition(vxyz, etov[:1], None, 2, 0)


def _rank_main(rank, world, port, model, N, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from paper_1602_07997_b200 import dg, halo
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    vxyz, etov = _mesh()
    K = len(etov)
    bc = None
    ref = refelem.build(N)
    if model == W.ACOUSTIC:
        mats = W.random_acoustic_materials(K, seed=2)
        rhs = physics.rhs_acoustic
    else:
        mats = W.random_elastic_materials(K, seed=2)
        rhs = physics.rhs_elastic
    nf = W.NFIELDS[model]
    qg = W.random_fields(K, model, ref.Np, seed=3)                         # the same global state on every rank
    part = dg.Partition(vxyz, etov, bc, world, rank)
    ids, no = part.global_ids, part.num_owned
    host = dg.Context(vxyz, part.etov, N, model, mats[0][ids], mats[1][ids], mats[2][ids] if model == W.ELASTIC else None, part.bc,
                      device=-1, owned_elements=no)
    fmask = host.reference_operators()["fmask"]
    q = qg[ids].copy()
    q[no:] = np.nan                                                         # ghosts hold nothing until the exchange
    ops, recv_bufs = [], []
    for peer, send, recv in part.peers:
        sb = torch.from_numpy(np.ascontiguousarray(halo.pack_host(q, send, fmask)))
        rb = torch.empty((len(recv), nf, ref.Nfp), dtype=torch.float64)
        recv_bufs.append((recv, rb))
        ops += [dist.P2POp(dist.isend, sb, peer), dist.P2POp(dist.irecv, rb, peer)]
    for wk in dist.batch_isend_irecv(ops):
        wk.wait()
    for recv, rb in recv_bufs:
        halo.unpack_host(q, recv, fmask, rb.numpy())
    m = omesh.build(ref, vxyz, part.etov, part.bc)
    local_mats = tuple(a[ids] for a in mats)
    r_loc = rhs(ref, m, *local_mats, q, np.arange(no))                      # r_k on the owned elements only
    out.put((rank, ids[:no].copy(), r_loc, sum(len(s) for _, s, _ in part.peers)))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("model,N", [(W.ACOUSTIC, 3), (W.ELASTIC, 2)])
def test_halo_exchange_two_gloo_ranks_reproduces_single_domain_rhs(dg, model, N):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29600 + (os.getpid() + 7 * N) % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, model, N, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = [out.get(timeout=300) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    vxyz, etov = _mesh()
    K = len(etov)
    ref = refelem.build(N)
    m = omesh.build(ref, vxyz, etov, None)
    qg = W.random_fields(K, model, ref.Np, seed=3)
    if model == W.ACOUSTIC:
        want = physics.rhs_acoustic(ref, m, *W.random_acoustic_materials(K, seed=2), qg)
    else:
        want = physics.rhs_elastic(ref, m, *W.random_elastic_materials(K, seed=2), qg)
    seen = np.zeros(K, dtype=bool)
    for rank, ids, r_loc, nsent in got:
        assert nsent > 0 and np.isfinite(r_loc).all()                       # no NaN left: every gathered ghost trace arrived
        assert np.abs(r_loc - want[ids]).max() <= 1e-11 * np.abs(want).max()
        seen[ids] = True
    assert seen.all()
