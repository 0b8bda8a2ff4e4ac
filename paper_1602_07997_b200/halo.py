"""Halo exchange plumbing for the multi-GPU form of the hot path: one process per GPU, `torch.distributed` moves the
packed face traces between peers (NCCL over NVLink on GPUs; gloo in the CPU tests), libdg packs and unpacks them
(dg_halo_pack / dg_halo_unpack) and advances the owned elements.  No method arithmetic here.

    part = dg.Partition(vxyz, etov, bc, world, rank)
    ctx = dg.Context(vxyz, part.etov, N, model, rho[ids], c[ids], vs, part.bc, owned_elements=part.num_owned)
    hx = HaloExchanger(part, ctx, torch.device("cuda", local_rank))
    for A, B in stages:  hx.exchange(q_cur); ctx.stage(q_cur.data_ptr(), q_next.data_ptr(), A, B, dt); swap

The path scales weakly: per stage and rank the exchange moves Nfields * Nfp floats per cut face and direction
("halo exchanges"), against Nfields * Np floats of state per element.
"""
from __future__ import annotations

from fractions import Fraction

import numpy as np

# the 2N-storage coefficients dg_run uses (Carpenter & Kennedy; reading Q2), for drivers that go stage by stage
LSRK_A = tuple(float(Fraction(*f)) for f in ((0, 1), (-567301805773, 1357537059087), (-2404267990393, 2016746695238),
                                             (-3550918686646, 2091501179385), (-1275806237668, 842570457699)))
LSRK_B = tuple(float(Fraction(*f)) for f in ((1432997174477, 9575080441755), (5161836677717, 13612068292357),
                                             (1720146321549, 2090206949498), (3134564353537, 4481467310338),
                                             (2277821191437, 14882151754819)))


class HaloExchanger:
    """Per-peer device face lists and buffers; `exchange` fills the ghost elements' face nodes of `q` from the peers."""

    def __init__(self, part, ctx, device, group=None):
        import torch
        self.torch, self.part, self.ctx, self.group = torch, part, ctx, group
        nf, nfp = ctx.NF, ctx.Nfp
        self.peers = []
        for rank, send, recv in part.peers:
            self.peers.append(dict(rank=rank,
                                   send=torch.from_numpy(send).to(device), recv=torch.from_numpy(recv).to(device),
                                   sbuf=torch.empty(len(send) * nf * nfp, dtype=torch.float32, device=device),
                                   rbuf=torch.empty(len(recv) * nf * nfp, dtype=torch.float32, device=device)))

    def bytes_per_exchange(self) -> int:
        return sum(4 * (p["sbuf"].numel() + p["rbuf"].numel()) for p in self.peers)

    def exchange(self, q, stream=None):
        """q: device tensor [K_local][Nf][Np] (owned elements then ghosts).  Packs on `stream`, exchanges, unpacks.
        With the NCCL backend the device buffers go out as they are (peer copies over NVLink); with gloo (tests: several
        processes on one GPU or none) they are staged through host memory."""
        import torch.distributed as dist
        torch = self.torch
        sptr = stream.cuda_stream if stream is not None else None
        for p in self.peers:
            self.ctx.halo_pack(q.data_ptr(), p["send"].data_ptr(), p["send"].numel(), p["sbuf"].data_ptr(), sptr)
        staged = dist.get_backend(self.group) != "nccl"
        if stream is not None:
            stream.synchronize()                   # the packed buffers are complete before they leave
        else:
            torch.cuda.current_stream().synchronize()
        ops, back = [], []
        for p in self.peers:
            sb = p["sbuf"].cpu() if staged else p["sbuf"]
            rb = torch.empty(p["rbuf"].shape, dtype=p["rbuf"].dtype) if staged else p["rbuf"]
            back.append((p, rb))
            ops.append(dist.P2POp(dist.isend, sb, p["rank"], group=self.group))
            ops.append(dist.P2POp(dist.irecv, rb, p["rank"], group=self.group))
        if ops:
            for w in dist.batch_isend_irecv(ops):
                w.wait()
        for p, rb in back:
            if staged:
                p["rbuf"].copy_(rb)
            self.ctx.halo_unpack(q.data_ptr(), p["recv"].data_ptr(), p["recv"].numel(), p["rbuf"].data_ptr(), sptr)

    def run_lsrk(self, q, dt: float, nsteps: int, stream=None):
        """nsteps LSRK(5,4) steps of the partitioned mesh: per stage exchange the cut faces' traces, then dg_stage on the owned
        elements (ping-pong between `q` and a scratch tensor; the result ends in `q`).  Coefficients: the library's
        (dg_run's) Carpenter-Kennedy pairs, passed stage by stage."""
        torch = self.torch
        sptr = stream.cuda_stream if stream is not None else None
        cur, nxt = q, torch.empty_like(q)
        for _ in range(nsteps):
            for a, b in zip(LSRK_A, LSRK_B):
                self.exchange(cur, stream)
                self.ctx.stage(cur.data_ptr(), nxt.data_ptr(), a, b, dt, sptr)
                cur, nxt = nxt, cur
        if cur is not q:
            q.copy_(cur)
        return q


def pack_host(q: np.ndarray, faces: np.ndarray, fmask: np.ndarray) -> np.ndarray:
    """What dg_halo_pack moves, on host arrays (CPU tests of the lists): [nfaces][Nf][Nfp] from q [K][Nf][Np]."""
    elem, face = faces >> 2, faces & 3
    return q[elem[:, None, None], np.arange(q.shape[1])[None, :, None], fmask[face][:, None, :]]


def unpack_host(q: np.ndarray, faces: np.ndarray, fmask: np.ndarray, buf: np.ndarray) -> None:
    elem, face = faces >> 2, faces & 3
    q[elem[:, None, None], np.arange(q.shape[1])[None, :, None], fmask[face][:, None, :]] = buf
