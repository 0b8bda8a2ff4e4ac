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

import numpy as np


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
        """q: device tensor [K_local][Nf][Np] (owned elements then ghosts).  Packs on `stream`, exchanges, unpacks."""
        import torch.distributed as dist
        torch = self.torch
        sptr = stream.cuda_stream if stream is not None else None
        for p in self.peers:
            self.ctx.halo_pack(q.data_ptr(), p["send"].data_ptr(), p["send"].numel(), p["sbuf"].data_ptr(), sptr)
        ops = []
        for p in self.peers:
            ops.append(dist.P2POp(dist.isend, p["sbuf"], p["rank"], group=self.group))
            ops.append(dist.P2POp(dist.irecv, p["rbuf"], p["rank"], group=self.group))
        if ops:
            for w in dist.batch_isend_irecv(ops):
                w.wait()
        for p in self.peers:
            self.ctx.halo_unpack(q.data_ptr(), p["recv"].data_ptr(), p["recv"].numel(), p["rbuf"].data_ptr(), sptr)


def pack_host(q: np.ndarray, faces: np.ndarray, fmask: np.ndarray) -> np.ndarray:
    """What dg_halo_pack moves, on host arrays (CPU tests of the lists): [nfaces][Nf][Nfp] from q [K][Nf][Np]."""
    elem, face = faces >> 2, faces & 3
    return q[elem[:, None, None], np.arange(q.shape[1])[None, :, None], fmask[face][:, None, :]]


def unpack_host(q: np.ndarray, faces: np.ndarray, fmask: np.ndarray, buf: np.ndarray) -> None:
    elem, face = faces >> 2, faces & 3
    q[elem[:, None, None], np.arange(q.shape[1])[None, :, None], fmask[face][:, None, :]] = buf
