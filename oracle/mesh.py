"""Geometry and face-node connectivity in fp64 (oracle; test infrastructure only).

PAPER.md:106 ("geometric factors g^vol_{k,i,j} and g^sur_{k,f} depend on the
shape of each element") and PAPER.md:171 (neighbour values through a mapping
array).  Readings: DESIGN.md Q4/Q5 (g^vol_{k,i,j} = d r_j / d x_i,
g^sur_{k,f} = sJ_f / J), Q12 (face numbering), Q13 (node matching by position).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .refelem import RefElem

# local vertex numbers of the four faces (f1: t=-1, f2: s=-1, f3: r+s+t=-1, f4: r=-1)
FACE_VERTS = np.array([[0, 1, 2], [0, 1, 3], [1, 2, 3], [0, 2, 3]])

BC_INTERIOR, BC_RIGID, BC_FREE, BC_SLIP = 0, 1, 2, 3


@dataclass
class Mesh:
    K: int
    etov: np.ndarray      # K x 4, positively oriented
    x: np.ndarray         # K x Np x 3 node coordinates
    J: np.ndarray         # K      Jacobian determinant of the affine map
    G: np.ndarray         # K x 3 x 3, G[k,i,j] = d r_j / d x_i   (g^vol of eq. (5)-(6))
    nrm: np.ndarray       # K x 4 x 3 outward unit normals
    Fscale: np.ndarray    # K x 4  sJ/J   (g^sur)
    elemP: np.ndarray     # K x 4Nfp  element holding the exterior (+) trace
    nodeP: np.ndarray     # K x 4Nfp  volume-node index of the exterior trace in elemP
    bctag: np.ndarray     # K x 4  0 = interior face, else boundary tag
    hmin: float


def orient(vxyz: np.ndarray, etov: np.ndarray) -> np.ndarray:
    """Swap the last two vertices of elements with negative Jacobian (faces 0 and 1 trade places);
    returns the new table and the mask of swapped elements."""
    etov = np.array(etov, dtype=np.int64, copy=True)
    v = vxyz[etov]
    det = np.linalg.det(np.stack([v[:, 1] - v[:, 0], v[:, 2] - v[:, 0], v[:, 3] - v[:, 0]], axis=2))
    neg = det < 0
    etov[neg, 2], etov[neg, 3] = etov[neg, 3].copy(), etov[neg, 2].copy()
    return etov, neg


def build(ref: RefElem, vxyz: np.ndarray, etov: np.ndarray, bc: np.ndarray | None = None,
          only_elems: np.ndarray | None = None) -> Mesh:
    """`only_elems`: restrict the face-node matching (the expensive part) to the faces of these
    elements; elemP/nodeP rows of all other elements are then left pointing at themselves."""
    vxyz = np.asarray(vxyz, dtype=np.float64)
    etov, swapped = orient(vxyz, etov)
    if bc is not None:
        bc = np.array(bc, dtype=np.int8, copy=True)
        bc[swapped, 0], bc[swapped, 1] = bc[swapped, 1].copy(), bc[swapped, 0].copy()
    K = etov.shape[0]
    Np, Nfp = ref.Np, ref.Nfp
    v = vxyz[etov]                                   # K x 4 x 3
    v1, v2, v3, v4 = v[:, 0], v[:, 1], v[:, 2], v[:, 3]
    # affine map x = 1/2[-(1+r+s+t) v1 + (1+r) v2 + (1+s) v3 + (1+t) v4]
    r, s, t = ref.r[None, :, None], ref.s[None, :, None], ref.t[None, :, None]
    x = 0.5 * (-(1 + r + s + t) * v1[:, None] + (1 + r) * v2[:, None] + (1 + s) * v3[:, None] + (1 + t) * v4[:, None])
    A = np.stack([(v2 - v1) / 2, (v3 - v1) / 2, (v4 - v1) / 2], axis=2)   # columns x_r, x_s, x_t
    J = np.linalg.det(A)
    if np.any(J <= 0):
        raise ValueError("degenerate element")
    Ainv = np.linalg.inv(A)                           # rows: grad r, grad s, grad t
    G = np.transpose(Ainv, (0, 2, 1)).copy()          # G[k,i,j] = d r_j / d x_i
    gr, gs, gt = Ainv[:, 0], Ainv[:, 1], Ainv[:, 2]
    ntil = np.stack([-gt, -gs, gr + gs + gt, -gr], axis=1)                # K x 4 x 3
    Fscale = np.linalg.norm(ntil, axis=2)
    nrm = ntil / Fscale[:, :, None]

    # ---- face pairing through sorted vertex triples
    fv = np.sort(etov[:, FACE_VERTS], axis=2).reshape(K * 4, 3)
    nv = int(vxyz.shape[0])
    key = (fv[:, 0] * nv + fv[:, 1]) * nv + fv[:, 2]
    order = np.argsort(key, kind="stable")
    ks = key[order]
    same_next = np.zeros(K * 4, dtype=bool)
    same_next[:-1] = ks[1:] == ks[:-1]
    if np.any(same_next[1:] & same_next[:-1]):
        raise ValueError("non-conforming mesh: a face has more than two owners")
    partner = np.full(K * 4, -1, dtype=np.int64)
    a = order[np.flatnonzero(same_next)]
    b = order[np.flatnonzero(same_next) + 1]
    partner[a], partner[b] = b, a

    elemP = np.repeat(np.arange(K)[:, None], 4 * Nfp, axis=1)
    nodeP = np.tile(ref.Fmask.reshape(-1)[None, :], (K, 1))
    bctag = np.zeros((K, 4), dtype=np.int8)
    bnd = partner < 0
    if bc is None:
        bctag.reshape(-1)[bnd] = BC_RIGID
    else:
        bctag.reshape(-1)[bnd] = np.asarray(bc, dtype=np.int8).reshape(-1)[bnd]
        if np.any(bctag.reshape(-1)[bnd] == 0):
            raise ValueError("boundary face without a boundary tag")

    # ---- node matching by physical position on every interior face
    hmin = float(np.min(2.0 / Fscale.max(axis=1)))
    ids = np.flatnonzero(~bnd)
    if only_elems is not None:
        keep = np.zeros(K, dtype=bool)
        keep[np.asarray(only_elems)] = True
        ids = ids[keep[ids // 4]]
    chunk = max(256, int(2e7 // (Nfp * Nfp)))
    for c0 in range(0, len(ids), chunk):
        me = ids[c0:c0 + chunk]
        ot = partner[me]
        k1, f1 = me // 4, me % 4
        k2, f2 = ot // 4, ot % 4
        xa = x[k1[:, None], ref.Fmask[f1]]                 # n x Nfp x 3
        xb = x[k2[:, None], ref.Fmask[f2]]
        d = np.linalg.norm(xa[:, :, None, :] - xb[:, None, :, :], axis=3)
        j = np.argmin(d, axis=2)
        dmin = np.take_along_axis(d, j[:, :, None], axis=2)[:, :, 0]
        if np.any(dmin > 1e-9 * hmin):
            raise ValueError("face nodes of neighbours do not coincide")
        if np.any(np.sort(j, axis=1) != np.arange(Nfp)[None, :]):
            raise ValueError("face-node matching is not one-to-one")
        cols = f1[:, None] * Nfp + np.arange(Nfp)[None, :]
        elemP[k1[:, None], cols] = k2[:, None]
        nodeP[k1[:, None], cols] = ref.Fmask[f2][np.arange(len(me))[:, None], j]
    return Mesh(K, etov, x, J, G, nrm, Fscale, elemP, nodeP, bctag, hmin)
