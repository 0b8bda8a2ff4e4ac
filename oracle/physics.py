"""Semi-discrete right-hand sides r_k in fp64 (oracle; test infrastructure only).

Acoustic  : PAPER.md:36-51 (system, penalty terms p_p, p_v, alpha_c, k_c) and
            eq. (5)-(6) at PAPER.md:146-152.
Elastic   : PAPER.md:53-84 (system, P_sigma, p_v, alpha_p, alpha_s, k_p, k_s)
            and the two unnumbered equations at; the mu-term
            of the second one is garbled in the text and is read as
            mu (d_j v_i + d_i v_j)   (reading Q6).
Boundaries: the paper never states them; mirror states of
            DESIGN.md reading Q9.

Layout: q is K x Nfields x Np, node index fastest (Table 1).
Field order: acoustic (p, vx, vy, vz); elastic (vx, vy, vz, sxx, syy, szz,
sxy, sxz, syz).  "-" is the local element, "+" the neighbour, n the outward
normal of the local element (reading Q8).
"""
from __future__ import annotations

import numpy as np

from .mesh import BC_FREE, BC_RIGID, BC_SLIP, Mesh
from .refelem import RefElem

# field index of sigma_ij in the elastic state vector
SIG = np.array([[3, 6, 7], [6, 4, 8], [7, 8, 5]])


def _face_geometry(ref: RefElem, mesh: Mesh, elems):
    """normal (E x 4Nfp x 3), g^sur (E x 4Nfp), boundary tag (E x 4Nfp)."""
    Nfp = ref.Nfp
    n = np.repeat(mesh.nrm[elems], Nfp, axis=1)
    gsur = np.repeat(mesh.Fscale[elems], Nfp, axis=1)
    tag = np.repeat(mesh.bctag[elems], Nfp, axis=1)
    return n, gsur, tag


def _ref_derivatives(ref: RefElem, u):
    """(D_1 u, D_2 u, D_3 u) for u of shape (..., Np)."""
    return u @ ref.Dr.T, u @ ref.Ds.T, u @ ref.Dt.T


# --------------------------------------------------------------------------
def acoustic_penalties(pm, vm, pp, vp, n, rho_m, c_m, rho_p, c_p):
    """Penalty terms of PAPER.md:47-51 at face nodes.

    pm, pp: (...,) pressures; vm, vp, n: (..., 3).  Returns p_p (...,) and the
    scalar p_v (...,); the velocity equation receives p_v * n.
    """
    jump_p = (pp - pm) / 2
    jump_vn = np.sum((vp - vm) * n, axis=-1) / 2
    alpha_c = jump_p - (rho_p * c_p) * jump_vn
    k_c = 1.0 / ((rho_m * c_m + rho_p * c_p) / 2)
    p_p = -(rho_m * c_m ** 2) * k_c * alpha_c
    p_v = c_m * k_c * alpha_c
    return p_p, p_v


def rhs_acoustic(ref: RefElem, mesh: Mesh, rho, c, q, elems=None):
    """r_k of eq. (5)-(6) for the elements `elems` (all when None)."""
    q = np.asarray(q, dtype=np.float64)
    if elems is None:
        elems = np.arange(mesh.K)
    elems = np.asarray(elems)
    rho = np.asarray(rho, dtype=np.float64)
    c = np.asarray(c, dtype=np.float64)
    g = mesh.G[elems]                                    # E x 3(i) x 3(j)
    rk, ck = rho[elems][:, None], c[elems][:, None]
    p = q[elems, 0]                                      # E x Np
    v = q[elems, 1:4]                                    # E x 3 x Np
    # ---- volume terms
    # eq. (5): -rho c^2 sum_j D_j [ sum_i g_ij q^{v_i} ]
    w = np.einsum("eij,ein->ejn", g, v)                  # E x 3(j) x Np
    Dw = _ref_derivatives(ref, w)
    r_p = -(rk * ck ** 2) * (Dw[0][:, 0] + Dw[1][:, 1] + Dw[2][:, 2])
    # eq. (6): -(1/rho) sum_j g_ij [ D_j q^p ]
    Dp = np.stack(_ref_derivatives(ref, p), axis=1)      # E x 3(j) x Np
    r_v = -(1.0 / rk)[:, None] * np.einsum("eij,ejn->ein", g, Dp)
    # ---- surface terms
    fm = ref.Fmask.reshape(-1)
    eP, nP = mesh.elemP[elems], mesh.nodeP[elems]
    n, gsur, tag = _face_geometry(ref, mesh, elems)
    pm = p[:, fm]
    vm = np.transpose(v[:, :, fm], (0, 2, 1))            # E x 4Nfp x 3
    pp = q[eP, 0, nP]
    vp = np.stack([q[eP, 1, nP], q[eP, 2, nP], q[eP, 3, nP]], axis=-1)
    rho_p, c_p = rho[eP], c[eP]
    # mirror states on boundary faces (Q9)
    vn_m = np.sum(vm * n, axis=-1)
    wall = (tag == BC_RIGID) | (tag == BC_SLIP)
    free = tag == BC_FREE
    pp = np.where(wall, pm, np.where(free, -pm, pp))
    vp = np.where(wall[..., None], vm - 2 * vn_m[..., None] * n, np.where(free[..., None], vm, vp))
    p_p, p_v = acoustic_penalties(pm, vm, pp, vp, n, rk, ck, rho_p, c_p)
    # eq. (5)-(6): - L (g^sur p)
    r_p = r_p - (gsur * p_p) @ ref.LIFT.T
    r_v = r_v - np.einsum("efi,nf->ein", (gsur * p_v)[..., None] * n, ref.LIFT)
    return np.concatenate([r_p[:, None, :], r_v], axis=1)


# --------------------------------------------------------------------------
def elastic_penalties(vm, Tm, vp, Tp, n, rho_m, cp_m, cs_m, rho_p, cp_p, cs_p):
    """P_sigma (..., 3, 3) and p_v (..., 3) of PAPER.md:73-84.

    vm, vp: velocities (..., 3); Tm, Tp: tractions sigma^-/+ . n (..., 3) with
    the local normal n on both sides; lambda^-, mu^- from (rho, c_p, c_s)^-.
    """
    mu_m = rho_m * cs_m ** 2
    lam_m = rho_m * cp_m ** 2 - 2 * mu_m
    jump_sn = (Tp - Tm) / 2                                   # [[sigma n]]
    jump_snn = np.sum(jump_sn * n, axis=-1)                   # [[sigma_nn]]
    jump_v = (vp - vm) / 2                                    # [[v]]
    jump_vn = np.sum(jump_v * n, axis=-1)                     # [[v_n]]
    alpha_p = jump_snn + (rho_p * cp_p) * jump_vn
    alpha_s_vec = jump_sn + (rho_p * cs_p)[..., None] * jump_v
    alpha_s = np.sum(alpha_s_vec * n, axis=-1)                # = [[sigma_nn]] + (rho c_s)^+ [[v_n]]
    k_p = 1.0 / ((rho_m * cp_m + rho_p * cp_p) / 2)
    k_s = 1.0 / ((rho_m * cs_m + rho_p * cs_p) / 2)
    eye = np.eye(3)
    NN = n[..., :, None] * n[..., None, :]
    sym = 0.5 * (n[..., :, None] * alpha_s_vec[..., None, :] + alpha_s_vec[..., :, None] * n[..., None, :])
    P_sigma = ((k_p * alpha_p * lam_m)[..., None, None] * eye
               + (2 * (k_p * alpha_p - k_s * alpha_s) * mu_m)[..., None, None] * NN
               + (2 * k_s * mu_m)[..., None, None] * sym)
    p_v = ((k_p * alpha_p * cp_m - k_s * alpha_s * cs_m)[..., None] * n
           + (k_s * cs_m)[..., None] * alpha_s_vec)
    return P_sigma, p_v


def rhs_elastic(ref: RefElem, mesh: Mesh, rho, vp_, vs_, q, elems=None):
    """r_k of PAPER.md:156-158 for the elements `elems` (all when None)."""
    q = np.asarray(q, dtype=np.float64)
    if elems is None:
        elems = np.arange(mesh.K)
    elems = np.asarray(elems)
    rho, cp, cs = (np.asarray(a, dtype=np.float64) for a in (rho, vp_, vs_))
    g = mesh.G[elems]
    rk = rho[elems][:, None]
    mu = (rho * cs ** 2)[elems][:, None]
    lam = (rho * cp ** 2)[elems][:, None] - 2 * mu
    v = q[elems, 0:3]                                       # E x 3 x Np
    sig = q[elems][:, SIG]                                  # E x 3 x 3 x Np
    # ---- volume terms
    # r^{v_i} = 1/rho sum_n D_n [ sum_m g_mn sigma_im ]
    w = np.einsum("emn,eimp->einp", g, sig)                 # E x i x n x Np
    Dw = _ref_derivatives(ref, w)
    r_v = (1.0 / rk)[:, None] * (Dw[0][:, :, 0] + Dw[1][:, :, 1] + Dw[2][:, :, 2])
    # grad v:  dv[e,i,j] = d_j v_i = sum_m g_jm [D_m v_i]
    Dv = np.stack(_ref_derivatives(ref, v), axis=2)         # E x i x m x Np
    dv = np.einsum("ejm,eimp->eijp", g, Dv)
    div = dv[:, 0, 0] + dv[:, 1, 1] + dv[:, 2, 2]
    r_s = np.empty((len(elems), 3, 3, ref.Np))
    for i in range(3):
        for j in range(3):
            r_s[:, i, j] = mu * (dv[:, i, j] + dv[:, j, i]) + (lam * div if i == j else 0.0)
    # ---- surface terms
    fm = ref.Fmask.reshape(-1)
    eP, nP = mesh.elemP[elems], mesh.nodeP[elems]
    n, gsur, tag = _face_geometry(ref, mesh, elems)
    vm = np.transpose(v[:, :, fm], (0, 2, 1))               # E x F x 3
    sm = np.transpose(sig[:, :, :, fm], (0, 3, 1, 2))       # E x F x 3 x 3
    Tm = np.einsum("efij,efj->efi", sm, n)
    qP = q[eP[:, :, None], np.arange(9)[None, None, :], nP[:, :, None]]   # E x F x 9
    vp = qP[:, :, 0:3]
    Tp = np.einsum("efij,efj->efi", qP[:, :, SIG], n)
    rho_p, cp_p, cs_p = rho[eP], cp[eP], cs[eP]
    # mirror states (Q9)
    vn_m = np.sum(vm * n, axis=-1)[..., None]
    Tn_m = np.sum(Tm * n, axis=-1)[..., None]
    rigid, free, slip = (tag == BC_RIGID)[..., None], (tag == BC_FREE)[..., None], (tag == BC_SLIP)[..., None]
    vp = np.where(rigid, -vm, np.where(free, vm, np.where(slip, vm - 2 * vn_m * n, vp)))
    Tp = np.where(rigid, Tm, np.where(free, -Tm, np.where(slip, -Tm + 2 * Tn_m * n, Tp)))
    P_sigma, p_v = elastic_penalties(vm, Tm, vp, Tp, n, rk, cp[elems][:, None], cs[elems][:, None],
                                     rho_p, cp_p, cs_p)
    r_v = r_v + np.einsum("efi,nf->ein", gsur[..., None] * p_v, ref.LIFT)
    r_s = r_s + np.einsum("efij,nf->eijn", gsur[..., None, None] * P_sigma, ref.LIFT)
    out = np.empty((len(elems), 9, ref.Np))
    out[:, 0:3] = r_v
    for a, (i, j) in enumerate(((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2))):
        out[:, 3 + a] = r_s[:, i, j]
    return out
