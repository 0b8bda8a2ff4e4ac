"""Pins for oracle.mesh / oracle.physics (T6-T9 of DESIGN.md "Oracle pins").  CPU only.

What fixes the oracle here: exact PDE right-hand sides for polynomial fields
(volume terms and vanishing interior penalties), an independent numerical
solve of the interface Riemann problem, the discrete divergence theorem, and
the semi-discrete energy identity (non-increasing energy under the upwind
flux, BASELINE.json north_star) including its brute-force matrix form.
"""
import numpy as np
import pytest

from oracle import mesh as omesh
from oracle import physics, refelem, timestep
from paper_1602_07997_b200 import workloads as W

RNG = np.random.default_rng(12345)


def make(N, n, jitter=0.05, top=W.BC_RIGID, other=W.BC_RIGID, refelems=None):
    ref = refelems(N) if refelems else refelem.build(N)
    vxyz, etov, cell = W.kuhn_cube(n, jitter, seed=1)
    bc = W.wall_tags(n, etov, top=top, other=other)
    return ref, omesh.build(ref, vxyz, etov, bc), cell


# ---------------------------------------------------------------- geometry
def test_mesh_volume_surface_and_normals(refelems):
    ref, m, _ = make(2, 3, jitter=0.08, refelems=refelems)
    assert abs(np.sum(m.J) * 4.0 / 3.0 - 1.0) < 1e-12                   # tets fill the unit cube
    # closed surface of every element: sum_f area_f n_f = 0; reference face areas 2,2,2,2 (parametric)
    area = m.Fscale * m.J[:, None] * 2.0
    assert np.abs(np.einsum("kf,kfi->ki", area, m.nrm)).max() < 1e-13
    # boundary faces of the cube: total area 6, normals are the axis directions
    bnd = m.bctag > 0
    assert abs(area[bnd].sum() - 6.0) < 1e-12
    assert np.allclose(np.abs(m.nrm[bnd]).max(axis=1), 1.0, atol=1e-12)
    # neighbour normals are opposite and traces coincide in space
    Nfp = ref.Nfp
    xm = m.x[:, ref.Fmask.reshape(-1)]
    xp = m.x[m.elemP, m.nodeP]
    assert np.abs(xm - xp).max() < 1e-12
    k2 = m.elemP[:, ::Nfp]
    for f in range(4):
        interior = m.bctag[:, f] == 0
        nb = k2[interior, f]
        # the neighbour's matching face: find it through the shared nodes
        nbr_face = np.array([[np.all(np.isin(m.nodeP[k, f * Nfp:(f + 1) * Nfp], ref.Fmask[g])) for g in range(4)]
                             for k in np.flatnonzero(interior)])
        assert np.all(nbr_face.sum(axis=1) == 1)
        g = np.argmax(nbr_face, axis=1)
        assert np.allclose(m.nrm[interior, f], -m.nrm[nb, g], atol=1e-12)
        assert np.allclose(area[interior, f], area[nb, g], rtol=1e-12)


def test_negative_orientation_is_fixed(refelems):
    ref = refelems(1)
    vxyz, etov, _ = W.kuhn_cube(2, 0.0)
    flipped = etov.copy()
    flipped[::2, [2, 3]] = flipped[::2, [3, 2]]
    a = omesh.build(ref, vxyz, etov)
    b = omesh.build(ref, vxyz, flipped)
    assert np.array_equal(a.etov, b.etov) and np.all(b.J > 0)
    assert np.array_equal(omesh.orient(vxyz, flipped)[1], np.arange(len(etov)) % 2 == 0)


def test_nonconforming_and_untagged_meshes_raise(refelems):
    ref = refelems(1)
    vxyz, etov, _ = W.kuhn_cube(1, 0.0)
    with pytest.raises(ValueError):
        omesh.build(ref, vxyz, np.concatenate([etov, etov[:1]]))       # a face with three owners
    with pytest.raises(ValueError):
        omesh.build(ref, vxyz, etov, bc=np.zeros((6, 4), dtype=np.int8))


@pytest.mark.parametrize("N", [1, 2, 4, 7])
def test_discrete_divergence_theorem(refelems, N):
    """sum_nodes J M (d_x u) = sum_faces sJ n_x (face mass . u) for polynomials of degree <= N."""
    ref, m, _ = make(N, 1, jitter=0.0, refelems=refelems)
    k = 3
    x = m.x[k]
    u = (1 + x[:, 0]) ** N + x[:, 1] * x[:, 2] ** (N - 1) if N > 1 else 1 + x @ np.array([0.3, -0.2, 0.9])
    du = [ref.Dr @ u, ref.Ds @ u, ref.Dt @ u]
    one = np.ones(ref.Np)
    for i in range(3):
        dxu = sum(m.G[k, i, j] * du[j] for j in range(3))
        lhs = m.J[k] * one @ ref.M @ dxu
        rhs = sum(m.J[k] * m.Fscale[k, f] * m.nrm[k, f, i]
                  * one @ ref.Emat[:, f * ref.Nfp:(f + 1) * ref.Nfp] @ u[ref.Fmask[f]] for f in range(4))
        assert abs(lhs - rhs) < 1e-11 * max(1.0, abs(lhs))


# ---------------------------------------------------------------- T6/T7 polynomial fields
def _interior_elements(m):
    return np.flatnonzero(np.all(m.bctag == 0, axis=1))


@pytest.mark.parametrize("N", [1, 2, 3, 5])
def test_acoustic_polynomial_fields_T7(refelems, N):
    """Globally continuous polynomials of degree <= N in a homogeneous medium: interior penalties
    vanish and r equals the PDE right-hand side on elements without boundary faces."""
    ref, m, _ = make(N, 3, jitter=0.07, refelems=refelems)
    rho, c = np.full(m.K, 1.7), np.full(m.K, 2.3)
    x, y, z = m.x[..., 0], m.x[..., 1], m.x[..., 2]
    A = RNG.standard_normal((3, 3))
    a = RNG.standard_normal(3)
    q = np.zeros((m.K, 4, ref.Np))
    q[:, 0] = 0.4 + a[0] * x + a[1] * y + a[2] * z + (x * y if N >= 2 else 0) + (z ** N if N >= 2 else 0)
    gradp = np.stack([a[0] + (y if N >= 2 else 0) + 0 * x, a[1] + (x if N >= 2 else 0) + 0 * x,
                      a[2] + (N * z ** (N - 1) if N >= 2 else 0) + 0 * x], axis=1)
    for i in range(3):
        q[:, 1 + i] = A[i, 0] * x + A[i, 1] * y + A[i, 2] * z + (x ** N if (N >= 2 and i == 0) else 0)
    divv = np.trace(A) + (N * x ** (N - 1) if N >= 2 else 0) + 0 * x
    r = physics.rhs_acoustic(ref, m, rho, c, q)
    ie = _interior_elements(m)
    assert len(ie) > 0
    assert np.abs(r[ie, 0] - (-(1.7 * 2.3 ** 2) * divv[ie])).max() < 1e-10
    assert np.abs(r[ie, 1:4] - (-(1 / 1.7) * gradp[ie])).max() < 1e-10


@pytest.mark.parametrize("N", [1, 2, 4])
def test_elastic_polynomial_fields_T6(refelems, N):
    """v = A x (+ quadratic), sigma linear: r^sigma = lambda tr(grad v) I + mu (grad v + grad v^T),
    r^v = div(sigma)/rho on interior elements; pins the garbled mu-term (Q6)."""
    ref, m, _ = make(N, 3, jitter=0.07, refelems=refelems)
    rho, vp, vs = np.full(m.K, 2.1), np.full(m.K, 3.0), np.full(m.K, 1.6)
    mu, lam = 2.1 * 1.6 ** 2, 2.1 * 3.0 ** 2 - 2 * 2.1 * 1.6 ** 2
    X = m.x
    A = RNG.standard_normal((3, 3))
    B = RNG.standard_normal((3, 3, 3))
    B = 0.5 * (B + np.transpose(B, (1, 0, 2)))                    # sigma_ij = B_ijk x_k, symmetric in ij
    q = np.zeros((m.K, 9, ref.Np))
    gradv = np.broadcast_to(A[None, :, :, None], (m.K, 3, 3, ref.Np)).copy()       # d_j v_i
    for i in range(3):
        q[:, i] = np.einsum("j,knj->kn", A[i], X)
    if N >= 2:
        q[:, 0] += X[..., 1] * X[..., 2]
        gradv[:, 0, 1] += X[..., 2]
        gradv[:, 0, 2] += X[..., 1]
    for a_, (i, j) in enumerate(((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2))):
        q[:, 3 + a_] = np.einsum("c,knc->kn", B[i, j], X)
    divsig = np.einsum("ijj->i", B)
    r = physics.rhs_elastic(ref, m, rho, vp, vs, q)
    ie = _interior_elements(m)
    div = gradv[:, 0, 0] + gradv[:, 1, 1] + gradv[:, 2, 2]
    for i in range(3):
        assert np.abs(r[ie, i] - divsig[i] / 2.1).max() < 1e-10
    for a_, (i, j) in enumerate(((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2))):
        want = mu * (gradv[:, i, j] + gradv[:, j, i]) + (lam * div if i == j else 0)
        assert np.abs(r[ie, 3 + a_] - want[ie]).max() < 1e-10


# ---------------------------------------------------------------- T8 interface Riemann solves
def _riemann(tm, um, tp, up, Zm, Zp):
    """Star state of tau_t = rho c^2 u_x, rho u_t = tau_x at an interface, '-' on the left:
    tau* - Z^- u* = tau^- - Z^- u^-  (carried by the wave running into '-' ... unchanged invariant)
    tau* + Z^+ u* = tau^+ + Z^+ u^+ ; solved numerically."""
    out = np.empty(tm.shape + (2,))
    for idx in np.ndindex(tm.shape):
        Amat = np.array([[1.0, -Zm[idx]], [1.0, Zp[idx]]])
        out[idx] = np.linalg.solve(Amat, [tm[idx] - Zm[idx] * um[idx], tp[idx] + Zp[idx] * up[idx]])
    return out[..., 0], out[..., 1]


def _unit(v):
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def test_acoustic_penalties_vs_riemann_solve_T8():
    S = 400
    n = _unit(RNG.standard_normal((S, 3)))
    pm, pp = RNG.standard_normal(S), RNG.standard_normal(S)
    vm, vp = RNG.standard_normal((S, 3)), RNG.standard_normal((S, 3))
    rm, rp = RNG.uniform(1, 2.5, S), RNG.uniform(1, 2.5, S)
    cm, cp = RNG.uniform(1, 3, S), RNG.uniform(1, 3, S)
    p_p, p_v = physics.acoustic_penalties(pm, vm, pp, vp, n, rm, cm, rp, cp)
    # tau = -p
    ts, us = _riemann(-pm, np.sum(vm * n, -1), -pp, np.sum(vp * n, -1), rm * cm, rp * cp)
    ps = -ts
    # strong form: dp/dt + kappa div v = kappa (v_n^- - v_n^*),  dv/dt + grad p / rho = n (p^- - p^*)/rho
    assert np.allclose(-p_p, rm * cm ** 2 * (np.sum(vm * n, -1) - us), atol=1e-12)
    assert np.allclose(-p_v, (pm - ps) / rm, atol=1e-12)
    # a pure wave leaving into '+' produces no penalty on '-': p+ - p- = Z+ (vn+ - vn-)
    dv = RNG.standard_normal(S)
    vp2 = vm + dv[:, None] * n
    pp2 = pm + rp * cp * dv
    p_p2, p_v2 = physics.acoustic_penalties(pm, vm, pp2, vp2, n, rm, cm, rp, cp)
    assert np.abs(p_p2).max() < 1e-12 and np.abs(p_v2).max() < 1e-12


def test_elastic_penalties_vs_riemann_solve_T8():
    S = 400
    n = _unit(RNG.standard_normal((S, 3)))
    t1 = _unit(np.cross(n, RNG.standard_normal((S, 3))))
    t2 = np.cross(n, t1)
    vm, vp = RNG.standard_normal((S, 3)), RNG.standard_normal((S, 3))
    sm = RNG.standard_normal((S, 3, 3)); sm = sm + np.transpose(sm, (0, 2, 1))
    sp_ = RNG.standard_normal((S, 3, 3)); sp_ = sp_ + np.transpose(sp_, (0, 2, 1))
    Tm, Tp = np.einsum("sij,sj->si", sm, n), np.einsum("sij,sj->si", sp_, n)
    rm, rp = RNG.uniform(1.5, 3, S), RNG.uniform(1.5, 3, S)
    cpm, cpp = RNG.uniform(2, 6, S), RNG.uniform(2, 6, S)
    csm, csp = cpm / RNG.uniform(1.6, 2, S), cpp / RNG.uniform(1.6, 2, S)
    P, pv = physics.elastic_penalties(vm, Tm, vp, Tp, n, rm, cpm, csm, rp, cpp, csp)
    vstar, Tstar = np.zeros((S, 3)), np.zeros((S, 3))
    for d, Zm, Zp in ((n, rm * cpm, rp * cpp), (t1, rm * csm, rp * csp), (t2, rm * csm, rp * csp)):
        ts, us = _riemann(np.sum(Tm * d, -1), np.sum(vm * d, -1), np.sum(Tp * d, -1), np.sum(vp * d, -1), Zm, Zp)
        vstar += us[:, None] * d
        Tstar += ts[:, None] * d
    dv = vstar - vm
    mu = rm * csm ** 2
    lam = rm * cpm ** 2 - 2 * mu
    # rho dv/dt = div sigma  ->  surface term (T* - T^-)/rho ;  dsigma/dt = C : grad v -> C : (n (x) dv)
    assert np.allclose(pv, (Tstar - Tm) / rm[:, None], atol=1e-11)
    want = (lam * np.sum(dv * n, -1))[:, None, None] * np.eye(3) \
        + mu[:, None, None] * (n[:, :, None] * dv[:, None, :] + dv[:, :, None] * n[:, None, :])
    assert np.allclose(P, want, atol=1e-11)
    assert np.allclose(P, np.transpose(P, (0, 2, 1)))


# ---------------------------------------------------------------- T9 energy
def _acoustic_setup(N, n, refelems, top=W.BC_RIGID, other=W.BC_RIGID):
    ref, m, _ = make(N, n, jitter=0.08, top=top, other=other, refelems=refelems)
    rho, c = W.random_acoustic_materials(m.K, seed=7)
    return ref, m, rho, c


def _elastic_setup(N, n, refelems, top=W.BC_FREE, other=W.BC_RIGID):
    ref, m, _ = make(N, n, jitter=0.08, top=top, other=other, refelems=refelems)
    rho, vp, vs = W.random_elastic_materials(m.K, seed=7, rho_rng=(1.5, 3.0), vp_rng=(2.0, 6.0))
    return ref, m, rho, vp, vs


@pytest.mark.parametrize("N,bcs", [(1, (W.BC_RIGID, W.BC_RIGID)), (3, (W.BC_FREE, W.BC_RIGID)), (4, (W.BC_RIGID, W.BC_FREE))])
def test_acoustic_energy_rate_T9(refelems, N, bcs):
    ref, m, rho, c = _acoustic_setup(N, 2, refelems, *bcs)
    for trial in range(3):
        q = RNG.standard_normal((m.K, 4, ref.Np))
        r = physics.rhs_acoustic(ref, m, rho, c, q)
        g = timestep.energy_gradient_acoustic(ref, m, rho, c, q)
        rate, scale = np.sum(g * r), np.sum(np.abs(g * r))
        assert rate <= 1e-12 * scale
        assert rate < -1e-3 * scale          # random (discontinuous) data does dissipate
    # energy functional and its gradient agree: E = 1/2 <q, Wq>
    assert abs(timestep.energy_acoustic(ref, m, rho, c, q) - 0.5 * np.sum(q * g)) < 1e-10 * scale


@pytest.mark.parametrize("N,bcs", [(1, (W.BC_FREE, W.BC_RIGID)), (2, (W.BC_SLIP, W.BC_FREE)), (4, (W.BC_RIGID, W.BC_SLIP))])
def test_elastic_energy_rate_T9(refelems, N, bcs):
    ref, m, rho, vp, vs = _elastic_setup(N, 2, refelems, *bcs)
    for trial in range(3):
        q = RNG.standard_normal((m.K, 9, ref.Np))
        r = physics.rhs_elastic(ref, m, rho, vp, vs, q)
        g = timestep.energy_gradient_elastic(ref, m, rho, vp, vs, q)
        rate, scale = np.sum(g * r), np.sum(np.abs(g * r))
        assert rate <= 1e-12 * scale
        assert rate < -1e-3 * scale
    assert timestep.energy_elastic(ref, m, rho, vp, vs, q) > 0


def test_continuous_fields_conserve_energy(refelems):
    """With continuous data and closed (rigid) walls obeyed by the data, the penalty terms vanish
    and the semi-discrete energy rate is zero to rounding: the decay above is all from jumps."""
    ref, m, _ = make(3, 2, jitter=0.05, refelems=refelems)
    rho, c = np.ones(m.K), np.ones(m.K)
    q = W.standing_mode(m.x, t=0.37)       # degree-3 interpolant of a smooth field: continuous across faces
    r = physics.rhs_acoustic(ref, m, rho, c, q)
    g = timestep.energy_gradient_acoustic(ref, m, rho, c, q)
    assert abs(np.sum(g * r)) < 2e-3 * np.sum(np.abs(g * r))


def _global_matrix(rhs, shape):
    n = int(np.prod(shape))
    A = np.empty((n, n))
    for j in range(n):
        e = np.zeros(n); e[j] = 1.0
        A[:, j] = rhs(e.reshape(shape)).ravel()
    return A


@pytest.mark.parametrize("model,N", [("acoustic", 1), ("acoustic", 2), ("elastic", 1), ("elastic", 2)])
def test_brute_force_operator_is_dissipative(refelems, model, N):
    """Matrix form of T9 on the single-cell mesh (K=6): W A + A^T W is negative semi-definite,
    and r(q) is linear in q."""
    if model == "acoustic":
        ref, m, rho, c = _acoustic_setup(N, 1, refelems, W.BC_FREE, W.BC_RIGID)
        rhs = lambda q: physics.rhs_acoustic(ref, m, rho, c, q)                     # noqa: E731
        grad = lambda q: timestep.energy_gradient_acoustic(ref, m, rho, c, q)       # noqa: E731
        shape = (m.K, 4, ref.Np)
    else:
        ref, m, rho, vp, vs = _elastic_setup(N, 1, refelems, W.BC_FREE, W.BC_SLIP)
        rhs = lambda q: physics.rhs_elastic(ref, m, rho, vp, vs, q)                 # noqa: E731
        grad = lambda q: timestep.energy_gradient_elastic(ref, m, rho, vp, vs, q)   # noqa: E731
        shape = (m.K, 9, ref.Np)
    A = _global_matrix(rhs, shape)
    Wm = _global_matrix(grad, shape)
    assert np.allclose(Wm, Wm.T, atol=1e-12)
    assert np.linalg.eigvalsh(Wm).min() > 0
    S = Wm @ A + A.T @ Wm
    ev = np.linalg.eigvalsh(0.5 * (S + S.T))
    assert ev.max() <= 1e-11 * np.abs(ev).max()
    q = RNG.standard_normal(shape)
    assert np.allclose(rhs(q).ravel(), A @ q.ravel(), atol=1e-10)
    # element subsets give the same rows as the full evaluation
    sub = np.array([4, 1])
    full = rhs(q)
    part = (physics.rhs_acoustic(ref, m, rho, c, q, sub) if model == "acoustic"
            else physics.rhs_elastic(ref, m, rho, vp, vs, q, sub))
    assert np.array_equal(part, full[sub])
