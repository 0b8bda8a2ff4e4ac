"""Pins for oracle.refelem (T1-T5 of DESIGN.md "Oracle pins").  CPU only.

None of these re-type the oracle's formulas: they use closed forms, scipy's
independent Jacobi/Gauss routines, quadrature, and algebraic identities that a
dropped term, wrong sign, wrong index or wrong normalisation would break.
"""
import itertools
import math
import os

import numpy as np
import pytest
import scipy.special as sp

from oracle import refelem

GOLD = os.path.join(os.path.dirname(__file__), "golden")
DEGREES = list(range(1, 11))


# ---------------------------------------------------------------- golden sizes
def test_np_matches_paper_table4(refelems):
    rows = [l.split() for l in open(os.path.join(GOLD, "table4_np.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 8
    for N, Np, Np3 in ((int(a), int(b), int(c)) for a, b, c in rows):
        e = refelems(N)
        assert e.Np == Np and 3 * e.Np == Np3
        assert e.Dr.shape == (Np, Np) and e.LIFT.shape == (Np, 4 * e.Nfp)
        assert e.Nfp == (N + 1) * (N + 2) // 2


# ---------------------------------------------------------------- Jacobi / GLL
@pytest.mark.parametrize("ab", [(0, 0), (1, 0), (3, 0), (1, 1), (8, 0), (22, 0)])
def test_jacobi_against_scipy(ab):
    a, b = ab
    x = np.linspace(-1, 1, 41)
    for n in range(0, 11):
        # squared norm of the classical Jacobi polynomial
        h = (2.0 ** (a + b + 1) / (2 * n + a + b + 1) * math.gamma(n + a + 1) * math.gamma(n + b + 1)
             / (math.gamma(n + a + b + 1) * math.factorial(n)))
        want = sp.eval_jacobi(n, a, b, x) / math.sqrt(h)
        got = refelem.jacobi_p(x, a, b, n)
        assert np.allclose(got, want, rtol=1e-11, atol=1e-11 * np.abs(want).max())
        # derivative by scipy's own derivative relation on the classical polynomial
        if n > 0:
            dwant = 0.5 * (n + a + b + 1) * sp.eval_jacobi(n - 1, a + 1, b + 1, x) / math.sqrt(h)
            assert np.allclose(refelem.grad_jacobi_p(x, a, b, n), dwant, rtol=1e-10, atol=1e-10 * np.abs(dwant).max())


def test_gauss_lobatto_closed_forms():
    env = {"sqrt": math.sqrt}
    for line in open(os.path.join(GOLD, "gauss_lobatto_nodes.txt")):
        if line.startswith("#") or not line.strip():
            continue
        n, exprs = line.split(":")
        want = np.array([-1.0] + [eval(e, env) for e in exprs.split()] + [1.0])
        assert np.allclose(refelem.gauss_lobatto(int(n)), want, atol=1e-13)
    for N in DEGREES:                       # zeros of (1-x^2) P_N'
        x = refelem.gauss_lobatto(N)
        dP = sp.eval_jacobi(N - 1, 1, 1, x[1:-1]) if N > 1 else np.zeros(0)
        assert np.allclose(dP, 0, atol=1e-10)


def test_gauss_jacobi_nodes_against_scipy():
    for (a, b, n) in [(0, 0, 5), (1, 0, 7), (2, 0, 9), (1, 1, 6)]:
        want, _ = sp.roots_jacobi(n + 1, a, b)
        assert np.allclose(refelem.jacobi_gauss(a, b, n), want, atol=1e-12)


# ---------------------------------------------------------------- T1 nodes
@pytest.mark.parametrize("N", DEGREES)
def test_nodes_T1(refelems, N):
    e = refelems(N)
    pts = np.stack([e.r, e.s, e.t], axis=1)
    assert pts.shape == (e.Np, 3)
    lam = np.stack([-(1 + e.r + e.s + e.t) / 2, (1 + e.r) / 2, (1 + e.s) / 2, (1 + e.t) / 2], axis=1)
    assert lam.min() > -1e-12                                      # inside the element
    # symmetric under all 24 vertex permutations (as a set)
    key = lambda a: np.array(sorted(map(tuple, np.round(a, 9))))   # noqa: E731
    base = key(lam)
    for perm in itertools.permutations(range(4)):
        assert np.allclose(key(lam[:, perm]), base, atol=1e-8)
    # every face holds Nfp nodes and every edge the Gauss-Lobatto points
    gl = refelem.gauss_lobatto(N)
    for f in range(4):
        assert len(e.Fmask[f]) == e.Nfp
    for (u, v) in itertools.combinations(range(4), 2):
        others = [w for w in range(4) if w not in (u, v)]
        on_edge = np.all(np.abs(lam[:, others]) < 1e-10, axis=1)
        xi = np.sort(lam[on_edge, v] - lam[on_edge, u])
        assert np.allclose(xi, gl, atol=1e-10)
    # the four face node sets are the same 2-D set (in face barycentrics)
    verts = [(0, 1, 2), (0, 1, 3), (1, 2, 3), (0, 2, 3)]
    sets = [key(lam[e.Fmask[f]][:, verts[f]]) for f in range(4)]
    for s_ in sets[1:]:
        assert np.allclose(s_, sets[0], atol=1e-8)
    assert np.linalg.cond(e.V) < 1e4
    # lattice order: t slowest, then s, r fastest (ABI convention, include/dg.h)
    idx = {(i, j, k): n for n, (i, j, k) in enumerate(
        (i, j, k) for k in range(N + 1) for j in range(N + 1 - k) for i in range(N + 1 - j - k))}
    for (i, j, k), n in idx.items():          # coordinates grow monotonically along each lattice line
        if (i + 1, j, k) in idx:
            assert e.r[idx[(i + 1, j, k)]] > e.r[n] + 1e-6
        if (i, j + 1, k) in idx:
            assert e.s[idx[(i, j + 1, k)]] > e.s[n] + 1e-6
        if (i, j, k + 1) in idx:
            assert e.t[idx[(i, j, k + 1)]] > e.t[n] + 1e-6
    assert np.array_equal(e.Fmask[0], np.arange(e.Nfp))


# ---------------------------------------------------------------- T2 exact differentiation
@pytest.mark.parametrize("N", DEGREES)
def test_exact_differentiation_T2(refelems, N):
    e = refelems(N)
    r, s, t = e.r, e.s, e.t
    tol = 1e-10 * N ** 4
    for a in range(N + 1):
        for b in range(N + 1 - a):
            for c in range(N + 1 - a - b):
                u = r ** a * s ** b * t ** c
                ur = a * r ** (a - 1) * s ** b * t ** c if a else 0 * u
                us = b * r ** a * s ** (b - 1) * t ** c if b else 0 * u
                ut = c * r ** a * s ** b * t ** (c - 1) if c else 0 * u
                assert np.abs(e.Dr @ u - ur).max() < tol
                assert np.abs(e.Ds @ u - us).max() < tol
                assert np.abs(e.Dt @ u - ut).max() < tol


def test_differentiation_beyond_degree_is_inexact(refelems):
    e = refelems(3)
    u = e.r ** 4
    assert np.abs(e.Dr @ u - 4 * e.r ** 3).max() > 1e-3           # the pin above is not vacuous


# ---------------------------------------------------------------- quadrature helpers (scipy only)
def tet_quadrature(n):
    """Collapsed tensor Gauss-Jacobi rule on the reference tet, exact to degree 2n-1."""
    xa, wa = sp.roots_jacobi(n, 0, 0)
    xb, wb = sp.roots_jacobi(n, 1, 0)
    xc, wc = sp.roots_jacobi(n, 2, 0)
    A, B, C = np.meshgrid(xa, xb, xc, indexing="ij")
    Wt = (wa[:, None, None] * wb[None, :, None] * wc[None, None, :]) / 8.0
    a, b, c = A.ravel(), B.ravel(), C.ravel()
    t = c
    s = (1 + b) * (1 - c) / 2 - 1
    r = (1 + a) * (-(s + t)) / 2 - 1
    return r, s, t, Wt.ravel()


def tri_quadrature(n):
    xa, wa = sp.roots_jacobi(n, 0, 0)
    xb, wb = sp.roots_jacobi(n, 1, 0)
    A, B = np.meshgrid(xa, xb, indexing="ij")
    W = (wa[:, None] * wb[None, :]) / 2.0
    a, b = A.ravel(), B.ravel()
    w = b
    u = (1 + a) * (1 - b) / 2 - 1
    return u, w, W.ravel()


def test_quadrature_helpers_closed_forms():
    r, s, t, w = tet_quadrature(6)
    assert abs(w.sum() - 4.0 / 3.0) < 1e-13
    # int r^2 over the reference tet = 2/5 ... check by the closed form of barycentric monomials:
    # int lam2^2 dV = |T| * 2!*3!/(5!) * ... = (4/3) * 2 * 6 / 120
    lam2 = (1 + r) / 2
    assert abs(np.sum(w * lam2 ** 2) - (4.0 / 3.0) * 2 * 6 / 120) < 1e-13
    u, v, w2 = tri_quadrature(6)
    assert abs(w2.sum() - 2.0) < 1e-13


# ---------------------------------------------------------------- T3 mass matrix
@pytest.mark.parametrize("N", DEGREES)
def test_mass_matrix_T3(refelems, N):
    e = refelems(N)
    M = e.M
    assert np.allclose(M, M.T, atol=1e-13)
    np.linalg.cholesky(M)                                            # SPD
    one = np.ones(e.Np)
    assert abs(one @ M @ one - 4.0 / 3.0) < 1e-11                    # volume of the reference tet
    assert np.allclose(e.V.T @ M @ e.V, np.eye(e.Np), atol=1e-9)
    # orthonormality of the modal basis by independent quadrature (pins 2 sqrt 2 and the Jacobi norms)
    r, s, t, w = tet_quadrature(N + 2)
    Vq = refelem.vandermonde3d(N, r, s, t)
    assert np.allclose(Vq.T @ (w[:, None] * Vq), np.eye(e.Np), atol=1e-10)
    # nodal mass matrix = int l_i l_j by the same quadrature
    Lq = np.linalg.solve(e.V.T, Vq.T).T                              # Lagrange functions at quadrature points
    assert np.allclose(Lq.T @ (w[:, None] * Lq), M, atol=1e-10)


# ---------------------------------------------------------------- T4/T5 lift
FACE_UV = (("r", "s"), ("r", "t"), ("s", "t"), ("s", "t"))


@pytest.mark.parametrize("N", DEGREES)
def test_face_mass_and_lift_T4_T5(refelems, N):
    e = refelems(N)
    Np, Nfp = e.Np, e.Nfp
    assert np.allclose(e.M @ e.LIFT, e.Emat, atol=1e-9)              # M LIFT = E
    coords = {"r": e.r, "s": e.s, "t": e.t}
    u, w, wq = tri_quadrature(N + 2)
    Ehat = []
    for f in range(4):
        # embed the quadrature points into the face
        if f == 0:
            rq, sq, tq = u, w, -np.ones_like(u)
        elif f == 1:
            rq, sq, tq = u, -np.ones_like(u), w
        elif f == 2:
            sq, tq = u, w
            rq = -1 - sq - tq
        else:
            rq, sq, tq = -np.ones_like(u), u, w
        Lq = np.linalg.solve(e.V.T, refelem.vandermonde3d(N, rq, sq, tq).T).T     # Np Lagrange fns on the face
        Mf = Lq.T @ (wq[:, None] * Lq)                               # Np x Np, nonzero only on face nodes
        off = np.setdiff1d(np.arange(Np), e.Fmask[f])
        assert np.abs(Mf[off]).max() < 1e-10
        assert np.allclose(Mf[np.ix_(e.Fmask[f], e.Fmask[f])], e.Emat[e.Fmask[f], f * Nfp:(f + 1) * Nfp], atol=1e-10)
        Ehat.append(Mf)
    # summation by parts: M D + D^T M = sum_f ntilde_f E_f with the reference normals
    M = e.M
    assert np.allclose(M @ e.Dr + e.Dr.T @ M, Ehat[2] - Ehat[3], atol=1e-9)
    assert np.allclose(M @ e.Ds + e.Ds.T @ M, Ehat[2] - Ehat[1], atol=1e-9)
    assert np.allclose(M @ e.Dt + e.Dt.T @ M, Ehat[2] - Ehat[0], atol=1e-9)
