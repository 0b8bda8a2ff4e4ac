"""Reference tetrahedron operators in fp64 (oracle; test infrastructure only).

Follows PAPER.md:88-106 (eq. (1)-(3)): nodal Lagrange representation with
Np=(N+1)(N+2)(N+3)/6 warp-and-blend nodes, differentiation matrices D_j and
lift matrices L_f merged into one Np x 4Nfp matrix L (Table 1).
The paper defers the definitions to its refs [33]/[20]/[44]; the readings
used here are DESIGN.md Q3 (nodes) and Q4 (operators):

reference element  {(r,s,t) : r,s,t >= -1, r+s+t <= -1}
vertices           v1=(-1,-1,-1) v2=(1,-1,-1) v3=(-1,1,-1) v4=(-1,-1,1)
faces              f1: t=-1 (v1,v2,v3)   f2: s=-1 (v1,v2,v4)
                   f3: r+s+t=-1 (v2,v3,v4)   f4: r=-1 (v1,v3,v4)
node order         lattice order, t slowest, then s, r fastest
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np


# --------------------------------------------------------------------------
# Jacobi polynomials, orthonormal on [-1,1] w.r.t. (1-x)^a (1+x)^b
# --------------------------------------------------------------------------
def jacobi_p(x, a: float, b: float, n: int):
    """Orthonormal Jacobi polynomial P_n^{(a,b)}(x), three-term recurrence."""
    x = np.asarray(x, dtype=np.float64)
    g0 = 2.0 ** (a + b + 1) / (a + b + 1) * math.gamma(a + 1) * math.gamma(b + 1) / math.gamma(a + b + 1)
    p_prev = np.full_like(x, 1.0 / math.sqrt(g0))
    if n == 0:
        return p_prev
    g1 = (a + 1) * (b + 1) / (a + b + 3) * g0
    p_cur = ((a + b + 2) * x / 2 + (a - b) / 2) / math.sqrt(g1)
    if n == 1:
        return p_cur
    a_old = 2.0 / (2 + a + b) * math.sqrt((a + 1) * (b + 1) / (a + b + 3))
    for i in range(1, n):
        h = 2 * i + a + b
        a_new = 2.0 / (h + 2) * math.sqrt((i + 1) * (i + 1 + a + b) * (i + 1 + a) * (i + 1 + b) / ((h + 1) * (h + 3)))
        b_new = -(a * a - b * b) / (h * (h + 2))
        p_next = (-a_old * p_prev + (x - b_new) * p_cur) / a_new
        p_prev, p_cur, a_old = p_cur, p_next, a_new
    return p_cur


def grad_jacobi_p(x, a: float, b: float, n: int):
    """d/dx of the orthonormal P_n^{(a,b)}: sqrt(n(n+a+b+1)) P_{n-1}^{(a+1,b+1)}."""
    x = np.asarray(x, dtype=np.float64)
    if n == 0:
        return np.zeros_like(x)
    return math.sqrt(n * (n + a + b + 1.0)) * jacobi_p(x, a + 1, b + 1, n - 1)


def jacobi_gauss(a: float, b: float, n: int):
    """(n+1)-point Gauss-Jacobi nodes (Golub-Welsch on the Jacobi matrix)."""
    if n == 0:
        return np.array([-(a - b) / (a + b + 2)])
    k = np.arange(1, n + 1, dtype=np.float64)
    h = 2 * k + a + b
    diag = np.empty(n + 1)
    diag[0] = (b - a) / (a + b + 2)
    diag[1:] = -(a * a - b * b) / (h * (h + 2))
    k1 = np.arange(1, n + 1, dtype=np.float64)
    off = 2.0 / (2 * k1 + a + b) * np.sqrt(k1 * (k1 + a + b) * (k1 + a) * (k1 + b) / ((2 * k1 + a + b - 1) * (2 * k1 + a + b + 1)))
    T = np.diag(diag) + np.diag(off, 1) + np.diag(off, -1)
    return np.sort(np.linalg.eigvalsh(T))


def gauss_lobatto(n: int):
    """(n+1) Gauss-Lobatto-Legendre points: +-1 and the zeros of P_n'."""
    if n == 1:
        return np.array([-1.0, 1.0])
    inner = jacobi_gauss(1.0, 1.0, n - 2)
    return np.concatenate(([-1.0], inner, [1.0]))


# --------------------------------------------------------------------------
# warp-and-blend nodes (ref [44]); Q3: blend parameter 0
# --------------------------------------------------------------------------
def _edge_warp(N: int, xi):
    """Displacement that carries the (N+1) equispaced points of [-1,1] onto the
    Gauss-Lobatto points, interpolated with the equispaced Lagrange basis and
    divided by (1 - xi^2)."""
    xi = np.asarray(xi, dtype=np.float64)
    xeq = np.linspace(-1.0, 1.0, N + 1)
    xgl = gauss_lobatto(N)
    w = np.zeros_like(xi)
    for i in range(N + 1):
        li = np.ones_like(xi)
        for j in range(N + 1):
            if j != i:
                li *= (xi - xeq[j]) / (xeq[i] - xeq[j])
        w += (xgl[i] - xeq[i]) * li
    # scaled by 1/(1 - xi^2): the blend 4 lam_u lam_v equals 1 - xi^2 on the edge itself
    inside = np.abs(xi) < 1.0 - 1e-10
    out = np.zeros_like(w)
    out[inside] = w[inside] / (1.0 - xi[inside] ** 2)
    return out


def nodes_tet(N: int, alpha: float = 0.0):
    """Warp-and-blend nodes of degree N on the reference tetrahedron -> r,s,t."""
    tol = 1e-10
    # barycentric lattice, t slowest, s, then r fastest
    ijk = [(i, j, k) for k in range(N + 1) for j in range(N + 1 - k) for i in range(N + 1 - j - k)]
    ijk = np.array(ijk, dtype=np.float64)
    lam = np.empty((len(ijk), 4))
    lam[:, 1] = ijk[:, 0] / N          # weight of v2 (r direction)
    lam[:, 2] = ijk[:, 1] / N          # weight of v3 (s direction)
    lam[:, 3] = ijk[:, 2] / N          # weight of v4 (t direction)
    lam[:, 0] = 1.0 - lam[:, 1] - lam[:, 2] - lam[:, 3]
    # equilateral tetrahedron with edge length 2
    V = np.array([[-1.0, -1 / math.sqrt(3), -1 / math.sqrt(6)],
                  [1.0, -1 / math.sqrt(3), -1 / math.sqrt(6)],
                  [0.0, 2 / math.sqrt(3), -1 / math.sqrt(6)],
                  [0.0, 0.0, 3 / math.sqrt(6)]])
    X = lam @ V
    shift = np.zeros_like(X)
    for a in range(4):                       # face opposite vertex a
        b, c, d = [v for v in range(4) if v != a]
        la, lb, lc, ld = lam[:, a], lam[:, b], lam[:, c], lam[:, d]
        # 2-D warp in the plane of the face: sum of the three edge warps
        W = np.zeros_like(X)
        for (u, v, o) in ((b, c, d), (c, d, b), (d, b, c)):
            lu, lv, lo = lam[:, u], lam[:, v], lam[:, o]
            e = (V[v] - V[u]) / np.linalg.norm(V[v] - V[u])
            mag = 4.0 * lu * lv * _edge_warp(N, lv - lu) * (1.0 + (alpha * lo) ** 2)
            W += mag[:, None] * e[None, :]
        denom = (lb + 0.5 * la) * (lc + 0.5 * la) * (ld + 0.5 * la)
        blend = np.zeros_like(la)
        ok = denom > tol
        blend[ok] = (1.0 + (alpha * la[ok]) ** 2) * lb[ok] * lc[ok] * ld[ok] / denom[ok]
        shift += blend[:, None] * W
        # nodes on the boundary of this face take the face's warp exactly
        on_rim = (la < tol) & (((lb > tol).astype(int) + (lc > tol) + (ld > tol)) < 3)
        shift[on_rim] = W[on_rim]
    X = X + shift
    # back to the reference element: barycentric weights of the moved point
    A = (V[1:] - V[0]).T
    mu = np.linalg.solve(A, (X - V[0]).T).T       # weights of v2, v3, v4
    r = -1.0 + 2.0 * mu[:, 0]
    s = -1.0 + 2.0 * mu[:, 1]
    t = -1.0 + 2.0 * mu[:, 2]
    return r, s, t


# --------------------------------------------------------------------------
# orthonormal Dubiner basis on the tetrahedron and the triangle
# --------------------------------------------------------------------------
def rst_to_abc(r, s, t):
    r, s, t = (np.asarray(v, dtype=np.float64) for v in (r, s, t))
    a = np.full_like(r, -1.0)
    m = np.abs(s + t) > 1e-14
    a[m] = 2.0 * (1.0 + r[m]) / (-s[m] - t[m]) - 1.0
    b = np.full_like(r, -1.0)
    m = np.abs(t - 1.0) > 1e-14
    b[m] = 2.0 * (1.0 + s[m]) / (1.0 - t[m]) - 1.0
    return a, b, t.copy()


def basis_index(N: int):
    """(i,j,k) with i+j+k <= N in the order of the Vandermonde columns."""
    return [(i, j, k) for i in range(N + 1) for j in range(N + 1 - i) for k in range(N + 1 - i - j)]


def dubiner3d(a, b, c, i: int, j: int, k: int):
    """psi_ijk = 2 sqrt2 P_i^{0,0}(a) P_j^{2i+1,0}(b)(1-b)^i P_k^{2i+2j+2,0}(c)(1-c)^{i+j}."""
    return (2.0 * math.sqrt(2.0) * jacobi_p(a, 0, 0, i) * jacobi_p(b, 2 * i + 1, 0, j) * (1 - b) ** i
            * jacobi_p(c, 2 * (i + j) + 2, 0, k) * (1 - c) ** (i + j))


def grad_dubiner3d(a, b, c, i: int, j: int, k: int):
    """(d/dr, d/ds, d/dt) psi_ijk by the chain rule through (a,b,c).

    With da/dr = 4/((1-b)(1-c)), da/ds = da/dt = 2(1+a)/((1-b)(1-c)),
    db/ds = 2/(1-c), db/dt = (1+b)/(1-c), dc/dt = 1 the singular factors
    cancel against the (1-b)^i (1-c)^{i+j} weights.
    """
    fa, dfa = jacobi_p(a, 0, 0, i), grad_jacobi_p(a, 0, 0, i)
    gb, dgb = jacobi_p(b, 2 * i + 1, 0, j), grad_jacobi_p(b, 2 * i + 1, 0, j)
    hc, dhc = jacobi_p(c, 2 * (i + j) + 2, 0, k), grad_jacobi_p(c, 2 * (i + j) + 2, 0, k)
    pb = lambda e: (1 - b) ** e if e > 0 else np.ones_like(b)   # noqa: E731
    pc = lambda e: (1 - c) ** e if e > 0 else np.ones_like(c)   # noqa: E731
    # pieces:  B = gb (1-b)^i,  C = hc (1-c)^{i+j}
    dB = dgb * pb(i) - (i * gb * pb(i - 1) if i > 0 else 0.0)
    dC = dhc * pc(i + j) - ((i + j) * hc * pc(i + j - 1) if i + j > 0 else 0.0)
    # fa' * B * C / ((1-b)(1-c))  (zero when i == 0 because fa' == 0)
    core = dfa * gb * hc * pb(i - 1) * pc(i + j - 1) if i > 0 else np.zeros_like(a)
    # fa * B' * C / (1-c)         (zero when i + j == 0 because B' == 0)
    mid = fa * dB * hc * pc(i + j - 1) if i + j > 0 else np.zeros_like(a)
    dr = 4.0 * core
    ds = 2.0 * (1 + a) * core + 2.0 * mid
    dt = 2.0 * (1 + a) * core + (1 + b) * mid + fa * gb * pb(i) * dC
    f = 2.0 * math.sqrt(2.0)
    return f * dr, f * ds, f * dt


def vandermonde3d(N: int, r, s, t):
    a, b, c = rst_to_abc(r, s, t)
    return np.stack([dubiner3d(a, b, c, i, j, k) for (i, j, k) in basis_index(N)], axis=1)


def grad_vandermonde3d(N: int, r, s, t):
    a, b, c = rst_to_abc(r, s, t)
    cols = [grad_dubiner3d(a, b, c, i, j, k) for (i, j, k) in basis_index(N)]
    return tuple(np.stack([col[d] for col in cols], axis=1) for d in range(3))


def dubiner2d(a, b, i: int, j: int):
    """sqrt2 P_i^{0,0}(a) P_j^{2i+1,0}(b) (1-b)^i on the reference triangle."""
    return math.sqrt(2.0) * jacobi_p(a, 0, 0, i) * jacobi_p(b, 2 * i + 1, 0, j) * (1 - b) ** i


def vandermonde2d(N: int, u, w):
    u, w = np.asarray(u, dtype=np.float64), np.asarray(w, dtype=np.float64)
    a = np.full_like(u, -1.0)
    m = np.abs(w - 1.0) > 1e-14
    a[m] = 2.0 * (1.0 + u[m]) / (1.0 - w[m]) - 1.0
    return np.stack([dubiner2d(a, w, i, j) for i in range(N + 1) for j in range(N + 1 - i)], axis=1)


# --------------------------------------------------------------------------
# the assembled reference element
# --------------------------------------------------------------------------
@dataclass
class RefElem:
    N: int
    Np: int
    Nfp: int
    r: np.ndarray
    s: np.ndarray
    t: np.ndarray
    V: np.ndarray          # Vandermonde, Np x Np
    Dr: np.ndarray
    Ds: np.ndarray
    Dt: np.ndarray
    M: np.ndarray          # mass matrix (V V^T)^-1
    Fmask: np.ndarray      # 4 x Nfp volume-node indices of each face
    Emat: np.ndarray       # Np x 4Nfp face-mass matrices scattered to face rows
    LIFT: np.ndarray       # Np x 4Nfp merged lift matrix  M^-1 E


def face_masks(r, s, t, Nfp: int, tol: float = 1e-10):
    f1 = np.flatnonzero(np.abs(1 + t) < tol)
    f2 = np.flatnonzero(np.abs(1 + s) < tol)
    f3 = np.flatnonzero(np.abs(1 + r + s + t) < tol)
    f4 = np.flatnonzero(np.abs(1 + r) < tol)
    for f in (f1, f2, f3, f4):
        if len(f) != Nfp:
            raise ValueError("face does not hold Nfp nodes")
    return np.stack([f1, f2, f3, f4])


def build(N: int, alpha: float = 0.0) -> RefElem:
    if N < 1:
        raise ValueError("N >= 1")
    Np = (N + 1) * (N + 2) * (N + 3) // 6
    Nfp = (N + 1) * (N + 2) // 2
    r, s, t = nodes_tet(N, alpha)
    V = vandermonde3d(N, r, s, t)
    Vr, Vs, Vt = grad_vandermonde3d(N, r, s, t)
    # D = V_r V^-1  <=>  D V = V_r  <=>  V^T D^T = V_r^T
    Dr = np.linalg.solve(V.T, Vr.T).T
    Ds = np.linalg.solve(V.T, Vs.T).T
    Dt = np.linalg.solve(V.T, Vt.T).T
    VVt = V @ V.T
    M = np.linalg.inv(VVt)
    M = 0.5 * (M + M.T)
    Fmask = face_masks(r, s, t, Nfp)
    E = np.zeros((Np, 4 * Nfp))
    face_uv = ((r, s), (r, t), (s, t), (s, t))     # free parametric coordinates of each face
    for f in range(4):
        idx = Fmask[f]
        Vf = vandermonde2d(N, face_uv[f][0][idx], face_uv[f][1][idx])
        Mf = np.linalg.inv(Vf @ Vf.T)
        E[idx, f * Nfp:(f + 1) * Nfp] = 0.5 * (Mf + Mf.T)
    LIFT = VVt @ E
    return RefElem(N, Np, Nfp, r, s, t, V, Dr, Ds, Dt, M, Fmask, E, LIFT)
