"""LSRK(5,4) update, stable time step and discrete energy (oracle; test
infrastructure only).

The paper integrates with AB3 (eq. (4)); BASELINE.json's
north_star and configs name the five-stage fourth-order low-storage
Runge-Kutta scheme of Carpenter & Kennedy instead (readings Q1, Q2):

    res <- A_s res + dt r(q) ;  q <- q + B_s res ,   s = 1..5,  A_1 = 0.

AB3 (eq. (4)) is provided as well because it is what the paper prints.
"""
from __future__ import annotations

from fractions import Fraction

import numpy as np

from .mesh import Mesh
from .refelem import RefElem

LSRK_A_FRAC = (Fraction(0),
               Fraction(-567301805773, 1357537059087),
               Fraction(-2404267990393, 2016746695238),
               Fraction(-3550918686646, 2091501179385),
               Fraction(-1275806237668, 842570457699))
LSRK_B_FRAC = (Fraction(1432997174477, 9575080441755),
               Fraction(5161836677717, 13612068292357),
               Fraction(1720146321549, 2090206949498),
               Fraction(3134564353537, 4481467310338),
               Fraction(2277821191437, 14882151754819))
LSRK_A = tuple(float(a) for a in LSRK_A_FRAC)
LSRK_B = tuple(float(b) for b in LSRK_B_FRAC)

AB3 = (23.0 / 12.0, -16.0 / 12.0, 5.0 / 12.0)       # eq. (4)


def lsrk_step(q, res, dt, rhs):
    """One LSRK(5,4) step in place on (q, res); rhs(q) returns r(q)."""
    for A, B in zip(LSRK_A, LSRK_B):
        res *= A
        res += dt * rhs(q)
        q += B * res
    return q


def lsrk_run(q0, dt, nsteps, rhs):
    q = np.array(q0, dtype=np.float64, copy=True)
    res = np.zeros_like(q)
    for _ in range(nsteps):
        lsrk_step(q, res, dt, rhs)
    return q


def ab3_step(q, r_hist, dt, rhs):
    """eq. (4):  q^{m+1} = q^m + dt (23/12 r^m - 16/12 r^{m-1} + 5/12 r^{m-2}).

    r_hist: the right-hand sides of earlier steps, newest first, at most two; updated in place.
    Start-up (reading Q21: eq. (4) needs r^{m-1}, r^{m-2}, and the paper does not say how the first two steps
    are taken): while fewer than two earlier right-hand sides exist the step is one LSRK(5,4) step -- fourth order, so
    the third order of eq. (4) survives; starting eq. (4) from a zero history instead leaves an O(dt) error that never
    decays -- and r(q^m) is recorded for the steps that follow."""
    r0 = rhs(q)
    if len(r_hist) < 2:
        lsrk_step(q, np.zeros_like(q), dt, rhs)
    else:
        q += dt * (AB3[0] * r0 + AB3[1] * r_hist[0] + AB3[2] * r_hist[1])
    r_hist.insert(0, r0)
    del r_hist[2:]
    return q


def stable_dt(ref: RefElem, mesh: Mesh, cmax, cfl: float = 0.5) -> float:
    """dt = CFL / ((N+1)^2 max_k [c_max,k max_f g^sur_{k,f}])   (Q10)."""
    cmax = np.asarray(cmax, dtype=np.float64)
    return float(cfl / ((ref.N + 1) ** 2 * np.max(cmax * mesh.Fscale.max(axis=1))))


def _mass_quadratic(ref: RefElem, mesh: Mesh, u, v):
    """sum_k J_k u_k^T M v_k for u, v of shape K x Np."""
    return float(np.sum(mesh.J * np.einsum("kn,nm,km->k", u, ref.M, v)))


def energy_acoustic(ref, mesh, rho, c, q):
    """1/2 int p^2/(rho c^2) + rho |v|^2."""
    rho, c = np.asarray(rho, float)[:, None], np.asarray(c, float)[:, None]
    p, v = q[:, 0], q[:, 1:4]
    e = _mass_quadratic(ref, mesh, p / (rho * c * c), p)
    for i in range(3):
        e += _mass_quadratic(ref, mesh, rho * v[:, i], v[:, i])
    return 0.5 * e


def energy_gradient_acoustic(ref, mesh, rho, c, q):
    """W q with E = 1/2 q^T W q (same layout as q, before the mass matrix)."""
    rho, c = np.asarray(rho, float)[:, None, None], np.asarray(c, float)[:, None, None]
    w = np.empty_like(q)
    w[:, 0:1] = q[:, 0:1] / (rho * c * c)
    w[:, 1:4] = rho * q[:, 1:4]
    return mesh.J[:, None, None] * (w @ ref.M)


def energy_gradient_elastic(ref, mesh, rho, vp, vs, q):
    """W q for E = 1/2 int rho |v|^2 + sigma : C^-1 : sigma, with
    sigma:C^-1:sigma = (1/2mu)[sigma:sigma - lambda/(3 lambda + 2 mu) (tr sigma)^2]."""
    rho, vp, vs = (np.asarray(a, float)[:, None] for a in (rho, vp, vs))
    mu = rho * vs ** 2
    lam = rho * vp ** 2 - 2 * mu
    w = np.empty_like(q)
    w[:, 0:3] = rho[:, None] * q[:, 0:3]
    tr = q[:, 3] + q[:, 4] + q[:, 5]
    for a in (3, 4, 5):
        w[:, a] = (q[:, a] - lam / (3 * lam + 2 * mu) * tr) / (2 * mu)
    for a in (6, 7, 8):
        w[:, a] = 2 * q[:, a] / (2 * mu)            # off-diagonals count twice
    return mesh.J[:, None, None] * (w @ ref.M)


def energy_elastic(ref, mesh, rho, vp, vs, q):
    return 0.5 * float(np.sum(q * energy_gradient_elastic(ref, mesh, rho, vp, vs, q)))
