"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests, and
therefore holds none of the method's arithmetic: it only draws meshes,
materials and initial fields.  It imports neither ``oracle`` nor the CUDA
binding.  Everything is numpy on the host, fp64, deterministic in the seed.

The paper measured on its own tetrahedral meshes of about 2 M nodes per degree
(PAPER.md:225); those meshes are not available, so BASELINE.json's configs
replace them by Kuhn-split unit cubes.

PRNG: SplitMix64 used as a counter-based generator -- draw i of stream `seed`
is mix(seed + (i+1)*0x9E3779B97F4A7C15); uniform = top 53 bits * 2^-53;
normals by Box-Muller on consecutive pairs.
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field

import numpy as np

BC_INTERIOR, BC_RIGID, BC_FREE, BC_SLIP = 0, 1, 2, 3
ACOUSTIC, ELASTIC = 0, 1
NFIELDS = {ACOUSTIC: 4, ELASTIC: 9}

# local vertex numbers of the four faces, the ABI's face convention (include/dg.h)
FACE_VERTS = np.array([[0, 1, 2], [0, 1, 3], [1, 2, 3], [0, 2, 3]])


# --------------------------------------------------------------------------
# counter-based PRNG
# --------------------------------------------------------------------------
def _splitmix64(seed: int, count: int, offset: int = 0) -> np.ndarray:
    with np.errstate(over="ignore"):
        i = np.arange(offset + 1, offset + count + 1, dtype=np.uint64)
        z = np.uint64(seed) + i * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniform(seed: int, count: int, lo: float = 0.0, hi: float = 1.0, offset: int = 0) -> np.ndarray:
    u = (_splitmix64(seed, count, offset) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
    return lo + (hi - lo) * u


def normal(seed: int, count: int) -> np.ndarray:
    m = (count + 1) // 2
    u = uniform(seed, 2 * m)
    u1 = 1.0 - u[0::2]                       # (0, 1]
    u2 = u[1::2]
    rad = np.sqrt(-2.0 * np.log(u1))
    out = np.empty(2 * m)
    out[0::2] = rad * np.cos(2 * np.pi * u2)
    out[1::2] = rad * np.sin(2 * np.pi * u2)
    return out[:count]


# --------------------------------------------------------------------------
# meshes
# --------------------------------------------------------------------------
def kuhn_cube(n: int, jitter: float = 0.05, seed: int = 1):
    """Unit cube of n^3 cells, each cut into the 6 Kuhn tetrahedra.

    Returns vxyz (nv x 3, float64), etov (K x 4, int32, positive orientation),
    cell (K,) lexicographic cell index (x fastest) of each element.  Interior
    vertices are moved by U[-jitter*h, jitter*h]^3; wall vertices stay put.
    """
    m = n + 1
    h = 1.0 / n
    iz, iy, ix = np.meshgrid(np.arange(m), np.arange(m), np.arange(m), indexing="ij")
    lat = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1)
    vxyz = lat.astype(np.float64) * h
    inner = np.all((lat > 0) & (lat < n), axis=1)
    d = uniform(seed, 3 * m ** 3, -jitter * h, jitter * h).reshape(-1, 3)
    vxyz[inner] += d[inner]
    cz, cy, cx = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    c0 = np.stack([cx.ravel(), cy.ravel(), cz.ravel()], axis=1)          # ncell x 3
    vid = lambda p: p[..., 0] + m * (p[..., 1] + m * p[..., 2])          # noqa: E731
    tets = []
    for perm in itertools.permutations(range(3)):
        e1 = np.zeros(3, dtype=np.int64); e1[perm[0]] = 1
        e2 = e1.copy(); e2[perm[1]] = 1
        corners = [c0, c0 + e1, c0 + e2, c0 + 1]
        # sign of the permutation = orientation of the tetrahedron
        sign = np.linalg.det(np.eye(3)[list(perm)])
        if sign < 0:
            corners[2], corners[3] = corners[3], corners[2]
        tets.append(np.stack([vid(p) for p in corners], axis=1))
    etov = np.stack(tets, axis=1).reshape(-1, 4).astype(np.int32)         # cell-major, 6 per cell
    cell = np.repeat(np.arange(n ** 3), 6)
    return vxyz, etov, cell


def wall_tags(n: int, etov: np.ndarray, top: int = BC_RIGID, other: int = BC_RIGID) -> np.ndarray:
    """K x 4 int8 tags: faces lying in a wall of the cube get `other`, the wall
    z = 1 gets `top`; all other faces 0 (interior)."""
    m = n + 1
    fv = etov[:, FACE_VERTS].astype(np.int64)                  # K x 4 x 3
    lat = np.stack([fv % m, (fv // m) % m, fv // (m * m)], axis=-1)   # K x 4 x 3verts x 3axes
    tag = np.zeros(etov.shape[0:1] + (4,), dtype=np.int8)
    for ax in range(3):
        for side in (0, n):
            on = np.all(lat[..., ax] == side, axis=2)
            tag[on] = top if (ax == 2 and side == n) else other
    return tag


# --------------------------------------------------------------------------
# materials and fields
# --------------------------------------------------------------------------
def random_acoustic_materials(K: int, seed: int = 2):
    """c in U[1,3], rho in U[1,2.5] per element (BASELINE.json configs[1])."""
    c = uniform(seed, K, 1.0, 3.0)
    rho = uniform(seed + 1000003, K, 1.0, 2.5)
    return rho, c


def random_elastic_materials(K: int, seed: int = 2, rho_rng=(1.0, 2.5), vp_rng=(1.0, 3.0)):
    """rho, vp uniform in the given ranges, vs = vp / U[1.6, 2.0] (configs[3], configs[4])."""
    vp = uniform(seed, K, *vp_rng)
    rho = uniform(seed + 1000003, K, *rho_rng)
    vs = vp / uniform(seed + 2000003, K, 1.6, 2.0)
    return rho, vp, vs


def layered_elastic_materials(n: int, cell: np.ndarray):
    """Three horizontal layers (configs[2]); top z in [2/3,1] is the slowest."""
    cz = cell // (n * n)
    layer = np.minimum((3 * cz) // n, 2)                        # 0 bottom .. 2 top
    table = np.array([[2.7, 4.5, 2.6], [2.4, 3.0, 1.7], [2.0, 2.0, 1.0]])
    m = table[layer]
    return m[:, 0].copy(), m[:, 1].copy(), m[:, 2].copy()


def standing_mode(xyz: np.ndarray, t: float = 0.0) -> np.ndarray:
    """Closed-form acoustic mode in the rigid unit cube for c = rho = 1
    (BASELINE.json north_star): p = cos(pi x)cos(pi y)cos(pi z)cos(sqrt3 pi t)."""
    x, y, z = np.pi * xyz[..., 0], np.pi * xyz[..., 1], np.pi * xyz[..., 2]
    w = np.sqrt(3.0) * np.pi
    q = np.empty(xyz.shape[:-2] + (4, xyz.shape[-2]))
    q[..., 0, :] = np.cos(x) * np.cos(y) * np.cos(z) * np.cos(w * t)
    f = np.sin(w * t) / np.sqrt(3.0)
    q[..., 1, :] = np.sin(x) * np.cos(y) * np.cos(z) * f
    q[..., 2, :] = np.cos(x) * np.sin(y) * np.cos(z) * f
    q[..., 3, :] = np.cos(x) * np.cos(y) * np.sin(z) * f
    return q


def gaussian_pulse(xyz: np.ndarray, model: int, width: float = 0.05) -> np.ndarray:
    """exp(-|x-xc|^2/(2 width^2)) at the cube centre: acoustic p; elastic
    sxx = syy = szz = -pulse (explosive source), everything else 0."""
    r2 = np.sum((xyz - 0.5) ** 2, axis=-1)
    g = np.exp(-r2 / (2 * width * width))
    q = np.zeros(xyz.shape[:-2] + (NFIELDS[model], xyz.shape[-2]))
    if model == ACOUSTIC:
        q[..., 0, :] = g
    else:
        for a in (3, 4, 5):
            q[..., a, :] = -g
    return q


def random_fields(K: int, model: int, Np: int, seed: int = 3) -> np.ndarray:
    """i.i.d. N(0,1) nodal values (a nodal vector is a degree-N polynomial)."""
    return normal(seed, K * NFIELDS[model] * Np).reshape(K, NFIELDS[model], Np)


# --------------------------------------------------------------------------
# BASELINE.json configs
# --------------------------------------------------------------------------
SWEEP_CELLS = {1: 101, 2: 75, 3: 59, 4: 49, 5: 42, 6: 37, 7: 33, 8: 29, 9: 27, 10: 24}


# the paper's own problem size (N = 1..8, "approximately 2 M nodes" per mesh): cells per side so that
# K Np is closest to 2.0e6
PAPER_CELLS = {1: 44, 2: 32, 3: 26, 4: 21, 5: 18, 6: 16, 7: 14, 8: 13}


@dataclass
class Workload:
    name: str
    model: int
    N: int
    n: int                       # cells per side
    jitter: float = 0.05
    materials: str = "unit"      # unit | random | layers | random_c5
    ic: str = "mode"             # mode | pulse | random
    top: int = BC_RIGID
    nsteps: int = 100
    seeds: dict = field(default_factory=lambda: {"mesh": 1, "materials": 2, "fields": 3})

    @property
    def K(self) -> int:
        return 6 * self.n ** 3

    @property
    def Np(self) -> int:
        return (self.N + 1) * (self.N + 2) * (self.N + 3) // 6

    def mesh(self):
        vxyz, etov, cell = kuhn_cube(self.n, self.jitter, self.seeds["mesh"])
        bc = wall_tags(self.n, etov, top=self.top)
        return vxyz, etov, bc, cell

    def material_arrays(self, cell=None):
        """(rho, c) for acoustic, (rho, vp, vs) for elastic."""
        K, s = self.K, self.seeds["materials"]
        if self.materials == "unit":
            one = np.ones(K)
            return (one, one.copy()) if self.model == ACOUSTIC else (one, 2 * one, one.copy())
        if self.materials == "random":
            return random_acoustic_materials(K, s) if self.model == ACOUSTIC else random_elastic_materials(K, s)
        if self.materials == "random_c5":
            return random_elastic_materials(K, s, rho_rng=(1.5, 3.0), vp_rng=(2.0, 6.0))
        if self.materials == "layers":
            if cell is None:
                cell = np.repeat(np.arange(self.n ** 3), 6)
            return layered_elastic_materials(self.n, cell)
        raise ValueError(self.materials)

    def initial_fields(self, xyz: np.ndarray) -> np.ndarray:
        """fp64 K x Nf x Np from node coordinates xyz (K x Np x 3)."""
        if self.ic == "mode":
            return standing_mode(xyz, 0.0)
        if self.ic == "pulse":
            return gaussian_pulse(xyz, self.model)
        if self.ic == "random":
            return random_fields(self.K, self.model, self.Np, self.seeds["fields"])
        raise ValueError(self.ic)


def config(i: int, N: int | None = None, model: int | None = None, n: int | None = None) -> Workload:
    """BASELINE.json configs, 1-based like SURVEY.md (C1..C5).  C4 takes N and model.
    `n` overrides the cube size (reduced-size parity cases)."""
    if i == 1:
        w = Workload("C1-acoustic-N3-mode", ACOUSTIC, 3, 4, nsteps=100)
    elif i == 2:
        w = Workload("C2-acoustic-N5-pulse", ACOUSTIC, 5, 40, materials="random", ic="pulse", nsteps=50)
    elif i == 3:
        w = Workload("C3-elastic-N7-layers", ELASTIC, 7, 30, materials="layers", ic="pulse", top=BC_FREE, nsteps=50)
    elif i == 4:
        if N is None or model is None:
            raise ValueError("config 4 needs N and model")
        w = Workload(f"C4-sweep-{'acoustic' if model == ACOUSTIC else 'elastic'}-N{N}", model, N,
                     SWEEP_CELLS[N], materials="random", ic="pulse", nsteps=20)
    elif i == 5:
        w = Workload("C5-elastic-N10-random", ELASTIC, 10, 24, jitter=0.10, materials="random_c5",
                     ic="random", top=BC_FREE, nsteps=20)
    elif i == 6:                      # not a BASELINE.json config: the paper's size, materials / IC as config 4
        if N is None or model is None or N not in PAPER_CELLS:
            raise ValueError("the paper-sized workload needs N in 1..8 and model")
        w = Workload(f"P-paper-sized-{'acoustic' if model == ACOUSTIC else 'elastic'}-N{N}", model, N,
                     PAPER_CELLS[N], materials="random", ic="pulse", nsteps=20)
    else:
        raise ValueError("config index 1..6")
    if n is not None:
        w.n = n
        w.name += f"-n{n}"
    return w
