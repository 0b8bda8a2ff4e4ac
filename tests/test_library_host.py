"""CPU-only tests of libdg: the library loads, exports every symbol include/dg.h declares, and its
host setup (its own C++ implementation of the reference operators, geometry and connectivity)
agrees with the oracle's independent numpy implementation.  No device entry point is called:
contexts are host-only (device = -1), on which dg_rhs & co. must refuse to run."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import mesh as omesh
from oracle import timestep
from paper_1602_07997_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def dg():
    from paper_1602_07997_b200 import build
    build.build()
    from paper_1602_07997_b200 import dg as mod
    return mod


def test_library_exports_every_declared_symbol(dg):
    hdr = open(os.path.join(ROOT, "include", "dg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(dg_[a-z0-9_]+)\s*\(", hdr))
    assert declared, "no declarations found"
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_1602_07997_b200", "libdg.so"))
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in include/dg.h but not exported"
    assert declared == set(dg.EXPORTS)


def test_no_cpu_fallback_on_host_only_context(dg):
    w = W.config(1, n=1)
    ctx = dg.from_workload(w, device=-1)
    for call in (lambda: ctx.rhs(16, 32), lambda: ctx.step(16, 1e-3), lambda: ctx.run(16, 1e-3, 2),
                 lambda: ctx.ab3_step(16, 1e-3)):
        with pytest.raises(dg.DGError) as ei:
            call()
        assert ei.value.code == -4 and "no CPU fallback" in str(ei.value)


@pytest.mark.parametrize("N", range(1, 11))
def test_reference_operators_match_oracle(dg, refelems, N):
    w = W.config(1, n=1)
    w.N = N
    ctx = dg.from_workload(w, device=-1)
    ops = ctx.reference_operators()
    ref = refelems(N)
    assert ctx.Np == ref.Np and ctx.Nfp == ref.Nfp
    assert np.abs(ops["rst"] - np.stack([ref.r, ref.s, ref.t], axis=1)).max() < 1e-12
    assert np.array_equal(ops["fmask"], ref.Fmask)
    scale = np.abs(ref.Dr).max()
    for a, b in ((ops["Dr"], ref.Dr), (ops["Ds"], ref.Ds), (ops["Dt"], ref.Dt)):
        assert np.abs(a - b).max() < 1e-10 * scale
    assert np.abs(ops["LIFT"] - ref.LIFT).max() < 1e-10 * np.abs(ref.LIFT).max()


@pytest.mark.parametrize("N,n,jitter", [(1, 3, 0.05), (3, 4, 0.05), (4, 2, 0.1), (6, 2, 0.1)])
def test_geometry_connectivity_and_dt_match_oracle(dg, refelems, N, n, jitter):
    vxyz, etov, _ = W.kuhn_cube(n, jitter, seed=1)
    bc = W.wall_tags(n, etov, top=W.BC_FREE)
    K = etov.shape[0]
    rho, vp, vs = W.random_elastic_materials(K, seed=2)
    ctx = dg.Context(vxyz, etov, N, dg.ELASTIC, rho, vp, vs, bc, device=-1)
    ref = refelems(N)
    m = omesh.build(ref, vxyz, etov, bc)
    geo = ctx.geometry()
    assert np.abs(geo["G"] - m.G).max() < 1e-11 * np.abs(m.G).max()
    assert np.abs(geo["J"] - m.J).max() < 1e-13
    assert np.abs(geo["nrm"] - m.nrm).max() < 1e-12
    assert np.abs(geo["fscale"] - m.Fscale).max() < 1e-11 * m.Fscale.max()
    assert np.abs(ctx.node_coords() - m.x).max() < 1e-13
    con = ctx.connectivity()
    assert np.array_equal(con["elemP"], m.elemP)          # vertex-number matching == position matching
    assert np.array_equal(con["nodeP"], m.nodeP)
    assert np.array_equal(con["bctag"], m.bctag)
    assert abs(ctx.stable_dt(0.5) / timestep.stable_dt(ref, m, vp, 0.5) - 1) < 1e-12


def test_orientation_fix_and_any_vertex_order(dg, refelems):
    """Elements given with negative orientation or rotated vertex order still match the oracle."""
    vxyz, etov, _ = W.kuhn_cube(2, 0.05, seed=1)
    rng = np.random.default_rng(0)
    et = etov.copy()
    for k in range(et.shape[0]):
        et[k] = et[k][rng.permutation(4)]
    ctx = dg.Context(vxyz, et, 3, dg.ACOUSTIC, np.ones(len(et)), np.ones(len(et)), None, None, device=-1)
    ref = refelems(3)
    m = omesh.build(ref, vxyz, et, None)
    con = ctx.connectivity()
    assert np.all(ctx.geometry()["J"] > 0)
    assert np.abs(ctx.node_coords() - m.x).max() < 1e-13
    assert np.array_equal(con["elemP"], m.elemP) and np.array_equal(con["nodeP"], m.nodeP)


def test_bad_inputs_are_rejected(dg):
    vxyz, etov, _ = W.kuhn_cube(1, 0.0)
    one = np.ones(6)
    with pytest.raises(dg.DGError) as e:
        dg.Context(vxyz, etov, 11, dg.ACOUSTIC, one, one, device=-1)
    assert e.value.code == -1
    with pytest.raises(dg.DGError) as e:
        dg.Context(vxyz, etov, 2, 7, one, one, device=-1)
    assert e.value.code == -1
    with pytest.raises(dg.DGError) as e:
        dg.Context(vxyz, etov, 2, dg.ACOUSTIC, -one, one, device=-1)
    assert e.value.code == -3
    with pytest.raises(dg.DGError) as e:          # vp <= vs sqrt(4/3)
        dg.Context(vxyz, etov, 2, dg.ELASTIC, one, one, one, device=-1)
    assert e.value.code == -3
    with pytest.raises(dg.DGError) as e:          # a face with three owners
        dg.Context(vxyz, np.concatenate([etov, etov[:1]]), 2, dg.ACOUSTIC, np.ones(7), np.ones(7), device=-1)
    assert e.value.code == -2
    flat = vxyz.copy(); flat[:, 2] = 0.0
    with pytest.raises(dg.DGError) as e:          # degenerate elements
        dg.Context(flat, etov, 2, dg.ACOUSTIC, one, one, device=-1)
    assert e.value.code == -2
    with pytest.raises(dg.DGError) as e:          # boundary faces tagged "interior"
        dg.Context(vxyz, etov, 2, dg.ACOUSTIC, one, one, None, np.zeros((6, 4), np.int8), device=-1)
    assert e.value.code == -2


def test_boundary_tags_follow_the_callers_face_numbering(dg, refelems):
    """include/dg.h: `bc[k][f]` refers to face f of element k in the CALLER's vertex order, whatever the orientation; the
    library permutes the tags together with the vertices when it fixes a negative Jacobian.  Every element is given in a
    random vertex order (half of them negatively oriented) with distinct tags on the cube's top (FREE) and the other
    walls (RIGID); afterwards every tagged face must carry the tag of the wall its normal points to."""
    n = 2
    vxyz, etov, _ = W.kuhn_cube(n, 0.05, seed=1)
    bc = W.wall_tags(n, etov, top=W.BC_FREE, other=W.BC_RIGID)
    opp = np.array([3, 2, 0, 1])                     # face f is opposite the local vertex opp[f]
    face_of_opp = np.argsort(opp)                    # vertex v is opposite face face_of_opp[v]
    rng = np.random.default_rng(5)
    et, tags = etov.copy(), bc.copy()
    for k in range(len(et)):
        perm = rng.permutation(4)
        et[k] = etov[k][perm]
        tags[k] = bc[k][face_of_opp[perm[opp]]]      # new face f = old face opposite the old vertex perm[opp[f]]
    one = np.ones(len(et))
    ctx = dg.Context(vxyz, et, 2, dg.ACOUSTIC, one, one, None, tags, device=-1)
    geo, con = ctx.geometry(), ctx.connectivity()
    assert np.all(geo["J"] > 0)
    lib_tags, nrm = con["bctag"], geo["nrm"]
    assert (lib_tags > 0).sum() == (bc > 0).sum() == 6 * 2 * n * n
    top = (lib_tags > 0) & (nrm[..., 2] > 0.99)       # boundary faces whose outward normal is +z (walls are planar)
    assert np.all(lib_tags[top] == W.BC_FREE) and top.sum() == 2 * n * n
    wall = (lib_tags > 0) & ~top
    assert np.all(lib_tags[wall] == W.BC_RIGID)
    assert np.all(np.abs(np.abs(nrm[wall]).max(axis=-1) - 1.0) < 1e-12)       # axis-aligned outward wall normals
    # and the oracle, given the same permuted input, agrees tag for tag
    m = omesh.build(refelems(2), vxyz, et, tags)
    assert np.array_equal(lib_tags, m.bctag)
    # a caller who "pre-swaps" tags as the old header text suggested would put FREE on a side wall: the library must not
    wrong = tags.copy()
    wrong[:, [0, 1]] = wrong[:, [1, 0]]
    if not np.array_equal(wrong, tags):
        try:
            bad = dg.Context(vxyz, et, 2, dg.ACOUSTIC, one, one, None, wrong, device=-1)
            lt = bad.connectivity()["bctag"]
            assert not np.all(lt[(lt > 0) & (bad.geometry()["nrm"][..., 2] > 0.99)] == W.BC_FREE)
        except dg.DGError as e:                      # or the swap leaves a boundary face untagged: also a loud failure
            assert e.code == -2


def test_element_dt_levels_for_multirate(dg, refelems):
    """dg_element_dt (multi-rate hook): every element's own stable step by the rule of DESIGN.md Q10; the
    global step of dg_stable_dt is its minimum; on a mesh with one refined corner the steps spread over > 2 octaves,
    which is what a local time stepping driver bins into levels."""
    vxyz, etov, _ = W.kuhn_cube(3, 0.05, seed=1)
    vxyz = vxyz ** 2.5                                   # grade the mesh towards the origin (walls stay planar)
    K = etov.shape[0]
    rho, vp, vs = W.random_elastic_materials(K, seed=2)
    ctx = dg.Context(vxyz, etov, 4, dg.ELASTIC, rho, vp, vs, None, device=-1)
    m = omesh.build(refelems(4), vxyz, etov, None)
    want = 0.5 / (25.0 * vp * m.Fscale.max(axis=1))
    got = ctx.element_dt(0.5)
    assert np.abs(got / want - 1).max() < 1e-12
    assert abs(got.min() / ctx.stable_dt(0.5) - 1) < 1e-12
    levels = np.floor(np.log2(got / got.min())).astype(int)
    assert levels.max() >= 2 and (np.bincount(levels) > 0).sum() >= 3
    assert ctx.range_alignment in (1, 14, 32) or ctx.range_alignment > 0


def test_option_values_are_validated(dg):
    """dg_options: unknown variant / surface values, a negative max_ctas and owned_elements beyond K are DG_ERR_ARG."""
    vxyz, etov, _ = W.kuhn_cube(1, 0.0)
    one = np.ones(6)
    for bad in (dict(variant=3), dict(surface=2), dict(max_ctas=-1), dict(owned_elements=7)):
        with pytest.raises(dg.DGError) as e:
            dg.Context(vxyz, etov, 2, dg.ACOUSTIC, one, one, device=-1, **bad)
        assert e.value.code == -1, bad
    ok = dg.Context(vxyz, etov, 2, dg.ACOUSTIC, one, one, device=-1, owned_elements=4, surface=1, max_ctas=3)
    assert ok.K == 6 and ok.K_owned == 4
    for call in (lambda: ok.stage(16, 32, 0.0, 1.0, 1e-3), lambda: ok.stage_range(16, 32, 0.0, 1.0, 1e-3, 0, 4),
                 lambda: ok.ab3_run(16, 1e-3, 2), lambda: ok.halo_pack(16, 32, 1, 48), lambda: ok.halo_unpack(16, 32, 1, 48)):
        with pytest.raises(dg.DGError) as e:
            call()
        assert e.value.code == -4 and "no CPU fallback" in str(e.value)
