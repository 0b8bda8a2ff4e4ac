"""Thin ctypes binding over libdg.so (include/dg.h).  Argument marshalling only: every step of the
hot path runs in the library's CUDA kernels.  PyTorch appears only in the caller, for device
memory and streams; device buffers are passed here as raw pointers (``tensor.data_ptr()``).

If libdg.so is missing the import of this module raises -- there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

ACOUSTIC, ELASTIC = 0, 1
BC_INTERIOR, BC_RIGID, BC_FREE, BC_SLIP = 0, 1, 2, 3
STATIC_SCRATCH_BYTES = 32 * 1024 * 1024      # include/dg.h: DG_STATIC_SCRATCH_BYTES (work memory of dg_step_static)

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libdg.so")
if not os.path.exists(_LIB_PATH):
    raise ImportError(f"{_LIB_PATH} not found: build it with `python -m paper_1602_07997_b200.build` "
                      "(the product path has no CPU fallback)")
_lib = C.CDLL(_LIB_PATH)


class _Mesh(C.Structure):
    _fields_ = [("nverts", C.c_int64), ("K", C.c_int64), ("vxyz", C.c_void_p), ("etov", C.c_void_p), ("bc", C.c_void_p)]


class _Materials(C.Structure):
    _fields_ = [("rho", C.c_void_p), ("c_or_vp", C.c_void_p), ("vs", C.c_void_p)]


class _Options(C.Structure):
    _fields_ = [("device", C.c_int), ("variant", C.c_int), ("elems_per_thread", C.c_int), ("groups_per_cta", C.c_int),
                ("max_ctas", C.c_int), ("surface", C.c_int), ("owned_elements", C.c_int64)]


EXPORTS = ["dg_create", "dg_destroy", "dg_num_fields", "dg_np", "dg_nfp", "dg_num_elements", "dg_node_coords",
           "dg_stable_dt", "dg_rhs", "dg_step", "dg_step_static", "dg_run", "dg_stage", "dg_stage_range", "dg_range_alignment", "dg_element_dt", "dg_ab3_step", "dg_ab3_run", "dg_ab3_reset", "dg_last_launch_count",
           "dg_variant_name", "dg_reference_operators", "dg_geometry", "dg_connectivity", "dg_last_error",
           "dg_partition_create", "dg_partition_destroy", "dg_partition_num_owned", "dg_partition_num_ghost",
           "dg_partition_global_ids", "dg_partition_local_mesh", "dg_partition_num_peers", "dg_partition_peer",
           "dg_partition_halo_faces", "dg_halo_pack", "dg_halo_unpack", "dg_num_owned_elements"]

_lib.dg_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(_Mesh), C.c_int, C.c_int, C.POINTER(_Materials), C.POINTER(_Options)]
_lib.dg_create.restype = C.c_int
_lib.dg_destroy.argtypes = [C.c_void_p]
for _n in ("dg_num_fields", "dg_np", "dg_nfp", "dg_last_launch_count"):
    getattr(_lib, _n).argtypes = [C.c_void_p]
    getattr(_lib, _n).restype = C.c_int
_lib.dg_num_elements.argtypes = [C.c_void_p]
_lib.dg_num_elements.restype = C.c_int64
_lib.dg_node_coords.argtypes = [C.c_void_p, C.c_void_p]
_lib.dg_stable_dt.argtypes = [C.c_void_p, C.c_double]
_lib.dg_stable_dt.restype = C.c_double
_lib.dg_rhs.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.dg_step.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_void_p]
_lib.dg_step_static.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_void_p]
_lib.dg_run.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_int, C.c_void_p]
_lib.dg_stage.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_void_p]
_lib.dg_stage_range.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_int64, C.c_int64, C.c_void_p]
_lib.dg_range_alignment.argtypes = [C.c_void_p]
_lib.dg_element_dt.argtypes = [C.c_void_p, C.c_double, C.c_void_p]
_lib.dg_ab3_step.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_void_p]
_lib.dg_ab3_run.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_int, C.c_void_p]
_lib.dg_ab3_reset.argtypes = [C.c_void_p, C.c_void_p]
_lib.dg_variant_name.argtypes = [C.c_void_p]
_lib.dg_variant_name.restype = C.c_char_p
_lib.dg_reference_operators.argtypes = [C.c_void_p] + [C.c_void_p] * 6
_lib.dg_geometry.argtypes = [C.c_void_p] + [C.c_void_p] * 4
_lib.dg_connectivity.argtypes = [C.c_void_p] + [C.c_void_p] * 3
_lib.dg_last_error.restype = C.c_char_p
_lib.dg_partition_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(_Mesh), C.c_int, C.c_int]
_lib.dg_partition_destroy.argtypes = [C.c_void_p]
for _n in ("dg_partition_num_owned", "dg_partition_num_ghost", "dg_num_owned_elements"):
    getattr(_lib, _n).argtypes = [C.c_void_p]
    getattr(_lib, _n).restype = C.c_int64
_lib.dg_partition_global_ids.argtypes = [C.c_void_p, C.c_void_p]
_lib.dg_partition_local_mesh.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.dg_partition_num_peers.argtypes = [C.c_void_p]
_lib.dg_partition_peer.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
_lib.dg_partition_halo_faces.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
_lib.dg_halo_pack.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
_lib.dg_halo_unpack.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]


class DGError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libdg error {code}: {msg}")
        self.code = code


def last_error() -> str:
    return _lib.dg_last_error().decode()


def _check(code: int) -> None:
    if code != 0:
        raise DGError(code, last_error())


def _ptr(a: np.ndarray | None):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Context:
    """dg_create / dg_destroy pair.  Host arrays are numpy; device buffers are raw pointers (ints)."""

    def __init__(self, vxyz, etov, N: int, model: int, rho, c_or_vp, vs=None, bc=None, device: int = 0,
                 elems_per_thread: int = 0, groups_per_cta: int = 0, variant: int = 0, max_ctas: int = 0, surface: int = 0, owned_elements: int = 0):
        vxyz = np.ascontiguousarray(vxyz, dtype=np.float64)
        etov = np.ascontiguousarray(etov, dtype=np.int32)
        bc = None if bc is None else np.ascontiguousarray(bc, dtype=np.int8)
        rho = np.ascontiguousarray(rho, dtype=np.float64)
        c_or_vp = np.ascontiguousarray(c_or_vp, dtype=np.float64)
        vs = None if vs is None else np.ascontiguousarray(vs, dtype=np.float64)
        mesh = _Mesh(vxyz.shape[0], etov.shape[0], _ptr(vxyz), _ptr(etov), _ptr(bc))
        mat = _Materials(_ptr(rho), _ptr(c_or_vp), _ptr(vs))
        opt = _Options(device, variant, elems_per_thread, groups_per_cta, max_ctas, surface, owned_elements)
        h = C.c_void_p()
        self._h = None
        _check(_lib.dg_create(C.byref(h), C.byref(mesh), int(N), int(model), C.byref(mat), C.byref(opt)))
        self._h = h
        self.N, self.model, self.device = int(N), int(model), device
        self.K = int(_lib.dg_num_elements(h))
        self.K_owned = int(_lib.dg_num_owned_elements(h))
        self.Np, self.Nfp, self.NF = int(_lib.dg_np(h)), int(_lib.dg_nfp(h)), int(_lib.dg_num_fields(h))

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) and _lib is not None:      # _lib is None while the interpreter shuts down
            _lib.dg_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- host queries
    @property
    def shape(self):
        return (self.K, self.NF, self.Np)

    @property
    def variant_name(self) -> str:
        return _lib.dg_variant_name(self._h).decode()

    @property
    def last_launch_count(self) -> int:
        return int(_lib.dg_last_launch_count(self._h))

    def node_coords(self) -> np.ndarray:
        xyz = np.empty((self.K, self.Np, 3), dtype=np.float64)
        _check(_lib.dg_node_coords(self._h, _ptr(xyz)))
        return xyz

    def stable_dt(self, cfl: float = 0.5) -> float:
        dt = float(_lib.dg_stable_dt(self._h, float(cfl)))
        if dt < 0:
            raise DGError(int(dt), last_error())
        return dt

    def reference_operators(self):
        Np, Nfp = self.Np, self.Nfp
        Dr, Ds, Dt = (np.empty((Np, Np)) for _ in range(3))
        LIFT = np.empty((Np, 4 * Nfp))
        rst = np.empty((Np, 3))
        fmask = np.empty((4, Nfp), dtype=np.int32)
        _check(_lib.dg_reference_operators(self._h, _ptr(Dr), _ptr(Ds), _ptr(Dt), _ptr(LIFT), _ptr(rst), _ptr(fmask)))
        return dict(Dr=Dr, Ds=Ds, Dt=Dt, LIFT=LIFT, rst=rst, fmask=fmask)

    def geometry(self):
        K = self.K
        G, J, nrm, fs = np.empty((K, 3, 3)), np.empty(K), np.empty((K, 4, 3)), np.empty((K, 4))
        _check(_lib.dg_geometry(self._h, _ptr(G), _ptr(J), _ptr(nrm), _ptr(fs)))
        return dict(G=G, J=J, nrm=nrm, fscale=fs)

    def connectivity(self):
        K, Nfp = self.K, self.Nfp
        eP = np.empty((K, 4 * Nfp), dtype=np.int32)
        nP = np.empty((K, 4 * Nfp), dtype=np.int32)
        tag = np.empty((K, 4), dtype=np.int8)
        _check(_lib.dg_connectivity(self._h, _ptr(eP), _ptr(nP), _ptr(tag)))
        return dict(elemP=eP, nodeP=nP, bctag=tag)

    # -- device entry points (raw device pointers, cudaStream_t as int or None)
    def rhs(self, d_q: int, d_rhs: int, stream: int | None = None):
        _check(_lib.dg_rhs(self._h, C.c_void_p(d_q), C.c_void_p(d_rhs), C.c_void_p(stream or 0)))

    def step(self, d_q: int, dt: float, stream: int | None = None):
        _check(_lib.dg_step(self._h, C.c_void_p(d_q), C.c_float(dt), C.c_void_p(stream or 0)))

    def step_static(self, d_q: int, dt: float, stream: int | None = None):
        """dg_step_static: the same step with its work memory in the library's static device array (no allocation;
        limit STATIC_SCRATCH_BYTES; calls that overlap on the GPU race on the array: include/dg.h)."""
        _check(_lib.dg_step_static(self._h, C.c_void_p(d_q), C.c_float(dt), C.c_void_p(stream or 0)))

    def run(self, d_q: int, dt: float, nsteps: int, stream: int | None = None):
        _check(_lib.dg_run(self._h, C.c_void_p(d_q), C.c_float(dt), int(nsteps), C.c_void_p(stream or 0)))

    def stage(self, d_q_in: int, d_q_out: int, a: float, b: float, dt: float, stream: int | None = None):
        _check(_lib.dg_stage(self._h, C.c_void_p(d_q_in), C.c_void_p(d_q_out), C.c_float(a), C.c_float(b), C.c_float(dt),
                             C.c_void_p(stream or 0)))

    def stage_range(self, d_q_in: int, d_q_out: int, a: float, b: float, dt: float, k_begin: int, k_end: int,
                    stream: int | None = None):
        _check(_lib.dg_stage_range(self._h, C.c_void_p(d_q_in), C.c_void_p(d_q_out), C.c_float(a), C.c_float(b), C.c_float(dt),
                                   int(k_begin), int(k_end), C.c_void_p(stream or 0)))

    @property
    def range_alignment(self) -> int:
        return int(_lib.dg_range_alignment(self._h))

    def element_dt(self, cfl: float = 0.5) -> np.ndarray:
        out = np.empty(self.K, dtype=np.float64)
        _check(_lib.dg_element_dt(self._h, float(cfl), _ptr(out)))
        return out

    def halo_pack(self, d_q: int, d_faces: int, nfaces: int, d_buf: int, stream: int | None = None):
        _check(_lib.dg_halo_pack(self._h, C.c_void_p(d_q), C.c_void_p(d_faces), int(nfaces), C.c_void_p(d_buf), C.c_void_p(stream or 0)))

    def halo_unpack(self, d_q: int, d_faces: int, nfaces: int, d_buf: int, stream: int | None = None):
        _check(_lib.dg_halo_unpack(self._h, C.c_void_p(d_q), C.c_void_p(d_faces), int(nfaces), C.c_void_p(d_buf), C.c_void_p(stream or 0)))

    def ab3_step(self, d_q: int, dt: float, stream: int | None = None):
        _check(_lib.dg_ab3_step(self._h, C.c_void_p(d_q), C.c_float(dt), C.c_void_p(stream or 0)))

    def ab3_run(self, d_q: int, dt: float, nsteps: int, stream: int | None = None):
        _check(_lib.dg_ab3_run(self._h, C.c_void_p(d_q), C.c_float(dt), int(nsteps), C.c_void_p(stream or 0)))

    def ab3_reset(self, stream: int | None = None):
        _check(_lib.dg_ab3_reset(self._h, C.c_void_p(stream or 0)))


class Partition:
    """dg_partition_*: one rank's slab of the element list, its ghost elements and the halo face lists per peer."""

    def __init__(self, vxyz, etov, bc, nranks: int, rank: int):
        vxyz = np.ascontiguousarray(vxyz, dtype=np.float64)
        etov = np.ascontiguousarray(etov, dtype=np.int32)
        bc = None if bc is None else np.ascontiguousarray(bc, dtype=np.int8)
        mesh = _Mesh(vxyz.shape[0], etov.shape[0], _ptr(vxyz), _ptr(etov), _ptr(bc))
        h = C.c_void_p()
        self._h = None
        _check(_lib.dg_partition_create(C.byref(h), C.byref(mesh), int(nranks), int(rank)))
        self._h = h
        self.nranks, self.rank = int(nranks), int(rank)
        self.num_owned = int(_lib.dg_partition_num_owned(h))
        self.num_ghost = int(_lib.dg_partition_num_ghost(h))
        n = self.num_owned + self.num_ghost
        self.global_ids = np.empty(n, dtype=np.int64)
        _check(_lib.dg_partition_global_ids(h, _ptr(self.global_ids)))
        self.etov = np.empty((n, 4), dtype=np.int32)
        self.bc = np.empty((n, 4), dtype=np.int8)
        _check(_lib.dg_partition_local_mesh(h, _ptr(self.etov), _ptr(self.bc)))
        self.peers = []                      # (peer rank, send faces, recv faces): 4 * local element + face
        for i in range(int(_lib.dg_partition_num_peers(h))):
            r, ns, nr = C.c_int(), C.c_int64(), C.c_int64()
            _check(_lib.dg_partition_peer(h, i, C.byref(r), C.byref(ns), C.byref(nr)))
            send, recv = np.empty(ns.value, dtype=np.int32), np.empty(nr.value, dtype=np.int32)
            _check(_lib.dg_partition_halo_faces(h, i, _ptr(send), _ptr(recv)))
            self.peers.append((r.value, send, recv))

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.dg_partition_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()


def from_workload(w, device: int = 0, **opts) -> Context:
    """Context for a workloads.Workload (mesh, materials and boundary tags from its seeds)."""
    vxyz, etov, bc, cell = w.mesh()
    mats = w.material_arrays(cell)
    if w.model == ACOUSTIC:
        return Context(vxyz, etov, w.N, w.model, mats[0], mats[1], None, bc, device=device, **opts)
    return Context(vxyz, etov, w.N, w.model, mats[0], mats[1], mats[2], bc, device=device, **opts)
