"""Shared helpers of the GPU parity tests: build the CUDA context and the oracle on the same seeded
workload, feed both the same fp32-rounded fields, compare element by element."""
import numpy as np

from oracle import mesh as omesh
from oracle import physics, refelem, timestep
from paper_1602_07997_b200 import workloads as W

RHS_TOL = 2e-6       # BASELINE.json north_star: rel-L2 per RHS evaluation
RUN_TOL = 1e-4       # after the configured number of LSRK steps

_REF = {}


def ref_of(N):
    if N not in _REF:
        _REF[N] = refelem.build(N)
    return _REF[N]


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def describe(got, want):
    """rel-L2 plus where the worst entry is: "rel-L2 3.1e-07, max |err| 2.4e-06 at (element, field, node) = (17, 2, 5)
    (got ..., want ...), worst element 17 (rel-L2 1.2e-06)" -- so that a failing parity assertion localises the defect."""
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    d = np.abs(got - want)
    idx = np.unravel_index(int(np.argmax(d)), d.shape)
    per_elem = np.sqrt((d.reshape(d.shape[0], -1) ** 2).sum(axis=1))
    k = int(np.argmax(per_elem))
    scale = max(float(np.linalg.norm(want.ravel())), 1e-300)
    return (f"rel-L2 {rel_l2(got, want):.3e}, max |err| {d[idx]:.3e} at (element, field, node) = {tuple(int(i) for i in idx)} "
            f"(got {got[idx]:.9g}, want {want[idx]:.9g}), worst element {k} carries {per_elem[k] / scale:.3e} of the rel-L2")


def assert_close(got, want, tol, what=""):
    assert np.isfinite(np.asarray(got)).all(), f"{what}: non-finite values in the GPU result"
    err = rel_l2(got, want)
    assert err <= tol, f"{what}: {describe(got, want)} > tolerance {tol:g}"
    return err


class Case:
    """One workload on both sides.  `only_elems` limits the oracle's connectivity to sampled elements."""

    def __init__(self, dg, w, only_elems=None, **ctx_opts):
        self.w = w
        self.vxyz, self.etov, self.bc, self.cell = w.mesh()
        self.mats = w.material_arrays(self.cell)
        vs = self.mats[2] if w.model == W.ELASTIC else None
        self.ctx = dg.Context(self.vxyz, self.etov, w.N, w.model, self.mats[0], self.mats[1], vs, self.bc, device=0, **ctx_opts)
        self.ref = ref_of(w.N)
        self.mesh = omesh.build(self.ref, self.vxyz, self.etov, self.bc, only_elems=only_elems)

    def oracle_rhs(self, q, elems=None):
        if self.w.model == W.ACOUSTIC:
            return physics.rhs_acoustic(self.ref, self.mesh, self.mats[0], self.mats[1], q, elems)
        return physics.rhs_elastic(self.ref, self.mesh, *self.mats, q, elems)

    def oracle_run(self, q0, dt, nsteps):
        return timestep.lsrk_run(q0, dt, nsteps, self.oracle_rhs)

    def initial_fields32(self):
        return self.w.initial_fields(self.mesh.x).astype(np.float32)

    def dt32(self, cfl=0.5):
        return float(np.float32(self.ctx.stable_dt(cfl)))

    def gpu_rhs(self, torch, q32):
        d_q = torch.from_numpy(np.ascontiguousarray(q32)).cuda()
        d_r = torch.full_like(d_q, float("nan"))
        self.ctx.rhs(d_q.data_ptr(), d_r.data_ptr(), torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        return d_r.cpu().numpy()

    def gpu_stage(self, torch, q32, a, b, dt, d_in=None):
        """One low-storage stage through dg_stage: returns (q_out as numpy, the device tensor of q_out)."""
        d_q = torch.from_numpy(np.ascontiguousarray(q32)).cuda() if d_in is None else d_in
        d_o = torch.full_like(d_q, float("nan"))
        self.ctx.stage(d_q.data_ptr(), d_o.data_ptr(), a, b, dt, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        return d_o.cpu().numpy(), d_o

    def gpu_run(self, torch, q32, dt, nsteps):
        d_q = torch.from_numpy(np.ascontiguousarray(q32)).cuda()
        self.ctx.run(d_q.data_ptr(), dt, nsteps, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        return d_q.cpu().numpy()
