"""Role timeline of the tensor-core stage kernel (development tool).

    DG_PROF=1 python -m paper_1602_07997_b200.build --force     # instrumented build (clock64 around every mbarrier wait)
    python -m paper_1602_07997_b200.role_timeline 2 3 5 4:3:acoustic
    python -m paper_1602_07997_b200.build --force                # back to the product build

For every workload (a BASELINE config number, or 4:N:model for a degree of the config-4 sweep) it runs two LSRK steps
and prints, per warp role of `tc3_stage_kernel`, the share of the last launch's cycles spent in each kind of wait and
the remainder ("busy").  The counters exist only in a -DDG_PROF build (`dg_prof_read`); timings of such a build are not
bench numbers.
"""
from __future__ import annotations

import ctypes as C
import sys

import numpy as np


def main(argv):
    import torch
    from . import dg, workloads as W
    if not hasattr(dg._lib, "dg_prof_read"):
        raise SystemExit("libdg.so was not built with DG_PROF=1")
    dg._lib.dg_prof_read.argtypes = [C.c_void_p, C.c_void_p]
    nwarps = 23                                       # tc3_kernels.cuh: 4 epilogue, 8 producers, 8 flux, 3 single-warp roles
    roles = [("epilogue", range(0, 4), ["accFull", "chunk loads", "tmem ld"]),
             ("producer", range(4, 12), ["emptyA", "tile / field chunk", "flFull"]),
             ("flux", range(12, 20), ["tile", "flEmpty"]),
             ("operator stream", [20], ["emptyB"]),
             ("mma", [21], ["accEmpty", "fullA", "fullB"]),
             ("loader", [22], ["slot empty", "chunk ring"])]
    for spec in argv:
        parts = spec.split(":")
        if parts[0] == "4":
            w = W.config(4, N=int(parts[1]), model=W.ELASTIC if parts[2].startswith("e") else W.ACOUSTIC)
        else:
            w = W.config(int(parts[0]))
        ctx = dg.from_workload(w, variant=4)
        q = torch.from_numpy(w.initial_fields(ctx.node_coords()).astype(np.float32)).cuda()
        ctx.run(q.data_ptr(), float(np.float32(ctx.stable_dt(0.5))), 2)
        torch.cuda.synchronize()
        buf = np.zeros((296, nwarps, 5), dtype=np.int64)
        if dg._lib.dg_prof_read(ctx._h, buf.ctypes.data_as(C.c_void_p)) != 0:
            raise SystemExit("dg_prof_read failed")
        b = buf[:148].astype(np.float64)
        b = b[b[:, 0, 0] > 0]                          # CTAs that ran
        tot = b[:, :, 0].mean()
        print(f"{w.name}: {ctx.variant_name}")
        print(f"  mean cycles per CTA {tot:.0f}")
        for name, ws, ids in roles:
            sub = b[:, list(ws), :]
            line = f"  {name:16s}"
            for i, nm in enumerate(ids):
                line += f"  wait {nm} {100 * sub[:, :, 1 + i].mean() / tot:5.1f} %"
            line += f"  busy {100 * (1 - sub[:, :, 1:].sum(axis=2).mean() / tot):5.1f} %"
            print(line)
        ctx.close()


if __name__ == "__main__":
    main(sys.argv[1:] or ["2"])
