"""Tile-phase timeline of the fused pair kernel (diagnostic; needs a library built with -DSIE_EXP_TRACE=1).

    SIE_NVCC_EXTRA="-DSIE_EXP_TRACE=1" python -m paper_2412_18553_b200.build --force
    python -m paper_2412_18553_b200.trace_phases config1          # or  o,v,naux   e.g. 120,216,1200
    python -m paper_2412_18553_b200.build --force                  # back to the product build

Every warp of CTA 3 stamps clock64 at five points of its first 8 tiles: A mainloop start, B mainloop end, C after the
barrier that frees the X tile, D after the X store + barrier, E end of its epilogue strip.  Printed per tile, in SM
cycles relative to the first warp's A: min/max over the 16 warps, and the period to the next tile's first A.
"""
import ctypes
import sys

import numpy as np
import torch

from workloads import ClusterSpec, config_specs, make_cluster

from . import ClusterSolver
from .binding import LIB_PATH


def main(name: str) -> None:
    if name.startswith("config"):
        spec = config_specs(int(name[6:]))[0]
    else:
        o, v, naux = (int(x) for x in name.split(","))
        spec = ClusterSpec(9, 0, o + v, o, v, naux, max(1, o // 2))
    lib = ctypes.CDLL(LIB_PATH)
    if not hasattr(lib, "sie_debug_trace"):
        raise SystemExit("libsie_dfmp2.so was not built with -DSIE_EXP_TRACE=1")
    x = make_cluster(spec)
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()  # noqa: E731
    s = ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux)
    s.transform(cu(x.C_occ), cu(x.C_vir), cu(x.L_packed(threads=8)), 0, spec.naux)
    for _ in range(2):  # second run: warm L2, warm instruction cache
        s.energy(cu(x.e_occ), cu(x.e_vir), cu(x.P_frag))
        torch.cuda.synchronize()
    buf = (ctypes.c_longlong * (8 * 16 * 5))()
    if lib.sie_debug_trace(buf) != 0:
        raise SystemExit("cudaMemcpyFromSymbol failed")
    t = np.array(buf[:]).reshape(8, 16, 5)
    print(f"{name}: o={spec.nocc} v={spec.nvir} naux={spec.naux}; cycles relative to the tile's first A")
    for tt in range(1, 7):
        r = t[tt] - t[tt, :, 0].min()
        print(f"tile {tt}: A {r[:, 0].min()}..{r[:, 0].max()}  B {r[:, 1].min()}..{r[:, 1].max()}  C {r[:, 2].max()}  "
              f"D {r[:, 3].max()}  E {r[:, 4].min()}..{r[:, 4].max()}  period {t[tt + 1, :, 0].min() - t[tt, :, 0].min()}")


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else "config1")
