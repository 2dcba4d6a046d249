"""TEST INFRASTRUCTURE: bytes the sweep REQUESTS from global memory per cell-update -- TMA boxes (halo lanes and rows
included), the z-geometry bulk copies, the cp.async of q, the streaming stores -- counted by the emulated build on the
tile / chunk decomposition the library picks for a grid (EMU_SM_COUNT = 148).  What DRAM actually moves (ncu,
profiles/r2_traffic.txt) lies between the algorithmic bytes and this figure: the difference to it is what L2 absorbs of the
halo re-reads.

    python tests/emu/traffic_report.py [config scale zscale steps] ...      e.g.  4 4 1 2   (config 4 at 256 x 256 x 192)
"""
import ctypes as C
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
sys.path.insert(0, HERE)

import workloads as W                      # noqa: E402
import emu_em                              # noqa: E402


def report(config, scale, zscale, steps, precision=32, thermal=False, **kw):
    p = W.make_config(config, scale=scale, steps=steps, **({"zscale": zscale} if zscale != 1 else {}))
    if thermal:
        p.thermal = W.thermal_table(p.table.shape[0])
    g = emu_em.EmuEM(p, precision=precision, **kw)
    out = (C.c_longlong * 4)()
    g._L.emu_traffic(out)                  # clear what the set-up moved
    g.em_step(steps)
    g._L.emu_traffic(out)
    cells = p.nx * p.ny * p.nz * steps
    tma, bulk, cpa, st = (out[q] / cells for q in range(4))
    print("config %d %dx%dx%d fp%d %s: TMA %.2f + bulk %.3f + cp.async %.2f = %.2f B read, %.2f B stored per cell-update; total %.2f B "
          "(algorithmic %d)" % (config, p.nx, p.ny, p.nz, precision, ("coupled " if thermal else "") + (kw.get("tag", "") or ""), tma, bulk, cpa, tma + bulk + cpa, st, tma + bulk + cpa + st,
                                57 if precision == 32 else 113))
    g.close()


if __name__ == "__main__":
    flags = [a for a in sys.argv[1:] if a.startswith("--")]
    args = [int(a) for a in sys.argv[1:] if not a.startswith("--")] or [4, 4, 1, 2]
    for q in range(0, len(args), 4):
        if "--thermal" in flags:          # the coupled sweep (k_diffuse's plain loads and stores are not counted) and the fused one
            import build_emu
            report(*args[q:q + 4], thermal=True)
            report(*args[q:q + 4], thermal=True, tag="fc", defines=build_emu.VARIANTS["fc"])
        else:
            report(*args[q:q + 4])
