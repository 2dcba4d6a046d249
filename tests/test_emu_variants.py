"""The compile-time experiment switches of the sweep (profiles/r2_experiments.md) on the emulated build (tests/emu): other
tile heights, 2 CTAs per SM, the L2 prefetch of later planes, other launch orders.  A scratch build of the 5-row / 2-CTA
variant once FAULTED on a B200 with "misaligned address" (one of the events after which GPU use was closed for this
repository); the emulation reproduces that fault on the host -- the material table of that layout sat at 8 mod 16 -- and
SweepLayout now rounds the offset and static_asserts the alignment of every region for every tile shape (the default build's
SASS is unchanged).  Slow (one build per variant): runs with EM_RUN_SLOW=1; outcome in profiles/r2_emulation.md."""
import os
import sys

import pytest

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "emu"))

import workloads as W
from oracle import emo
from parity import TOL, compare_state
import emu_em

VARIANTS = {
    "ty5-2ctas": ["-DEM_SWEEP_TY=5", "-DEM_SWEEP_OCC=2"],
    "ty10": ["-DEM_SWEEP_TY=10"],
    "ty12": ["-DEM_SWEEP_TY=12"],
    "ty64-8": ["-DEM_SWEEP_TY64=8"],
    "l2ahead2": ["-DEM_SWEEP_L2AHEAD=2", "-DEM_SWEEP_PFPOL=1"],
    "order-4x2": ["-DEM_SWEEP_ORDER_BY=4", "-DEM_SWEEP_ORDER_BX=2"],
    "order-tile-major": ["-DEM_SWEEP_ORDER_BY=0"],
}


@pytest.mark.slow
@pytest.mark.parametrize("name", sorted(VARIANTS))
def test_experiment_switch_variant(name, monkeypatch):
    monkeypatch.setenv("EMU_SEED", "2")
    p = W.random_problem(130, 31, 13, seed=5, steps=4, n_ports=4, bc=(0, 1, 1, 0, 1, 0), init_scale=4.0e6)
    for thermal in (False, True):
        if thermal:
            th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
            p.thermal = th
        for precision in (32, 64):
            g = emu_em.EmuEM(p, precision=precision, z_chunks=3, tag="var_" + name.replace("-", "_"), defines=VARIANTS[name])
            o = emo.Oracle(p)
            g.em_step(4); o.step(4)
            compare_state(g, o, TOL[precision])
            g.close(); o.close()
