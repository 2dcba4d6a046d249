"""The small case run under compute-sanitizer (racecheck / synccheck / memcheck):

    compute-sanitizer --tool racecheck python tests/sanitizer_case.py

The sweep's plane loop has NO CTA barrier: row-to-row hand-offs go through per-row mbarriers and 64-thread named
barriers, staged slots are released on "empty" mbarriers (csrc/em_sweep.cuh).  The case covers 2 x 2 tiles (fp32; more in
fp64), 2 z chunks, a PMC wall at -z (the warm-up plane runs), ports on chunk-boundary planes, both loss modes'
instantiations in use by the configs (CD), the leapfrog, the E-only recurrence and the thermally coupled sweep, in fp32
and fp64, 3 steps each; every run is also compared with the oracle so that a sanitizer-clean run is a correct run."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT); sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np

import workloads as W
import paper_2603_07038_b200 as P
from oracle import emo
from parity import rel_l2


def main():
    steps = 3
    for precision in (32, 64):
        tol = 2e-5 if precision == 32 else 1e-11
        p = W.random_problem(130, 20, 11, seed=4242, steps=steps, n_ports=30, bc=(0, 1, 0, 0, 1, 0))
        # leapfrog
        g = P.EM(p, precision=precision, z_chunks=2); o = emo.Oracle(p)
        g.em_step(steps); o.step(steps)
        assert rel_l2(g.fields()[:3], o.fields()[:3]) <= tol
        g.close(); o.close()
        # E-only recurrence
        g = P.EM(p, precision=precision, z_chunks=2, formulation=P.EM_FORM_EONLY); o = emo.OracleEOnly(p)
        g.em_step(steps); o.step(steps)
        assert rel_l2(g.fields()[:3], o.fields(0)) <= tol
        g.close(); o.close()
        # thermally coupled sweep
        p.thermal = W.thermal_table(); p.thermal[:, 1] *= 2.0e5; p.thermal[:, 2] *= 1.0e4
        g = P.EM(p, precision=precision, z_chunks=2); o = emo.Oracle(p)
        g.em_step(steps); o.step(steps)
        assert rel_l2(g.fields()[:3], o.fields()[:3]) <= tol
        assert rel_l2([g.em_get_temperature_rise()], [o.temperature_rise()]) <= tol
        g.close(); o.close()
        print("precision %d: leapfrog, E-only and coupled sweeps match the oracle" % precision, flush=True)


if __name__ == "__main__":
    main()
