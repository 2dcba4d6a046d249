"""Schedule fuzzing of the sweep's barrier-free plane loop (the race / sync evidence SURVEY.md section 5 asks for;
compute-sanitizer is closed on this GPU pool, see profiles/r2_sanitizer.md).

libem_fuzz.so is the same library compiled with -DEM_SWEEP_FUZZ: every mbarrier arrive / wait, named-barrier arrive /
sync, TMA issue and phase boundary of k_sweep_tma delays its warp by a pseudo-random 0-8 us (several plane-times; a plane
takes ~2.5 us per CTA), differently in every run.  If an ordering edge of the hand-off protocol were missing -- a row
read before its producer published it, a staged slot refilled before every warp consumed it, an exchange row overwritten
while a neighbour still reads it -- some schedule among these would produce different bits.  All outputs must stay
BIT-IDENTICAL to the unfuzzed run, for the leapfrog, the E-only recurrence and the thermally coupled sweep."""
import numpy as np
import pytest

import workloads as W
import paper_2603_07038_b200 as P

pytestmark = pytest.mark.gpu


def _outputs(p, lib, steps, **kw):
    import torch
    g = P.EM(p, lib=lib, **kw)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); g.em_step(steps); e1.record(); torch.cuda.synchronize()
    _outputs.ms = e0.elapsed_time(e1)
    out = g.fields() + [g.joule_maps()[1]]
    if getattr(p, "thermal", None) is not None:
        out.append(g.em_get_temperature_rise())
    g.close()
    return out


CASES = [pytest.param(dict(precision=32), False, id="leapfrog-fp32"),
         pytest.param(dict(precision=64), False, id="leapfrog-fp64"),
         pytest.param(dict(precision=32, formulation=P.EM_FORM_EONLY), False, id="eonly-fp32"),
         pytest.param(dict(precision=64, formulation=P.EM_FORM_EONLY), False, id="eonly-fp64"),
         pytest.param(dict(precision=32), True, id="coupled-fp32"),
         pytest.param(dict(precision=64), True, id="coupled-fp64")]


@pytest.mark.parametrize("kw,thermal", CASES)
def test_random_warp_delays_do_not_change_a_bit(kw, thermal):
    fuzz = P.load_fuzz()
    # 250 x 45 cells: 3 x 4 (fp32) .. 5 x 5 (fp64) tiles, 3 z chunks of ~11 planes, PMC at -z (warm-up plane), 40 ports
    p = W.random_problem(250, 45, 33, seed=31337, steps=12, n_ports=40, bc=(0, 1, 0, 0, 1, 0))
    if thermal:
        p.thermal = W.thermal_table(); p.thermal[:, 1] *= 2.0e5; p.thermal[:, 2] *= 1.0e4
    assert fuzz.em_fuzz_seed(0) == 0
    ref = _outputs(p, P.load(), 12, z_chunks=3, **kw)
    assert all(np.isfinite(a).all() for a in ref) and np.abs(ref[0]).max() > 0
    same = _outputs(p, fuzz, 12, z_chunks=3, **kw)                   # seed 0: the fuzz build itself is the same arithmetic
    ms_plain = _outputs.ms
    assert all(np.array_equal(a, b) for a, b in zip(ref, same))
    slow = []
    for seed in (1, 2, 3, 4, 5):
        assert fuzz.em_fuzz_seed(seed) == 0
        got = _outputs(p, fuzz, 12, z_chunks=3, **kw)
        slow.append(_outputs.ms / ms_plain)
        for n, (a, b) in enumerate(zip(ref, got)):
            assert np.array_equal(a, b), (seed, n)
    fuzz.em_fuzz_seed(0)
    print("fuzzed runs took %s x the unfuzzed time" % ["%.1f" % s for s in slow])
    assert min(slow) > 1.5                                         # the delays are really there
