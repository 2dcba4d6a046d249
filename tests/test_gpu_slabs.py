"""z-slab decomposition (NEXT-3) on ONE GPU: the slab contexts run one after another and exchange
their wall planes by device copies; the assembled result must equal the single-domain run of the same library
(itself parity-checked against the oracle) and the oracle."""
import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP
import paper_2603_07038_b200 as P
from paper_2603_07038_b200 import slabs
from oracle import emo
from parity import rel_l2, TOL

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_ranks", [2, 3])
@pytest.mark.parametrize("kernel", [P.EM_KERNEL_TMA, P.EM_KERNEL_SPLIT])
@pytest.mark.parametrize("precision", [64, 32])
def test_slabs_equal_single_domain(n_ranks, kernel, precision):
    p = W.random_problem(21, 18, 13, seed=9000 + n_ranks, loss_mode=LOSS_CD, steps=40, n_ports=25, bc=(0, 1, 0, 0, 0, 1))
    ranks = slabs.make_ranks_inprocess(p, n_ranks, precision=precision, kernel=kernel)
    single = P.EM(p, precision=precision, kernel=kernel)
    o = emo.Oracle(p)
    slabs.step_inprocess(ranks, 40); single.em_step(40); o.step(40)
    fields, pw, q = slabs.gather_inprocess(ranks)
    fs = single.fields(); ps, qs, _ = single.joule_maps()
    # same kernels, same inputs plane by plane: identical bits
    for c in range(6):
        assert fields[c].shape == fs[c].shape
        assert np.array_equal(fields[c], fs[c]), c
    assert np.array_equal(q, qs) and np.array_equal(pw, ps)
    fo = o.fields(); _, qo, _ = o.joule()
    tol = TOL[precision]
    assert rel_l2(fields[:3], fo[:3]) <= tol and rel_l2(fields[3:], fo[3:]) <= tol and rel_l2([q], [qo]) <= tol
    for r in ranks:
        r.em.close()
    single.close(); o.close()


def test_slabs_config4_scaled_exp_ports_everywhere():
    p = W.make_config(4, scale=16, zscale=4, steps=60)            # 64 x 64 x 48, ports in several layers
    ranks = slabs.make_ranks_inprocess(p, 4, precision=32)
    o = emo.Oracle(p)
    slabs.step_inprocess(ranks, 60); o.step(60)
    fields, pw, q = slabs.gather_inprocess(ranks)
    fo = o.fields(); _, qo, _ = o.joule()
    assert rel_l2(fields[:3], fo[:3]) <= 2e-5 and rel_l2(fields[3:], fo[3:]) <= 2e-5 and rel_l2([q], [qo]) <= 2e-5
    for r in ranks:
        r.em.close()
