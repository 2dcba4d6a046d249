"""Mutation test of the sweep's synchronisation under the emulation (tests/emu): who checks that the checks can fail?

Each case copies paper_2603_07038_b200/csrc to a scratch folder, REMOVES one ordering edge of k_sweep_tma's barrier-free
plane loop (a __syncwarp, an mbarrier wait, a named-barrier sync, the producer's wait for the 'empty' barrier ...),
builds the emulated racecheck library from the mutated copy and runs a few steps of a multi-tile, multi-chunk grid with
EMU_RACECHECK=1.  Every mutation must be REPORTED -- as a race (whatever the schedule), a deadlock or a barrier misuse --
while the unmutated sources run clean (tests/test_emu_sweep.py).  Slow (one instrumented build per mutation): runs with
EM_RUN_SLOW=1; the outcome of this round's run is in profiles/r2_emulation.md."""
import os
import shutil
import sys

import pytest

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "emu"))

import workloads as W
import paper_2603_07038_b200 as P
from oracle import emo
from parity import TOL, compare_state
import build_emu
import emu_em

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2603_07038_b200", "csrc")

# (file, text to find exactly once, replacement, what is removed)
MUTATIONS = {
    "syncwarp-before-publish": ("em_sweep.cuh", "        __syncwarp();\n        if (lane == 0) {\n            mbar_arrive(bar_rowH(w));",
                                "        if (lane == 0) {\n            mbar_arrive(bar_rowH(w));",
                                "the __syncwarp that orders the lanes' H' row stores before lane 0 publishes the row"),
    "wait-for-row-below": ("em_sweep.cuh", "        if (w != 0) mbar_wait(bar_rowH(w - 1), (unsigned)it & 1u);", "",
                           "row j waiting for H'(k) of row j-1"),
    "pair-sync": ("em_sweep.cuh", "        if (!is_top) pair_sync(w + 1);", "        if (!is_top && k != ks + 2) pair_sync(w + 1);",
                  "row j waiting for the (2 Ebar)^2 row of row j+1, on one plane"),
    "producer-waits-for-empty": ("em_sweep.cuh", "            mbar_wait(bar_empty(it & 1), (unsigned)(it >> 1) & 1u);\n            if (!EO) issue_H(k + 2);",
                                 "            if (!EO) issue_H(k + 2);", "the producer waiting until every warp has pulled the staged plane before refilling its slots"),
    "wait-for-H-planes": ("em_sweep.cuh", "                mbar_wait(bar_fullH(it & 1), (unsigned)(it >> 1) & 1u);   // H(k) has landed", "",
                          "the wait for the staged H planes"),
    "wait-for-q": ("em_sweep.cuh", "        cp_async_wait<0>();                       // q(k-1) has landed (private slot: no barrier needed)", "",
                   "the wait for the cp.async of q"),
}


def _mutated_lib(tmp_path, name):
    fname, old, new, _ = MUTATIONS[name]
    dst = os.path.join(str(tmp_path), "csrc")
    shutil.copytree(CSRC, dst)
    path = os.path.join(dst, fname)
    src = open(path).read()
    assert src.count(old) == 1, "mutation target not found exactly once: " + name
    open(path, "w").write(src.replace(old, new))
    return build_emu.build_emu("race", ["-fsanitize=thread", "-I", os.path.join(ROOT, "include")], opt="-O1", csrc_dir=dst, out_dir=str(tmp_path))


@pytest.mark.slow
@pytest.mark.parametrize("name", sorted(MUTATIONS))
def test_removed_ordering_edge_is_reported(tmp_path, name, monkeypatch):
    import ctypes as C
    import paper_2603_07038_b200.binding as B
    lib = _mutated_lib(tmp_path, name)
    L = B._open(lib)
    L.emu_alloc.restype = C.c_void_p; L.emu_alloc.argtypes = [C.c_size_t]; L.emu_free.argtypes = [C.c_void_p, C.c_size_t]
    monkeypatch.setitem(emu_em._libs, "mut-" + name, L)
    monkeypatch.setenv("EMU_RACECHECK", "1")
    p = W.random_problem(130, 31, 13, seed=5, steps=3, n_ports=4, bc=(0, 1, 1, 0, 1, 0))
    reports = []
    for seed in ("0", "1", "2"):
        monkeypatch.setenv("EMU_SEED", seed)
        try:
            g = emu_em.EmuEM(p, precision=32, z_chunks=3, tag="mut-" + name)
            o = emo.Oracle(p)
            g.em_step(3); o.step(3)
            try:
                compare_state(g, o, TOL[32])
                reports.append(None)
            except AssertionError as e:
                reports.append("PARITY LOST: " + str(e)[:200])
            g.close(); o.close()
        except P.EMError as e:
            reports.append(str(e))
    print(name, "(%s removed) ->" % MUTATIONS[name][3], [r[:400] if r else "NOT REPORTED" for r in reports])
    assert all(r is not None for r in reports), (name, reports)
    if name != "wait-for-q":          # (q lives in the thread's private slot: a missing wait shows as stale data, not as a race)
        assert any("RACE" in r or "DEADLOCK" in r or "more arrivals" in r for r in reports), reports
