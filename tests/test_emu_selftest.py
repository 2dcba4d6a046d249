"""The CPU emulation of the CUDA primitives (tests/emu: fibers, mbarriers, named barriers, TMA / bulk / cp.async copies)
checked on small kernels of its own: correct ones must reproduce the definition of the operation, and each deliberate bug
-- a missing wait, a misaligned TMA destination, an address out of range, a barrier that can never complete -- must be
REPORTED.  This is what entitles tests/test_emu_sweep.py to call a clean run of the product kernels evidence."""
import ctypes as C
import os
import sys

import pytest

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "emu"))
from build_emu import build_selftest        # noqa: E402

CASES = {
    0: "TMA box: inside the tensor and hanging over its faces (zero fill)",
    11: "named-barrier hand-off between two warps + shuffles and votes",
    12: "cp.async group, waited for",
    2: "BUG consumer reads the staged box without waiting on its mbarrier",
    1: "BUG consumer warp skips one bar.sync of the hand-off",
    3: "BUG expect_tx announces more bytes than the copy delivers (deadlock)",
    13: "BUG mbarrier with two expected arrivals gets one (deadlock)",
    4: "BUG TMA destination not 128-byte aligned",
    5: "BUG store behind the dynamic shared memory",
    6: "BUG more arrivals than the mbarrier expects",
    7: "BUG mbarrier used without mbarrier.init",
    8: "BUG cp.async from a misaligned global address",
    9: "BUG thread exits with a cp.async group never waited for",
    10: "BUG streaming store outside every allocation",
}


RACE_CASES = {
    20: "lanes exchange through shared memory, ordered by __syncwarp",
    23: "two-slot TMA staging ring, refilled after the 'empty' mbarrier collected every warp",
    21: "RACE lanes exchange through shared memory with only a shuffle in between (not an ordering edge)",
    22: "RACE lanes exchange through shared memory with nothing in between",
    24: "RACE staging slot refilled by TMA before the consumers released it",
    25: "RACE consumer warp skips one bar.sync of the hand-off",
    26: "RACE consumer reads the staged box without waiting on its mbarrier",
}


@pytest.fixture(scope="module")
def race_lib():
    L = C.CDLL(build_selftest(race=True))
    L.selftest_run.argtypes = [C.c_int, C.c_char_p, C.c_int]
    return L


@pytest.mark.parametrize("seed", [0, 3, 4])
@pytest.mark.parametrize("case", sorted(RACE_CASES), ids=lambda c: "%02d" % c)
def test_racecheck_selftest(race_lib, case, seed, monkeypatch):
    """the happens-before race detector (EMU_RACECHECK=1 on a -fsanitize=thread build whose hooks the emulation
    implements): races are reported for EVERY schedule, also those in which the values come out right"""
    monkeypatch.setenv("EMU_SEED", str(seed))
    monkeypatch.setenv("EMU_RACECHECK", "1")
    buf = C.create_string_buffer(4096)
    rc = race_lib.selftest_run(case, buf, 4096)
    assert rc == 0, (RACE_CASES[case], buf.value.decode())
    if RACE_CASES[case].startswith("RACE"):
        print(RACE_CASES[case], "->", buf.value.decode())


@pytest.fixture(scope="module")
def lib():
    L = C.CDLL(build_selftest())
    L.selftest_run.argtypes = [C.c_int, C.c_char_p, C.c_int]
    return L


@pytest.mark.parametrize("seed", [0, 3])
@pytest.mark.parametrize("case", sorted(CASES), ids=lambda c: "%02d" % c)
def test_emulation_selftest(lib, case, seed, monkeypatch):
    monkeypatch.setenv("EMU_SEED", str(seed))
    buf = C.create_string_buffer(2048)
    rc = lib.selftest_run(case, buf, 2048)
    assert rc == 0, (CASES[case], buf.value.decode())
    if CASES[case].startswith("BUG"):
        print(CASES[case], "->", buf.value.decode())
