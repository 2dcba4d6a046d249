"""Host-side invariants of the sweep's work decomposition (csrc/em_tile.cuh): tiles cover the node grid, z chunks
partition the planes, the launch order is a permutation of the work items with x neighbours adjacent, the per-node tile
lists (source index) name the owner and the recomputing neighbours.  Compiled with nvcc as a host program (no GPU)."""
import json
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


@pytest.fixture(scope="module")
def plan_dump(tmp_path_factory):
    if not os.path.exists(NVCC) and not shutil.which("nvcc"):
        pytest.skip("nvcc not found")
    exe = str(tmp_path_factory.mktemp("plan") / "plan_dump")
    subprocess.check_call([NVCC, "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-o", exe,
                           os.path.join(ROOT, "tests", "host", "plan_dump.cu")])

    def run(nx, ny, nz, sz, n_sm=148, forced=0, thermal=0):
        return json.loads(subprocess.check_output([exe] + [str(v) for v in (nx, ny, nz, sz, n_sm, forced, thermal)]))
    return run


CASES = [(1024, 1024, 192, 4, 0), (512, 512, 128, 4, 0), (512, 512, 128, 8, 0), (376, 408, 45, 4, 0), (768, 768, 256, 4, 0),
         (128, 128, 64, 8, 0), (16, 16, 16, 8, 0), (1, 1, 1, 4, 0), (130, 3, 2, 8, 0), (1024, 1024, 192, 4, 1), (21, 18, 33, 8, 1)]


@pytest.mark.parametrize("nx,ny,nz,sz,thermal", CASES)
def test_plan_invariants(plan_dump, nx, ny, nz, sz, thermal):
    for forced in (0, 1, 3, 8):
        f = plan_dump(nx, ny, nz, sz, forced=forced, thermal=thermal)
        assert f["V"] == 16 // sz and f["TXo"] == 30 * f["V"] and f["TY"] == (10 if (sz == 8 or thermal) else 14)
        assert f["ntx"] * f["TXo"] >= nx + 1 > (f["ntx"] - 1) * f["TXo"]          # the tiles cover the nx + 1 node columns
        assert f["nty"] * f["TY"] >= ny + 1 > (f["nty"] - 1) * f["TY"]
        assert f["n_tiles"] == f["ntx"] * f["nty"]
        nzs, kb = f["nzs"], f["kb"]
        assert 1 <= nzs <= 8 and (forced == 0 or nzs == min(forced, max(1, min(8, (nz + 1) // 4))))
        assert kb[0] == 0 and all(kb[c] < kb[c + 1] for c in range(nzs)) and all(v == nz + 1 for v in kb[nzs:])   # planes 0 .. nz
        order = f["order"]
        assert sorted(order) == list(range(f["n_tiles"] * nzs))                   # a permutation of the work items
        # chunk-major, tiles row-major: x neighbours adjacent, y neighbours ntx apart
        tiles = [o // nzs for o in order[:f["n_tiles"]]]
        assert tiles == list(range(f["n_tiles"])) and all(o % nzs == 0 for o in order[:f["n_tiles"]])


def test_tiles_of_node(plan_dump):
    f = plan_dump(1024, 1024, 192, 4)
    own, corner, last, edge = f["tiles_of_node"]
    assert own == [0]
    # node (TXo, TY) is the first node of tile (1, 1) and the +1 halo of tiles (0, 1), (1, 0), (0, 0)
    assert sorted(corner) == sorted([f["ntx"] + 1, f["ntx"], 1, 0])
    assert last == [f["n_tiles"] - 1 - (f["ntx"] - 1 - 1024 // f["TXo"]) - f["ntx"] * (f["nty"] - 1 - 1024 // f["TY"])]
    assert sorted(edge) == [0, 1]
