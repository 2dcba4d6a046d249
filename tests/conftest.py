import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: minutes of host-side oracle time per test; runs only with EM_RUN_SLOW=1")


# GPU tests written AFTER GPU use was closed for this repository in round 2: green on the emulated
# build (tests/emu), never run on a B200.  They are collected LAST: the suite runs with `pytest -x`, and a first-contact
# failure in one of them must not hide the hardware-verified suite behind it.
HARDWARE_UNSEEN = {
    "test_checkpoint_resume_is_bit_exact_and_check_finite",
    "test_slabs_initial_state_with_pec_material_across_the_cut",
    "test_nodal_thermally_coupled_slabs",
    "test_peer_halo_argument_errors",
    "test_nodal_coupled_random_grids",
    "test_nodal_with_pmc_walls_diffusion_and_api",
    "test_nodal_paper_mesh_unknown_count_and_package_slice",
}

# GPU tests that passed on a B200 but run the SPLIT strategy, whose E / Joule kernels changed after the closure
# (profiles/r2_sass_check.md): the cases with "split" in their id, and these, which pick the strategy inside.  Second to last.
SPLIT_INSIDE = {"test_pure_diffusion_and_set_get_temperature", "test_coupled_config4_scaled", "test_thermally_coupled_slabs"}


def pytest_collection_modifyitems(config, items):
    def tier(it):                           # 0: code measured on a B200; 1: seen tests over changed kernels; 2: unseen tests
        name = getattr(it, "originalname", None)
        if name in HARDWARE_UNSEEN:
            return 2
        return 1 if ("split" in it.name or name in SPLIT_INSIDE) and "gpu" in it.keywords else 0
    items.sort(key=tier)                    # stable: the order is kept within a tier
    if os.environ.get("EM_RUN_SLOW", "") != "1":
        slow = pytest.mark.skip(reason="slow: set EM_RUN_SLOW=1")
        for it in items:
            if "slow" in it.keywords:
                it.add_marker(slow)
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)
