"""The larger parity cases of the -m gpu suite (configs 1-6 at their test scales, the E-only cavity, the coupled package
slice) on the emulated build (tests/emu) compiled with UBSan traps (-fsanitize=alignment,bounds,null,shift,
signed-integer-overflow -fsanitize-undefined-trap-on-error: a misaligned vector access, an index outside a static array or
an overflowing index computation kills the process).  Slow (minutes each on 8 host cores): runs with EM_RUN_SLOW=1; this
round's run is recorded in profiles/r2_emulation.md."""
import os
import sys

import pytest

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "emu"))

import paper_2603_07038_b200 as P
import emu_em

import test_gpu_parity as TP
import test_gpu_thermal as TT
import test_gpu_eonly as TE

UBSAN = ["-fsanitize=alignment,bounds,null,shift,signed-integer-overflow", "-fsanitize-undefined-trap-on-error"]
FC = ["-DEM_SWEEP_FUSED_CONDUCTION=1"]

JOBS = {
    "config1-te101": lambda: TP.test_config1_cavity_te101(P.EM_KERNEL_TMA),
    "config2-scaled-5000-steps": lambda: TP.test_config2_slab_scaled_full_steps(P.EM_KERNEL_TMA),
    "config3-scaled-fp32": lambda: TP.test_config3_interposer_scaled(32, 1.0),
    "config3-scaled-fp64-kappa100": lambda: TP.test_config3_interposer_scaled(64, 100.0),
    "config4-scaled": lambda: TP.test_config4_package_scaled(P.EM_KERNEL_TMA),
    "config5-scaled": lambda: TP.test_config5_graded_scaled(),
    "config6-paper-mesh-scaled": lambda: TP.test_config6_paper_mesh_scaled(P.EM_KERNEL_TMA),
    "e-only-te101": lambda: TE.test_config1_te101_three_level(),
    "coupled-config4-scaled": lambda: TT.test_coupled_config4_scaled(),
}


@pytest.mark.slow
@pytest.mark.parametrize("fused_conduction", [False, True], ids=["default", "fused-conduction"])
@pytest.mark.parametrize("job", sorted(JOBS))
def test_larger_cases_under_ubsan_traps(monkeypatch, job, fused_conduction):
    if fused_conduction and not job.startswith("coupled"):
        pytest.skip("the switch only changes the coupled sweep")
    tag, defines = ("ubsan_fc", UBSAN + FC) if fused_conduction else ("ubsan", UBSAN)

    def make(p, precision=None, kernel=P.EM_KERNEL_AUTO, device=None, stream=None, lib=None, **kw):
        return emu_em.EmuEM(p, precision=precision, kernel=kernel, tag=tag, defines=defines, **kw)
    monkeypatch.setattr(P, "EM", make)
    monkeypatch.setenv("EMU_SEED", "7" if fused_conduction else "0")
    JOBS[job]()
