"""The instruction-level claims DESIGN.md makes about the timed kernel, held against the built library (no GPU needed:
cuobjdump / nvdisasm read libcavity.so).  profiles/r3_sass.md is the same report as text."""
import shutil

import pytest


@pytest.fixture(scope="module")
def rep():
    if not (shutil.which("cuobjdump") or shutil.which("/usr/local/cuda/bin/cuobjdump")):
        pytest.skip("no CUDA binary utilities here")
    from paper_0809_3098_b200 import binding, sass_report
    binding.lib()                                   # builds the library if the sources are newer
    return sass_report.report(sass_report.disassemble())


def test_sweep_loops_are_120_fp64_of_at_most_176_instructions_without_local_memory(rep):
    sweeps = [l for l in rep["loops"] if l["fp64"] > 0]
    assert len(sweeps) == 24                        # 6 wall-column classes x 2 wall-row classes x 2 origin parities (which local colour is red)
    for l in sweeps:
        # a sweep of the 4 x 6 micro-tile: 24 point updates x 5 fp64 instructions (3 DADD + 2 DFMA; a masked pair sum turns a
        # DADD into a DFMA in the wall classes), 24 shuffles, 8 + 8 shared-memory accesses, 2 barriers
        assert l["fp64"] == 120 and l["DMUL"] == 0, l
        assert l["len"] <= 176, l
        assert l["SHFL"] == 24 and l["LDS"] == 8 and l["STS"] == 8 and l["BAR"] == 2, l
        assert l["LDL"] == 0 and l["STL"] == 0 and l["LDG"] == 0 and l["STG"] == 0, l


def test_exchange_uses_128_bit_strong_accesses_and_spills_stay_outside_the_sweeps(rep):
    assert rep["mem"]["STG.E.128.STRONG.GPU"] > 0 and rep["mem"]["LDG.E.128.STRONG.GPU"] > 0
    assert sum(n for (op, _), n in rep["local_lines"].items()) <= 48
