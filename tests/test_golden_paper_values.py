"""What the paper prints, read from tests/golden/paper_values.txt (each value with its PAPER.md citation), against the
oracle and the library's host-side rules.  CPU only."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def golden():
    vals = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "paper_values.txt")):
        m = re.match(r"\s*(\w+)\s*=\s*(\d+)\s*#\s*PAPER\.md:\d+", line)
        if m:
            vals[m.group(1)] = int(m.group(2))
    assert len(vals) == 4                      # every value line carries its citation
    return vals


def test_variable_counts(golden, oracle):
    assert oracle.NVARS[oracle.SYS_BSSN] == golden["bssn_evolved_variables"]
    assert oracle.NVARS[oracle.SYS_WAVE1] == golden["sample1_variables"]
    from paper_1307_6488_b200 import inputs
    assert len(inputs.BSSN_NAMES) == golden["bssn_evolved_variables"]


def test_ghost_zone_rule_of_the_upwinded_8th_order_system(golden):
    """chemora_create applies g >= order/2 + 1 to the upwinded BSSN system: exactly the paper's 5 at 8th order"""
    from paper_1307_6488_b200 import binding
    lib = binding.load()
    g = golden["ghost_zones_8th_order_upwinded"]
    assert g == 8 // 2 + 1
    h = ctypes.c_void_p()
    rc = lib.chemora_create(ctypes.byref(h), 8, 8, 8, g - 1, 8, binding.SYS_BSSN, 0.1, None, binding._ALLOC_T(),
                            binding._DEALLOC_T(), None)
    assert rc == binding.EINVAL and not h.value          # one fewer is refused before any device is touched


def test_flop_count_is_of_the_papers_magnitude(golden):
    """the 8th-order fused kernel executes 6908 flop per point and evaluation (S14, counted from its SASS in
    tests/test_abi.py::test_flop_counts_of_the_fused_kernels): the paper's figure within 15 %"""
    assert abs(6908 - golden["flop_per_point_rhs_8th_order"]) / golden["flop_per_point_rhs_8th_order"] < 0.15
