"""The host-side launch validator (VERDICT r1 task 1a): every rule rejects the plan that breaks it.  CPU only: the
probe is a host program compiled with nvcc (the checker lives in a .cuh next to the kernels)."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_every_rule_rejects_its_violation(tmp_path):
    nvcc = os.environ.get("NVCC") or shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    exe = str(tmp_path / "tma_check_probe")
    subprocess.run([nvcc, "-std=c++17", "-O0", "-o", exe, os.path.join(ROOT, "tests", "native", "tma_check_probe.cu")],
                   check=True, capture_output=True)
    out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout.split()
    got = dict(zip(out[0::2], map(int, out[1::2])))
    assert got.pop("good") == 0 and got.pop("layout_good") == 0
    assert len(got) == 13 and all(v == 1 for v in got.values()), got
