"""DESIGN.md section 7, rule 5: under `pytest -m gpu -x` code no GPU has run yet is collected after code that has.
A device fault is sticky for the process, so the order of the `-m gpu` files is part of the safety scheme; this test
pins it, and pins that only the last file may select or sweep the fused tile ids that have not run on hardware."""
import os
import re
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
ORDER = ["test_gpu_a_parity.py", "test_gpu_z_fullsize.py", "test_gpu_zz_round2.py", "test_gpu_zzz_new_fused_ids.py"]


def test_gpu_files_collect_in_the_documented_order():
    r = subprocess.run([sys.executable, "-m", "pytest", "tests", "-m", "gpu", "--collect-only", "-q", "-p", "no:cacheprovider"],
                       cwd=ROOT, capture_output=True, text=True, timeout=300)
    files = []
    for ln in r.stdout.splitlines():
        if "::" in ln:
            f = os.path.basename(ln.split("::")[0])
            if not files or files[-1] != f:
                files.append(f)
    assert files == ORDER, (files, r.stdout[-400:], r.stderr[-400:])


def test_only_the_last_file_reaches_the_new_fused_ids():
    for name in ORDER[:-1]:
        src = open(os.path.join(ROOT, "tests", name)).read()
        # an explicit choice of a fused BSSN tile id: literals only, and below 5
        for m in re.finditer(r"set_variant\(\s*1\s*,\s*(\w+)\s*\)", src):
            arg = m.group(1)
            assert not arg.isdigit() or int(arg) < 5, (name, m.group(0))
        # every sweep on a 4th-order BSSN handle in these files is bounded; count the calls against the bounds
        if name != "test_gpu_a_parity.py":
            continue
        assert "autotune_fused_ids\", ROUND1_FUSED_IDS" in src
    src = open(os.path.join(ROOT, "tests", "test_gpu_zz_round2.py")).read()
    assert src.count("h.autotune()") == src.count('h.set_param("autotune_fused_ids", fused_ids)') == 2
    src = open(os.path.join(ROOT, "tests", "test_gpu_z_fullsize.py")).read()
    # its four sweeps: one 4th-order BSSN handle (bounded), two wave systems and the 8th-order BSSN system (one fused id)
    assert src.count("h.autotune()") == 4 and src.count('h.set_param("autotune_fused_ids", 5)') == 1
