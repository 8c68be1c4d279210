"""CPU-side checks of the boundary: libchemora.so loads, exports every symbol include/chemora.h declares,
rejects bad arguments, and refuses to compute without a CUDA device (no CPU fallback).  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_1307_6488_b200 import build, binding as b
    build.build()
    b.load()
    return b


def test_exports_every_declared_symbol(binding):
    header = open(os.path.join(ROOT, "include", "chemora.h")).read()
    declared = set(re.findall(r"\b(chemora_[a-z0-9_]+)\s*\(", header))
    declared.discard("chemora_t")
    assert declared == set(binding.SYMBOLS)
    lib = ctypes.CDLL(binding.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name


def test_tile_table(binding):
    shapes = [binding.tile_shape(t, binding.SYS_BSSN, 0) for t in range(binding.NUM_TILES)]
    assert shapes[:6] == [(32, 4, 8), (32, 8, 8), (64, 2, 8), (64, 4, 8), (128, 2, 8), (16, 16, 8)]
    assert shapes[6:] == [shapes[t % 6] for t in range(6, binding.NUM_TILES)]                                   # ids >= 6 repeat id - 6 for marching kernels
    ids = binding.variants(binding.SYS_BSSN, 4, 1)
    assert ids == [0, 1, 2, 3, 4, 5, 6, 7] and binding.variants(binding.SYS_BSSN, 8, 1) == [0]
    assert binding.variants(binding.SYS_BSSN, 4, 0) == binding.variants(binding.SYS_BSSN, 8, 0) == list(range(6))
    assert binding.variants(binding.SYS_WAVE, 4, 1) == list(range(9)) and binding.variants(binding.SYS_WAVE, 4, 0) == []
    fused = [binding.tile_shape(t, binding.SYS_BSSN, 1) for t in ids]
    assert fused[0] == (16, 4, 4) and all(x * y * z in (128, 256) for x, y, z in fused)      # one grid point per thread
    with pytest.raises(binding.ChemoraError):
        binding.tile_shape(8, binding.SYS_BSSN, 1)
    with pytest.raises(binding.ChemoraError):
        binding.tile_shape(binding.NUM_TILES)


@pytest.mark.parametrize("args", [
    (0, 8, 8, 2, 4, 0, 0.1),      # non-positive dim
    (8, 8, 8, 1, 4, 0, 0.1),      # wave O4 needs g >= 2
    (8, 8, 8, 3, 8, 0, 0.1),      # wave O8 needs g >= 4
    (8, 8, 8, 2, 4, 1, 0.1),      # BSSN O4 upwinded needs g >= 3 (PAPER.md:382 rule order/2+1)
    (8, 8, 8, 4, 8, 1, 0.1),      # BSSN O8 upwinded needs g >= 5
    (8, 8, 8, 3, 6, 1, 0.1),      # order not in {4,8}
    (8, 8, 8, 3, 4, 3, 0.1),      # unknown system
    (8, 8, 8, 3, 8, 2, 0.1),      # first-order wave system O8 needs g >= 4
    (8, 8, 8, 3, 4, 1, 0.0),      # dx <= 0
    (2, 8, 8, 3, 4, 1, 0.1),      # dim < ghost
])
def test_create_rejects_bad_arguments(binding, args):
    lib = binding.load()
    h = ctypes.c_void_p()
    rc = lib.chemora_create(ctypes.byref(h), *args[:6], float(args[6]), None, binding._ALLOC_T(), binding._DEALLOC_T(),
                            None)
    assert rc == binding.EINVAL and not h.value


def test_selfcheck_accepts_every_tma_launch_plan(binding):
    """host only: the validator every TMA launcher runs before <<<>>> accepts the plan (shared-memory destinations
    128-byte aligned, 16-byte box rows, even x coordinates, mbarrier byte counts = bytes delivered, shared memory
    within the opt-in limit) of every template instance, Runge-Kutta mode and ghost width (task 1a)"""
    n, report = binding.selfcheck()
    # 7 fused launch plans (ids 5 and 6 share one) x 5 modes x 4 ghost widths + the 8th-order tile x 5 modes x 2 widths, plus the plane-ring kernels
    assert n >= 7 * 5 * 4 + 5 * 2 + 10, report
    assert "0 rejected" in report, report


def test_device_error_codes_are_described(binding):
    """the plumbing of the bounded mbarrier waits: a code a kernel would leave in the device error word maps to a
    message naming the kernel family and the wait that timed out"""
    assert binding.describe_device_error(0) == "no device error"
    assert "section 12" in binding.describe_device_error(0x10000 + 13)
    assert "point-value" in binding.describe_device_error(0x10080)
    assert "plane-ring" in binding.describe_device_error(0x20002)
    assert "unknown" in binding.describe_device_error(0x70001)


def test_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.ChemoraError) as e:
        binding.Chemora(8, 8, 8, 2, 4, 0, 0.1)
    assert e.value.code == binding.ECUDA


def test_null_handle_is_safe(binding):
    lib = binding.load()
    assert lib.chemora_destroy(None) == 0
    assert lib.chemora_rk4_step(None, 0.1) == binding.EINVAL
    assert lib.chemora_launch_count(None) == 0


def test_product_never_touches_the_oracle():
    """the CUDA path must not import, link or read anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1307_6488_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert "oracle" not in open(os.path.join(dirpath, f)).read().replace("oracle/.", "").lower() or \
                    f in ("inputs.py", "common.cuh", "__init__.py"), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1307_6488_b200" not in src and "from paper_1307_6488_b200" not in src
            assert "libchemora" not in src and "csrc" not in src


def test_flop_counts_of_the_fused_kernels(binding):
    """the paper's ~7900 flop per grid point and RHS evaluation at 8th order is an
    order-of-magnitude check on the 8th-order kernel's own FP64 work, and the 4th-order count must be lower.
    Counted from the SASS of the middle-stage instances (DADD + DMUL + 2 DFMA).  The code is straight-line and runs
    once per point, except the loop over the six At_ij advection stencils, whose body appears once and runs six
    times: the static count (3708 / 6108) is the executed one (4088 / 6908; bench.py uses the 4th-order figure) minus
    five such stencils (76 / 160 flops each; the 8th-order one carries the five dissipation weights of S6b)."""
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", binding.LIB_PATH], capture_output=True, text=True, check=True).stdout
    counts, cur = {}, None
    for line in sass.splitlines():
        if "Function :" in line:
            cur = None
            for order in (4, 8):
                if "bssn_tma_kernelILi16ELi4ELi4ELi2ELi%dE" % order in line:
                    cur = order
                    counts[cur] = 0
        elif cur is not None:
            for op, w in (("DADD", 1), ("DMUL", 1), ("DFMA", 2)):
                if " %s " % op in line or " %s." % op in line:
                    counts[cur] += w
    assert set(counts) == {4, 8}, counts
    executed = {4: counts[4] + 5 * 76, 8: counts[8] + 5 * 160}
    assert 3000 < executed[4] < executed[8]
    assert 7900 / 2 < executed[8] < 7900 * 2


def test_static_sass_comparison_tool(binding, capsys):
    """`python -m paper_1307_6488_b200.build --compare OLD.o NEW.o` (how profiles/r02_sass_vs_round1.md was made): an
    object compared with itself shows no change, its counts are those of real instructions (the check it replaces
    filtered every instruction line away and compared nothing), and a differing pair shows as `a -> b`"""
    import shutil
    from paper_1307_6488_b200 import build
    if not (shutil.which("cuobjdump") or os.path.exists("/usr/local/cuda/bin/cuobjdump")):
        pytest.skip("cuobjdump not available")
    obj = os.path.join(os.path.dirname(binding.LIB_PATH), "build", "kernels_boundary.o")
    basic = os.path.join(os.path.dirname(binding.LIB_PATH), "build", "kernels_basic.o")
    if not (os.path.exists(obj) and os.path.exists(basic)):
        pytest.skip("object files of the in-tree build not present")
    g = build._sass_groups(obj)
    assert {"radiative_kernel", "maxdiff_kernel"} <= set(g)
    assert g["radiative_kernel"]["STG"] > 0 and g["radiative_kernel"]["LDG"] > 0
    assert sum(v for o, v in g["radiative_kernel"].items() if o) > 100 and g["radiative_kernel"][""] != g["maxdiff_kernel"][""]
    build.compare(obj, obj)
    out = capsys.readouterr().out
    assert "`radiative_kernel`" in out and "->" not in out and "differs" not in out and out.count("| same |") == 2
    a = build._sass_groups(basic)
    assert a["fill_ghosts_kernel"]["UTMALDG"] == 0 and a["enforce_kernel"]["DMUL"] > 0
