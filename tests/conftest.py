import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle():
    from oracle import oracle as o
    o.lib()
    return o


_EMU = {}          # (name, shared, flags) -> Future of the built path
_EMU_POOL = None

# every emulator build the CPU suite uses: started together on the first request, so the compiles overlap
_EMU_ALL = [("fused_emu", False, ()), ("wave_emu", False, ()), ("boundary_emu", False, ()), ("basic_emu", False, ()),
            ("libchemora_emu", True, ()),
            ("fused_emu", False, ("-O0", "-fsanitize=address")), ("wave_emu", False, ("-O0", "-fsanitize=address")),
            ("boundary_emu", False, ("-O0", "-fsanitize=address")),
            ("fused_emu", False, ("-O0", "-fsanitize=thread")), ("wave_emu", False, ("-O0", "-fsanitize=thread")),
            ("fused_emu", False, ("-O0", "-fsanitize=thread", "-DCHM_EMU_DROP_NAMED_BARRIERS"))]


def _build_one(name, shared, flags):
    import subprocess
    import tempfile
    d = tempfile.mkdtemp(prefix="chm_emu_")
    exe = os.path.join(d, name + (".so" if shared else ""))
    opt = [] if any(f.startswith("-O") for f in flags) else ["-O1"]
    r = subprocess.run(["g++", "-std=c++17", "-DCHM_EMULATE", "-pthread"] + opt + list(flags) +
                       (["-shared", "-fPIC"] if shared else []) +
                       ["-o", exe, os.path.join(ROOT, "tests", "native", name + ".cpp")], capture_output=True, text=True)
    return exe, r.returncode, r.stderr


def build_emulator(name, shared=False, flags=()):
    """g++ -DCHM_EMULATE build of tests/native/<name>.cpp (a kernel source on top of cta_emu.hpp), once per session.
    shared=True: as a shared library; flags: extra compiler flags (sanitizers).  Returns the path; a failed build
    raises, except a missing sanitizer runtime, which skips the test."""
    global _EMU_POOL
    from concurrent.futures import ThreadPoolExecutor
    key = (name, bool(shared), tuple(flags))
    if _EMU_POOL is None:
        # the longest build (libchemora_emu, ~50 s) bounds the total: four at a time is as fast as eight, at half the memory
        _EMU_POOL = ThreadPoolExecutor(max_workers=max(2, min(4, (os.cpu_count() or 2))))
        for k in _EMU_ALL:
            _EMU[k] = _EMU_POOL.submit(_build_one, *k)
    if key not in _EMU:
        _EMU[key] = _EMU_POOL.submit(_build_one, *key)
    exe, rc, err = _EMU[key].result()
    if rc != 0:
        if any("sanitize" in f for f in flags) and ("asan" in err.lower() or "tsan" in err.lower()):
            pytest.skip("sanitizer runtime not available")
        raise RuntimeError("emulator build failed: %s\n%s" % (name, err[-3000:]))
    return exe
