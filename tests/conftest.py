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


_EMU = {}


def build_emulator(name, shared=False):
    """g++ -DCHM_EMULATE build of tests/native/<name>.cpp (a kernel source on top of cta_emu.hpp), once per session;
    shared=True: as a shared library"""
    import subprocess
    import tempfile
    if name not in _EMU:
        d = tempfile.mkdtemp(prefix="chm_emu_")
        exe = os.path.join(d, name + (".so" if shared else ""))
        subprocess.run(["g++", "-std=c++17", "-O1", "-DCHM_EMULATE", "-pthread"] + (["-shared", "-fPIC"] if shared else []) + ["-o", exe,
                        os.path.join(ROOT, "tests", "native", name + ".cpp")], check=True, capture_output=True)
        _EMU[name] = exe
    return _EMU[name]
