"""CPU-only: the C-ABI library builds (nvcc cross-compiles sm_100a), loads, and exports every
symbol include/lbm_ibm.h declares.  No compute calls (there is no GPU here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    txt = open(os.path.join(ROOT, "include", "lbm_ibm.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    names = re.findall(r"\b((?:lbm|ibm)_[a-z_]+)\s*\(", txt)
    return sorted(set(names))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_1904_02108_b200 import _build
    path = _build.build()
    lib = ctypes.CDLL(path)
    names = _declared_symbols()
    assert {"lbm_create", "ibm_set_markers", "ibm_set_kinematics", "lbm_ibm_step", "lbm_read_fields"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in lbm_ibm.h but not exported"


def test_binding_lists_the_same_entry_points():
    from paper_1904_02108_b200 import api
    assert sorted(api.EXPORTS) == _declared_symbols()


def test_sass_is_sm100a_only():
    from paper_1904_02108_b200 import _build
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        return
    out = subprocess.run([cuobjdump, "--list-elf", _build.build()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs
