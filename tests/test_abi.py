"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/ile.h declares
(no compute calls: there is no GPU in the CPU test run)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "ile.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ile_[a-z_A-Z0-9]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2505_11655_b200 import build, load_library
    path = build.build()
    assert os.path.exists(path)
    lib = load_library()
    names = _declared()
    assert len(names) >= 25 and "ile_integrator_run" in names and "ile_lnL" in names
    missing = [n for n in names if not hasattr(lib, n)]
    assert not missing, missing
    assert b"sm_100a" in lib.ile_version()


def test_create_fails_loudly_without_a_gpu_or_with_bad_arguments():
    from paper_2505_11655_b200 import load_library
    lib = load_library()
    assert lib.ile_create(None, 0, None) == -1                          # ILE_EINVAL: null out pointer
    ctx = ctypes.c_void_p()
    rc = lib.ile_create(ctypes.byref(ctx), 10 ** 6, None)               # no such device
    assert rc == -4 and not ctx.value                                   # ILE_ECUDA, no CPU fallback
    assert lib.ile_integrator_opts_default(None, 0, 6) == -1


def test_binding_struct_layouts_match_the_header():
    from paper_2505_11655_b200 import binding
    assert ctypes.sizeof(binding.Result) == binding.RESULT_DTYPE.itemsize == 8 * (14 + 8 + 8)
    assert ctypes.sizeof(binding.IntegratorOpts) == 8 + 128 + 16 + 8 + 16 + 16 + 8 + 32 + 3 * 32 + 8
