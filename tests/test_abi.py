"""The C-ABI library loads and exports every symbol include/*.h declares (heget.h: the product
surface; heget_bench.h: the bench hooks) -- no GPU needed, no compute calls -- and the binding fails
loudly without a CUDA device."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols(headers=("heget.h", "heget_bench.h")):
    syms = set()
    for h in headers:
        text = open(os.path.join(ROOT, "include", h)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        syms |= set(re.findall(r"\b(heget_[a-z0-9_]+)\s*\(", text))
    return sorted(syms)


def test_header_declares_the_north_star_entry_points():
    syms = declared_symbols(("heget.h",))
    for name in ("heget_init", "heget_rambo", "heget_amp2", "heget_xsec_reduce"):
        assert name in syms
    # the bench hooks and the paper's List 2 program are not part of the product header
    for name in ("heget_fma_peak", "heget_launch_count", "heget_list2"):
        assert name not in syms and name in declared_symbols(("heget_bench.h",))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_0908_4403_b200 import binding, build
    lib_path = build.build()
    lib = ctypes.CDLL(lib_path)
    syms = declared_symbols()
    assert len(syms) >= 11
    for name in syms:
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == syms


def test_library_contains_sm100a_code_only():
    import subprocess
    from paper_0908_4403_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, out


def test_strerror_and_einval_without_gpu():
    from paper_0908_4403_b200 import binding
    lib = binding.load_library()
    assert lib.heget_strerror(0) == b"success"
    assert b"invalid" in lib.heget_strerror(-1)
    ctx = ctypes.c_void_p()
    assert lib.heget_init(0, 1 / 128.0, 2 / 3.0, 20.0, 2.5, 0.4, None) == -1      # null out pointer
    assert lib.heget_init(-1, 1 / 128.0, 2 / 3.0, 20.0, 2.5, 0.4, ctypes.byref(ctx)) == -1
    assert lib.heget_amp2(None, None, 4, 1, None, 0, None) == -1
    assert lib.heget_launch_count(None) == 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback():
    from paper_0908_4403_b200 import Heget, HegetError
    with pytest.raises(HegetError):
        Heget(0)
