"""The C-ABI boundary without a GPU: the in-tree library loads, exports every function that
include/ttt.h declares (and the binding names the same set), and the argument checks that run before
any CUDA call behave as the header says. No compute call is made here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ttt.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)             # comments name functions too
    return sorted(set(re.findall(r"\b(ttt_[a-z_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2604_08542_b200 import _build, binding
    _build.build()
    return binding.load_library()


def test_library_exports_every_declared_function(lib):
    names = _declared()
    assert "ttt_chunk_step" in names and "ttt_init" in names and len(names) >= 14
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/ttt.h but not exported"


def test_binding_names_match_the_header():
    from paper_2604_08542_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()


def test_status_strings_and_version(lib):
    assert lib.ttt_version().decode().startswith("ttt-b200")
    seen = {lib.ttt_strerror(s).decode() for s in range(0, -8, -1)}
    assert len(seen) == 8 and "ok" in seen
    assert lib.ttt_strerror(-99).decode() == "unknown status"


def test_create_argument_checks_run_before_any_cuda_call(lib):
    from paper_2604_08542_b200.binding import _Config
    ctx = ctypes.c_void_p()
    assert lib.ttt_create(None, None) == -1                                         # TTT_ERR_ARG
    bad = _Config(0, 64, 128, 1, 0, 0, 0, 0, 256, 0, 0)                            # nh = 0
    assert lib.ttt_create(ctypes.byref(ctx), ctypes.byref(bad)) == -1 and not ctx.value
    shape = _Config(2, 66, 128, 1, 0, 0, 0, 0, 256, 0, 0)                          # hd % 4 != 0
    assert lib.ttt_create(ctypes.byref(ctx), ctypes.byref(shape)) == -2 and not ctx.value
    # a bf16 shape no tcgen05 kernel takes: refused with a reason, no silent CUDA-core path
    slow = _Config(2, 64, 512, 1, 0, 0, 0, 0, 256, 0, 0)
    assert lib.ttt_create(ctypes.byref(ctx), ctypes.byref(slow)) == -5 and not ctx.value
    assert b"cuda_core_fallback" in lib.ttt_create_error()
    resv = _Config(2, 64, 128, 1, 0, 0, 0, 0, 256, 0, 7)                           # reserved != 0
    assert lib.ttt_create(ctypes.byref(ctx), ctypes.byref(resv)) == -1
    assert lib.ttt_launch_count(None) == 0
    lib.ttt_destroy(None)                                                           # NULL is allowed
