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


# (nh, hd, hidden, act_dtype, ns_iters, renorm, linear, cuda_core_fallback) -> expected ttt_create outcome.
# "ok" = the shape passes every check that precedes the device query: the call then returns 0 on a B200
# and TTT_ERR_CUDA (-7, "device ... does not exist") on a box without one — never a shape status.
_SHAPES = [
    # BASELINE.json's five configs
    ((1, 64, 128, 0, 0, 0, 0, 0), "ok"),      # cfg1: fp32 path
    ((16, 64, 128, 1, 0, 0, 0, 0), "ok"),     # cfg2
    ((16, 64, 256, 1, 5, 0, 0, 0), "ok"),     # cfg3
    ((16, 64, 256, 1, 0, 1, 0, 0), "ok"),     # cfg4
    ((8, 128, 512, 1, 5, 0, 0, 0), "ok"),     # cfg5
    # the paper's own shape (Table 3): one head of 1024, k = 1, 2, 4
    ((1, 1024, 1024, 1, 0, 0, 0, 0), "ok"),
    ((1, 1024, 2048, 1, 0, 0, 0, 0), "ok"),
    ((1, 1024, 4096, 1, 0, 0, 0, 0), "ok"),
    ((2, 256, 384, 1, 0, 0, 0, 0), "ok"),     # large path: hd % 256 == 0, hidden % 128 == 0
    # hidden sizes that run zero-padded to the next multiple of 128 (k = 1 at hd 64)
    ((4, 64, 64, 1, 0, 0, 0, 0), "ok"),
    ((4, 64, 192, 1, 5, 0, 0, 0), "ok"),
    ((2, 128, 320, 1, 0, 1, 0, 0), "ok"),
    # explicit CUDA-core route for a shape without a tensor kernel
    ((2, 64, 512, 1, 0, 0, 0, 1), "ok"),
    ((2, 32, 64, 1, 0, 0, 0, 1), "ok"),
    # refused: no tensor kernel and no opt-in
    ((2, 64, 512, 1, 0, 0, 0, 0), -5),
    ((2, 32, 64, 1, 0, 0, 0, 0), -5),
    ((2, 128, 2048, 1, 5, 0, 0, 0), -5),      # hd 128 Newton-Schulz: hidden <= 1024
    ((2, 64, 32, 0, 5, 0, 0, 0), -5),         # Newton-Schulz needs hidden >= hd
    # refused: shape outside every path
    ((1, 1024, 4096, 1, 5, 0, 0, 0), -2),     # large path offers no Newton-Schulz
    ((1, 1024, 4096, 1, 0, 1, 0, 0), -2),     # ... and no re-normalisation
    ((1, 1024, 4096, 0, 0, 0, 0, 0), -2),     # fp32 path: hd <= 128
    ((1, 192, 384, 1, 0, 0, 0, 0), -2),       # hd > 128 must be a multiple of 256
    ((1, 4096, 4096, 1, 0, 0, 0, 0), -2),     # hd <= 2048
    ((1, 1024, 1000, 1, 0, 0, 0, 0), -2),     # large path: hidden % 128 == 0
    ((1, 64, 96, 0, 0, 0, 1, 0), -2),         # linear test mode needs hidden == hd
    ((1, 64, 130, 1, 0, 0, 0, 0), -2),        # hidden % 4 == 0
]


@pytest.mark.parametrize("shape,expect", _SHAPES)
def test_supported_shape_set_is_decided_before_the_device_query(lib, shape, expect):
    """include/ttt.h's shape table (ttt_dtype comment) as data: which configs ttt_create takes and
    which status the others get. Runs with or without a GPU."""
    from paper_2604_08542_b200.binding import _Config
    nh, hd, hidden, dt, ns, renorm, linear, fb = shape
    cfg = _Config(nh, hd, hidden, dt, ns, renorm, linear, 0, 256, fb, 0)
    ctx = ctypes.c_void_p()
    rc = lib.ttt_create(ctypes.byref(ctx), ctypes.byref(cfg))
    if expect == "ok":
        assert rc in (0, -7), (rc, lib.ttt_create_error())
        if rc == 0:
            lib.ttt_destroy(ctx)
        else:
            assert not ctx.value and lib.ttt_create_error()
    else:
        assert rc == expect, (rc, lib.ttt_create_error())
        assert not ctx.value and len(lib.ttt_create_error()) > 0


def test_binding_fails_loudly_when_the_library_is_missing(monkeypatch, tmp_path):
    """No CPU / PyTorch fallback: without the built library the binding raises at load time."""
    from paper_2604_08542_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_LIB_PATH", str(tmp_path / "libttt_b200.so"))
    with pytest.raises(ImportError, match="no CPU or PyTorch fallback"):
        binding.load_library()
    with pytest.raises(ImportError):
        binding.TTT(nh=1, hd=64, hidden=128)


def test_context_creation_fails_loudly_without_a_b200(lib):
    """On a box without a CUDA device ttt_create returns TTT_ERR_CUDA and the binding raises; nothing
    routes the call anywhere else (on a B200 the same call succeeds: covered by the -m gpu tests)."""
    import torch
    from paper_2604_08542_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(binding.TTTError) as e:
        binding.TTT(nh=16, hd=64, hidden=128, max_tokens=1024)
    assert e.value.status == -7 and "device" in str(e.value)


def test_product_package_does_not_reach_for_the_oracle():
    """oracle/ is test infrastructure: nothing under paper_2604_08542_b200/ imports, opens or links it,
    and oracle/ does not import the package (the two share only ttt_inputs.py)."""
    pkg = os.path.join(ROOT, "paper_2604_08542_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                hit = re.search(r"import\s+oracle|from\s+oracle|oracle[/.]|ttt_oracle|libttt_oracle", src)
                assert hit is None, (os.path.join(dirpath, f), hit.group(0))   # (comments may name it)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            hit = re.search(r"import\s+paper_2604_08542_b200|from\s+paper_2604_08542_b200|libttt_b200|csrc/", src)
            assert hit is None, (f, hit.group(0))                              # (docstrings may name it)
