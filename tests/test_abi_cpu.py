"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/subquad.h declares; host-only entry points behave; no compute is attempted."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "subquad.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2602_17330_b200 import build
    build.build()
    from paper_2602_17330_b200 import binding
    return binding.load_library()


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sq_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    names = _declared_functions()
    assert len(names) >= 15
    for name in names:
        assert hasattr(lib, name), f"{name} declared in subquad.h but not exported"
    from paper_2602_17330_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_strerror_and_workspace_arithmetic(lib):
    from paper_2602_17330_b200 import binding
    assert binding.strerror(0) == "ok"
    for code in range(-7, 0):
        assert binding.strerror(code) not in ("ok", "unknown error")
    assert binding.strerror(-99) == "unknown error"
    s = binding.SqSizes(100000, 1500000, 28, 64, 16, 512, 4_000_000)
    pack = lib.sq_workspace_bytes(None, binding.OP_PACK, C.byref(s))
    lsh = lib.sq_workspace_bytes(None, binding.OP_LSH, C.byref(s))
    pipe = lib.sq_workspace_bytes(None, binding.OP_PIPELINE_HOST, C.byref(s))
    assert 0 < pack < lsh < pipe
    assert pack >= 100000 * 32            # one 32-byte slot per CDR3
    assert lib.sq_workspace_bytes(None, 99, C.byref(s)) == 0


def test_null_context_is_rejected(lib):
    assert lib.sq_pack(None, None, None, 0, 20, 10) == -1
    assert lib.sq_minhash(None, 3, 64, 0, None) == -1
    assert lib.sq_packed_n(None) == -1


def test_no_cpu_fallback_in_product_path():
    """The package must not import the oracle, and must refuse to run without CUDA."""
    import torch
    pkg = os.path.join(ROOT, "paper_2602_17330_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "sq_oracle" not in text, f
    if not torch.cuda.is_available():
        from paper_2602_17330_b200 import binding
        with pytest.raises(RuntimeError):
            binding.SubQuad(0)
