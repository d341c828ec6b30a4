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


def test_batch_size_matches_oracle_eq12():
    """sq_batch_size is host arithmetic: the library must agree with the oracle's Eq. 12 everywhere,
    including exact squares and values near 2^64."""
    import numpy as np
    import oracle
    from paper_2602_17330_b200 import binding
    rng = np.random.default_rng(0)
    cases = [(10**7, 10**9, 4, 25), (10**7, 10**5, 8, 130), (20, 10**9, 4, 25), (10**6, 640000, 2, 32),
             (10**6, 639999, 2, 32), (0, 10**9, 1, 1), (10**12, 2**64 - 1, 1, 1), (10**12, (2**32 - 1)**2, 1, 1),
             (10**12, (2**32 - 1)**2 - 1, 1, 1)]
    for _ in range(2000):
        s = int(rng.integers(1, 2**31))
        cl = int(rng.integers(1, 5000))
        delta = int(rng.integers(-2, 3))
        cases.append((int(rng.integers(0, 2**40)), max(0, s * s * cl + delta), cl, 1))
        cases.append((int(rng.integers(0, 2**40)), int(rng.integers(0, 2**63)), int(rng.integers(1, 2**20)),
                      int(rng.integers(1, 241))))
    for n, m, c, l in cases:
        if m >= 2**64:
            continue
        assert binding.batch_size(n, m, c, l) == oracle.batch_size(n, m, c, l), (n, m, c, l)
