"""CPU-side checks of the CUDA library's boundary: it loads, exports every symbol include/avm.h
declares, validates arguments before touching CUDA, and its host-compiled Hilbert function is a
Hilbert curve.  No compute calls are made here (no GPU in this container)."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1702_02939_b200 import build as avm_build


@pytest.fixture(scope="module")
def binding():
    avm_build.build()
    from paper_1702_02939_b200 import binding as b
    return b


def test_library_exports_every_declared_symbol(binding, repo_root):
    header = open(os.path.join(repo_root, "include", "avm.h")).read()
    declared = set(re.findall(r"\b(avm_[a-z0-9_]+)\s*\(", header))
    assert declared, "no declarations found"
    assert declared == set(binding.ABI_SYMBOLS)
    for name in declared:
        assert hasattr(binding.lib, name), f"{name} not exported"


def test_params_struct_matches_header(binding, repo_root):
    header = open(os.path.join(repo_root, "include", "avm.h")).read()
    body = re.search(r"typedef struct avm_params \{(.*?)\} avm_params;", header, re.S).group(1)
    names = []
    for line in body.splitlines():
        line = line.split("/*")[0].strip().rstrip(";")
        if not line:
            continue
        typ, rest = line.split(None, 1)
        names += [n.strip() for n in rest.split(",")]
    assert names == [f[0] for f in binding.AvmParams._fields_]
    sbody = re.search(r"typedef struct avm_stats \{(.*?)\} avm_stats;", header, re.S).group(1)
    snames = re.findall(r"int64_t\s+(\w+);", sbody)
    assert snames == [f[0] for f in binding.AvmStats._fields_]


def test_observables_struct_matches_header(binding, repo_root):
    header = open(os.path.join(repo_root, "include", "avm.h")).read()
    body = re.search(r"typedef struct avm_observables \{(.*?)\} avm_observables;", header, re.S).group(1)
    names = []
    for line in body.splitlines():
        line = line.split("/*")[0].strip().rstrip(";")
        if not line:
            continue
        typ, rest = line.split(None, 1)
        names += [(typ, n.strip()) for n in rest.split(",")]
    want = [("double" if f[1] is ctypes.c_double else "int64_t", f[0]) for f in binding.AvmObservables._fields_]
    assert names == want
    # the mixed-precision library is the same ABI
    mixed = ctypes.CDLL(binding.LIB_MIXED_PATH)
    for name in binding.ABI_SYMBOLS:
        assert hasattr(mixed, name), f"{name} not exported by the mixed library"
    mixed.avm_precision.restype = ctypes.c_char_p
    assert mixed.avm_precision() == b"mixed"


def test_argument_validation_needs_no_gpu(binding):
    b = binding
    good = b.make_params(64, 16, Lx=8.0, Ly=8.0)
    assert b.lib.avm_workspace_bytes(ctypes.byref(good)) > 0
    for bad in (b.AvmParams(64, 127, 16, 0, 8.0, 8.0),            # V != 2N
                b.AvmParams(64, 128, 15, 0, 8.0, 8.0),            # stride not a multiple of 4
                b.AvmParams(64, 128, 16, 0, -1.0, 8.0),           # bad box
                b.AvmParams(2, 4, 16, 0, 8.0, 8.0)):              # too few cells
        assert b.lib.avm_workspace_bytes(ctypes.byref(bad)) == 0
        h = ctypes.c_void_p()
        rc = b.lib.avm_create(ctypes.byref(bad), None, None, None, None, None, None, None, 0, None, ctypes.byref(h))
        assert rc == -1 and not h.value
    assert b.lib.avm_step(None, 1) == -1
    assert b"workspace" in b.lib.avm_strerror(-2)
    # workspace grows linearly and covers at least the resident state (224 B/cell)
    w1 = b.lib.avm_workspace_bytes(ctypes.byref(b.make_params(1 << 16, 16, Lx=256.0, Ly=256.0)))
    w2 = b.lib.avm_workspace_bytes(ctypes.byref(b.make_params(1 << 17, 16, Lx=256.0, Ly=256.0)))
    assert w1 > 224 * (1 << 16) and 1.9 < w2 / w1 < 2.1


@pytest.mark.parametrize("m", [1, 2, 5, 7])
def test_hilbert_index_is_a_hilbert_curve(binding, m):
    """Bijection onto 0..4^m-1 and consecutive indices are edge-adjacent grid cells (the defining
    locality property, "chosen for its optimal data-locality properties")."""
    g = 1 << m
    d = np.array([[binding.hilbert_index_host(m, x, y) for y in range(g)] for x in range(g)])
    assert sorted(d.ravel().tolist()) == list(range(g * g))
    inv = np.empty((g * g, 2), dtype=np.int64)
    for x in range(g):
        for y in range(g):
            inv[d[x, y]] = (x, y)
    step = np.abs(np.diff(inv, axis=0)).sum(axis=1)
    assert (step == 1).all()
    # nested: the first quarter of the curve stays inside one quadrant
    q = inv[: g * g // 4] // (g // 2) if g > 1 else None
    assert q is None or (q == q[0]).all()


def test_missing_library_fails_loudly(binding, tmp_path, monkeypatch):
    import importlib
    with pytest.raises(binding.AvmError):
        binding._load(str(tmp_path / "nope.so"))


def test_mixed_precision_library_has_the_same_abi(binding):
    """libavm_b200_mixed.so (NEXT-3): same sources, same exported symbols, says what it is"""
    mixed = binding.library("mixed")
    for name in binding.ABI_SYMBOLS:
        assert hasattr(mixed, name), f"{name} not exported by the mixed library"
    assert mixed.avm_precision() == b"mixed" and binding.lib.avm_precision() == b"f64"
    good = binding.make_params(64, 16, Lx=8.0, Ly=8.0)
    assert mixed.avm_workspace_bytes(ctypes.byref(good)) == binding.lib.avm_workspace_bytes(ctypes.byref(good))
