"""C-ABI checks that need no GPU: the library loads, exports every symbol include/gda.h declares,
validates arguments before touching the device, and fails loudly (no CPU fallback) without one."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

from paper_2509_21064_b200 import api, build, workloads as wl

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def L():
    build.build()
    return api.lib()


def declared_symbols():
    text = (ROOT / "include" / "gda.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gda_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(L):
    names = declared_symbols()
    assert set(names) == set(api.EXPORTS)
    for name in names:
        assert getattr(L, name) is not None


def test_struct_layouts_match_header():
    assert C.sizeof(api.Params) == 48 and api.Params.seed.offset == 32 and api.Params.dual.offset == 40
    assert C.sizeof(api.Extra) == 56 and api.Extra.ones.offset == 48
    assert C.sizeof(api.Info) == 40


def has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def test_invalid_arguments_are_rejected_before_the_device(L):
    P = wl.config(1).problem
    with pytest.raises(api.GdaError) as e:
        api.Problem.create_qubo_csr(0, P.rowptr, P.col, P.val, P.c)
    assert e.value.status == 1
    bad = P.val.copy()
    bad[0] = 7.0
    with pytest.raises(api.GdaError) as e:                       # asymmetric Q
        api.Problem.create_qubo_csr(P.n, P.rowptr, P.col, bad, P.c)
    assert e.value.status == 1 and "symmetric" in str(e.value)
    badc = P.col.copy()
    badc[3] = P.n
    with pytest.raises(api.GdaError) as e:                       # column out of range
        api.Problem.create_qubo_csr(P.n, P.rowptr, badc, P.val, P.c)
    assert e.value.status == 1
    S = wl.random_ksat(10, 20, 3, 1)
    lit = S.lit.copy()
    lit[1] = -lit[0]                                              # a variable twice in one clause (reading R2)
    with pytest.raises(api.GdaError) as e:
        api.Problem.create_maxsat(S.n, S.m, S.cptr, lit, S.w)
    assert e.value.status == 1 and "repeated" in str(e.value)
    cptr = S.cptr.copy()
    cptr[1] = 0                                                   # empty clause
    with pytest.raises(api.GdaError) as e:
        api.Problem.create_maxsat(S.n, S.m, cptr, S.lit, S.w)
    assert e.value.status == 1
    Q = np.zeros((100, 100), dtype=np.float32)
    with pytest.raises(api.GdaError) as e:                       # only the bf16 / tcgen05 dense path exists
        api.Problem.create_qubo_dense(100, Q, None, flags=0)
    assert e.value.status == 4
    # Max-k-Cut: a malformed CSR is an INVALID_ARG, never a host fault (validated before the diagonal scan reads it)
    one = np.array([1.0], np.float32)
    for rowptr, col, val in ((np.array([0, 2, 1], np.int32), np.array([1, 0], np.int32), np.array([1.0, 1.0], np.float32)),
                             (np.array([1, 1, 2], np.int32), np.array([1, 0], np.int32), np.array([1.0, 1.0], np.float32)),
                             (np.array([0, 1, 2], np.int32), None, None),
                             (np.array([0, 1, 2], np.int32), np.array([1, 0], np.int32), None),
                             (np.array([0, 1, 2], np.int32), np.array([5, 0], np.int32), np.array([1.0, 1.0], np.float32))):
        with pytest.raises(api.GdaError) as e:
            api.Problem.create_maxkcut(2, 3, rowptr, col, val)
        assert e.value.status == 1, (rowptr, col)
    del one
    Q = np.zeros((256, 256), dtype=np.float32)
    Q[0, 1] = 1.0
    with pytest.raises(api.GdaError) as e:
        api.Problem.create_qubo_dense(256, Q, None)
    assert e.value.status == 1
    h = C.c_void_p(123)
    assert L.gda_create_qubo_csr(4, None, None, None, None, C.byref(h)) == 1 and h.value is None   # out set to NULL
    L.gda_destroy(None)                                           # NULL-safe
    assert L.gda_set_option(None, api.OPT_GRAPHS, 0) == 1 and b"null handle" in L.gda_last_error()


@pytest.mark.skipif(has_gpu(), reason="only meaningful on a box without a GPU")
def test_no_cpu_fallback_without_a_device(L):
    P = wl.config(1).problem
    with pytest.raises(api.GdaError) as e:
        api.Problem.create_qubo_csr(P.n, P.rowptr, P.col, P.val, P.c)
    assert e.value.status == 3 and "no CPU fallback" in str(e.value)


def test_static_score_checks_sizes_before_the_device(L):
    """gda_score_qubo_csr_static (the entry point that allocates nothing): sizes beyond its fixed scratch array and null
    pointers are refused before any CUDA call, with a message that names the limit."""
    text = (ROOT / "include" / "gda.h").read_text()
    assert int(re.search(r"#define GDA_STATIC_SCORE_MAX_B (\d+)", text).group(1)) == api.STATIC_SCORE_MAX_B
    one = C.c_void_p(256)                                         # never dereferenced: the checks below fail first
    f = L.gda_score_qubo_csr_static
    assert f(5, one, one, one, None, api.STATIC_SCORE_MAX_B + 1, one, one, None) == 4
    assert b"GDA_STATIC_SCORE_MAX_B = 4096" in L.gda_last_error()
    assert f(0, one, one, one, None, 8, one, one, None) == 1
    assert f(5, one, one, one, None, 0, one, one, None) == 1
    assert f(5, None, one, one, None, 8, one, one, None) == 1
    assert f(5, one, one, one, None, 8, one, None, None) == 1
    if not has_gpu():                                             # valid sizes, no device: loud failure, no CPU path
        assert f(5, one, one, one, None, 8, one, one, None) == 3


def test_product_path_does_not_import_the_oracle():
    pkg = ROOT / "paper_2509_21064_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")):
        text = f.read_text()
        assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
        assert not re.search(r"oracle[/.](pdbo|_build)", text), f
        assert not re.search(r"#include\s*[<\"][^>\"]*oracle", text), f
