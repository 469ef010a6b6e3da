"""CPU-side checks of the C-ABI boundary: the library builds/loads, exports every symbol include/afqmc.h
declares, the ctypes struct matches the header, and argument errors are reported before any launch.
No compute call is made here (no GPU needed)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def afq():
    from paper_1804_03310_b200 import build as b
    b.build()
    import paper_1804_03310_b200 as afq
    return afq


def _header():
    return open(os.path.join(ROOT, "include", "afqmc.h")).read()


def test_every_declared_symbol_is_exported(afq):
    declared = set(re.findall(r"AFQMC_API\s+[\w\s\*]+?\b(afqmc_\w+)\s*\(", _header()))
    assert declared, "no AFQMC_API declarations found"
    assert declared == set(afq.SYMBOLS)
    lib = afq.load_library()
    for name in declared:
        assert hasattr(lib, name), name


def test_header_cites_the_paper_for_every_entry_point():
    h = _header()
    for name in ("afqmc_init", "afqmc_overlap_green", "afqmc_force_bias", "afqmc_propagate", "afqmc_local_energy",
                 "afqmc_step"):
        i = h.index("AFQMC_API afqmc_status " + name + "(")
        comment = h[h.rfind("/*", 0, i):i]
        assert "PAPER.md:" in comment, name


def test_params_struct_matches_header(afq):
    body = re.search(r"typedef struct \{(.*?)\} afqmc_params;", _header(), re.S).group(1)
    fields = re.findall(r"\b(int32_t|double)\s+(\w+);", body)
    want = [(n, C.c_int32 if t == "int32_t" else C.c_double) for t, n in fields]
    assert want == list(afq.AfqmcParams._fields_)
    assert C.sizeof(afq.AfqmcParams) == 4 * 12 + 8 * 2


def test_query_bytes_and_argument_errors(afq):
    p = afq.make_params(200, 13, 12, 1000, 2048, "c64", 0.005)
    cb, wb = afq.afqmc_query_bytes(p)
    assert cb % 256 == 0 and wb % 256 == 0
    # L^T (160 MB) + R (20 MB) + Y (2624^2 + 2400^2 floats) dominate the constants; x2 for the TF32 hi/lo planes
    assert 3.0e8 < cb < 4.0e8 and wb > 2048 * 200 * 200 * 8   # L^T is symmetric-block packed on this path
    cb1, _ = afq.afqmc_query_bytes(afq.make_params(200, 13, 12, 1000, 2048, "c64", 0.005, gemm_path=1))
    assert 2.0e8 < cb1 < 3.0e8
    bad = [afq.make_params(0, 1, 1, 4, 4, "c64", 0.01), afq.make_params(8, 9, 1, 4, 4, "c64", 0.01),
           afq.make_params(8, 2, 2, 4, 4, "c64", -1.0), afq.make_params(8, 2, 2, 4, 4, "c64", 0.01, taylor_order=0),
           afq.make_params(8, 2, 2, 4, 4, "c64", 0.01, n_det=3, n_act=1)]
    for q in bad:
        with pytest.raises(afq.AfqmcError) as e:
            afq.afqmc_query_bytes(q)
        assert e.value.status == afq.AFQMC_EINVAL
    with pytest.raises(afq.AfqmcError) as e:
        afq.afqmc_query_bytes(afq.make_params(80, 40, 2, 4, 4, "c64", 0.01))
    assert e.value.status == afq.AFQMC_EUNSUPPORTED
    lib = afq.load_library()
    assert lib.afqmc_query_bytes(None, None, None) == afq.AFQMC_EINVAL
    assert lib.afqmc_launch_count(None) == 0


def test_init_rejects_bad_inputs_before_touching_the_device(afq):
    import numpy as np
    lib = afq.load_library()
    p = afq.make_params(4, 1, 1, 2, 2, "c128", 0.01)
    ctx = C.c_void_p(None)
    h = np.eye(4)
    L = np.zeros((2, 4, 4)); L[0, 0, 1] = 1.0            # not symmetric
    psi = np.eye(4)[:, :1].copy()
    fake = C.c_void_p(256)                                 # never dereferenced: the check fails first
    st = lib.afqmc_init(C.byref(ctx), C.byref(p), h.ctypes.data_as(C.c_void_p), L.ctypes.data_as(C.c_void_p),
                        psi.ctypes.data_as(C.c_void_p), psi.ctypes.data_as(C.c_void_p), None, None, None, fake, fake,
                        None)
    assert st == afq.AFQMC_EINVAL and b"symmetric" in lib.afqmc_last_error(None)
    st = lib.afqmc_init(C.byref(ctx), C.byref(p), None, None, None, None, None, None, None, fake, fake, None)
    assert st == afq.AFQMC_EINVAL and ctx.value is None


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1804_03310_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f
