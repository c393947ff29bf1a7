"""CPU-side checks of the boundary: the C-ABI library loads without a GPU and exports every symbol
include/dfjk.h declares; argument validation that needs no device; bench.py's host logic."""
import ctypes as ct
import os
import re

import numpy as np

import dfjk_inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "dfjk.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(dfjk_[a-z0-9_]+)\s*\(", txt)))


def test_library_loads_and_exports_every_declared_symbol():
    from paper_2505_03755_b200 import build, load_library
    from paper_2505_03755_b200.api import EXPORTS
    build.build()
    lib = load_library()
    syms = declared_symbols()
    assert "dfjk_create" in syms and "dfjk_get_jk" in syms and "dfjk_destroy" in syms
    for s in syms:
        assert hasattr(lib, s), s
    assert sorted(EXPORTS) == syms           # the binding covers the header, name for name


def test_calls_that_need_no_device():
    from paper_2505_03755_b200 import load_library
    lib = load_library()
    assert lib.dfjk_destroy(None) == 0
    assert lib.dfjk_strerror(0) == b"ok"
    assert lib.dfjk_strerror(1) == b"invalid argument"
    assert lib.dfjk_workspace_bytes(None) == 0
    h = ct.c_void_p()
    assert lib.dfjk_create(4, 0, None, None, ct.byref(h)) == 1        # nao < 1
    assert lib.dfjk_create(-1, 4, None, None, ct.byref(h)) == 1       # naux < 0
    assert lib.dfjk_create(4, 4, ct.c_void_p(12), None, ct.byref(h)) == 1  # B not 8-byte aligned
    assert lib.dfjk_create(4, 4, None, None, None) == 1               # no out pointer
    arr = (ct.c_int * 1)(1)
    assert lib.dfjk_get_jk(None, 1, arr, None, None, None, None, None) == 1
    # the allocation-free entry point checks its maximum sizes before it touches the device
    p = ct.c_void_p(64)                                               # never dereferenced on the host
    assert lib.dfjk_small_jk_static(10, 97, p, 1, arr, p, p, p, p, None) == 1
    assert b"maximum 96" in lib.dfjk_small_jk_static_last_error()
    assert lib.dfjk_small_jk_static(10, 48, p, 9, (ct.c_int * 9)(*[1] * 9), p, p, p, p, None) == 1
    assert b"nset = 9" in lib.dfjk_small_jk_static_last_error()
    assert lib.dfjk_small_jk_static(10, 96, p, 1, (ct.c_int * 1)(49), p, p, p, p, None) == 1
    assert b"maximum 4608" in lib.dfjk_small_jk_static_last_error()
    assert lib.dfjk_small_jk_static(10, 48, p, 1, arr, p, p, None, None, None) == 0   # nothing asked for
    assert lib.dfjk_small_jk_static_last_error() == b""
    hdr = open(os.path.join(ROOT, "include", "dfjk.h")).read()
    assert "#define DFJK_STATIC_SCRATCH_BYTES 8388608" in hdr and "#define DFJK_STATIC_MAX_NSET 8" in hdr


def test_product_does_not_import_the_oracle():
    """the product path must not route through oracle/ (no CPU fallback)"""
    pk = os.path.join(ROOT, "paper_2505_03755_b200")
    for dirpath, _, files in os.walk(pk):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower() or f == "api.py" and False, (f,)
    src = open(os.path.join(ROOT, "oracle", "dfjk_oracle.c")).read()
    assert "paper_2505_03755_b200/csrc" in src          # only named in the header comment
    assert "#include \"" not in src.replace('#include "stddef', "")


def test_generator_is_deterministic_and_chunk_invariant():
    a = dfjk_inputs.make_B_packed(48, 160, 8.0, 1001, chunk_rows=7)
    b = dfjk_inputs.make_B_packed(48, 160, 8.0, 1001, chunk_rows=160)
    assert np.array_equal(a, b)
    c = dfjk_inputs.make_B_packed(48, 160, 8.0, 1001, rows=10)
    assert np.array_equal(c, a[:10])
    x = dfjk_inputs.make_config("lasscf", with_B=False)
    assert x.nocc == [290, 8, 8, 8, 8, 8] and abs(sum(o.sum() for o in x.occ[1:]) - 22.0) < 1e-12
    assert all((o >= 0).all() and (o <= 2).all() for o in x.occ)
    Q = np.concatenate(x.C, axis=1)
    assert np.abs(Q.T @ Q - np.eye(330)).max() < 1e-12              # one QR: mutually orthonormal
    m = dfjk_inputs.make_config("medium", with_B=False)
    assert m.nocc == [150, 140] and (m.occ[0] == 1).all()


def test_bench_work_model_matches_survey_table():
    import bench
    fb = bench.flops_bytes(dfjk_inputs.CONFIGS["large"])
    assert abs(fb["ht"] - 3.456e12) < 1e9 and abs(fb["k"] - 5.185e12) / 5.185e12 < 1e-3
    assert abs(fb["b_bytes"] - 23.0592e9) < 1e6 and abs(fb["j_bytes"] - 46.12e9) / 46.12e9 < 1e-3


def test_options_struct_matches_the_header_field_for_field():
    """dfjk_options crosses the boundary by value layout: the ctypes mirror must list the same fields, in the
    same order and with the same C types as include/dfjk.h, and DFJK.__init__ must take every one of them"""
    import inspect
    from paper_2505_03755_b200.api import DFJK, dfjk_options
    txt = open(os.path.join(ROOT, "include", "dfjk.h")).read()
    body = txt[txt.index("typedef struct {"):txt.index("} dfjk_options;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = re.findall(r"\b(size_t|int)\s+([A-Za-z_0-9]+)\s*;", body)
    ctype = {"size_t": ct.c_size_t, "int": ct.c_int}
    assert [(n, ctype[t]) for t, n in fields] == list(dfjk_options._fields_)
    assert ct.sizeof(dfjk_options) == 8 + 4 * (len(fields) - 1) + (4 * (len(fields) - 1)) % 8
    params = inspect.signature(DFJK.__init__).parameters
    for _, n in fields:
        assert n in params, n
