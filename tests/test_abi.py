"""CPU-only checks of the boundary: librchfsi.so loads, exports every symbol include/rchfsi.h
declares, the ctypes struct layouts match the header, and (without a GPU) compute entry points
fail loudly instead of falling back."""
import ctypes as C
import os
import re

import pytest

import paper_2503_22652_b200 as P

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "rchfsi.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rchfsi_[a-z_0-9]+)\s*\(", text)))


def test_library_is_built_and_exports_every_declared_symbol():
    from paper_2503_22652_b200 import build
    build.build()
    lib = P.load_library()
    declared = _declared_symbols()
    assert len(declared) >= 12
    for name in declared:
        assert hasattr(lib, name), name
        assert name in P.SYMBOLS, "binding does not type %s" % name
    assert b"sm_100a" in lib.rchfsi_version()


def test_default_options_and_struct_layout():
    lib = P.load_library()
    opt = P.RchfsiOptions()
    opt.apply_prec = 99
    lib.rchfsi_default_options(C.byref(opt))
    assert (opt.apply_prec, opt.store_prec, opt.normalize_columns_before_rr) == (P.FP64, P.FP64, 1)
    assert (opt.adaptive_bounds, opt.noise_eps, opt.noise_seed, opt.g_input_f32) == (0, 0.0, 0, 0)
    assert C.sizeof(P.RchfsiOptions) == 40
    assert C.sizeof(P.RchfsiOperator) == 104


def test_create_rejects_bad_arguments_before_touching_the_device():
    lib = P.load_library()
    h = C.c_void_p()
    op = P.RchfsiOperator()
    op.kind, op.m, op.dense, op.lda = P.OP_DENSE, 8, 4096, 8
    assert lib.rchfsi_create(None, C.byref(op), None, None, 2, None, None) == P.EINVAL
    assert lib.rchfsi_create(C.byref(h), None, None, None, 2, None, None) == P.EINVAL
    assert lib.rchfsi_create(C.byref(h), C.byref(op), None, None, 0, None, None) == P.EINVAL
    assert lib.rchfsi_create(C.byref(h), C.byref(op), None, None, 9, None, None) == P.EINVAL   # N > m
    op.lda = 4
    assert lib.rchfsi_create(C.byref(h), C.byref(op), None, None, 2, None, None) == P.EINVAL
    assert b"lda" in lib.rchfsi_last_error(None)
    op.lda = 8
    opt = P.RchfsiOptions()
    lib.rchfsi_default_options(C.byref(opt))
    opt.store_prec = P.BF16
    assert lib.rchfsi_create(C.byref(h), C.byref(op), None, None, 2, C.byref(opt), None) == P.EINVAL
    opt.store_prec, opt.apply_prec = P.FP32, P.FP64
    assert lib.rchfsi_create(C.byref(h), C.byref(op), None, None, 2, C.byref(opt), None) == P.EINVAL
    bad = P.RchfsiOperator()
    bad.kind, bad.m = 7, 8
    assert lib.rchfsi_create(C.byref(h), C.byref(bad), None, None, 2, None, None) == P.EINVAL


def test_null_handle_is_einval_everywhere():
    lib = P.load_library()
    assert lib.rchfsi_filter(None, 1, None, None, None, 3, 0.0, 1.0, 2.0) == P.EINVAL
    assert lib.rchfsi_filter_host(None, 1, None, None, None, 3, 0.0, 1.0, 2.0) == P.EINVAL
    assert lib.rchfsi_rayleigh_ritz(None, None, None, None, None) == P.EINVAL
    assert lib.rchfsi_apply(None, 0, None, None) == P.EINVAL
    assert lib.rchfsi_destroy(None) == P.EINVAL
    assert lib.rchfsi_launch_count(None) == -1
    assert lib.rchfsi_workspace_bytes(None, None, 4, None, P.USE_FILTER, 10) == 0
    assert lib.rchfsi_add_workspace(None, None, 0) == P.EINVAL
    assert lib.rchfsi_workspace_shortfall(None) == 0 and lib.rchfsi_workspace_used(None) == 0
    assert lib.rchfsi_operator_changed(None) == P.EINVAL
    assert lib.rchfsi_estimate_bounds(None, 10, 0, 0, None) == P.EINVAL
    assert lib.rchfsi_rotate(None, None, None) == P.EINVAL


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    lib = P.load_library()
    h = C.c_void_p()
    op = P.RchfsiOperator()
    op.kind, op.m, op.dense, op.lda = P.OP_DENSE, 8, 4096, 8
    assert lib.rchfsi_create(C.byref(h), C.byref(op), None, None, 2, None, None) == P.ECUDA
    assert b"no CPU fallback" in lib.rchfsi_last_error(None)


def test_workspace_bytes_scales_with_the_block():
    lib = P.load_library()
    op = P.RchfsiOperator()
    op.kind, op.m, op.dense, op.lda = P.OP_DENSE, 1000, 4096, 1000
    a = lib.rchfsi_workspace_bytes(C.byref(op), None, 60, None, P.USE_FILTER, 20)
    b = lib.rchfsi_workspace_bytes(C.byref(op), None, 120, None, P.USE_FILTER, 20)
    assert 1000 * 60 * 8 * 3 <= a < b       # R_X, R_Y and the unfused operator output
    # more entry points need more; the plan needs no device
    c = lib.rchfsi_workspace_bytes(C.byref(op), None, 60, None, P.USE_FILTER | P.USE_SOLVE, 20)
    d = lib.rchfsi_workspace_bytes(C.byref(op), None, 60, None, P.USE_FILTER | P.USE_SOLVE | P.USE_FILTER_HOST | P.USE_BOUNDS, 20)
    assert a < c < d
    # configs[4] as BASELINE.json states it: the filter-only plan fits one B200 next to X (58.5 GB) and G (29.3 GB)
    fe = P.RchfsiOperator()
    fe.kind, fe.m, fe.n_cells, fe.n_loc, fe.conn, fe.cell_mats_f32 = P.OP_FE, 145 ** 3, 24 ** 3, 343, 4096, 4096
    opt = P.RchfsiOptions()
    lib.rchfsi_default_options(C.byref(opt))
    opt.apply_prec, opt.store_prec, opt.g_input_f32 = P.BF16, P.FP32, 1
    w5 = lib.rchfsi_workspace_bytes(C.byref(fe), None, 2400, C.byref(opt), P.USE_FILTER, 50)
    assert 75e9 < w5 < (180e9 - 58.6e9 - 29.3e9)


def test_allocation_free_entry_point_validates_before_touching_the_device():
    """rchfsi_residual_static (static device scratch, N <= RCHFSI_STATIC_MAX_N): bad sizes and null pointers are
    RCHFSI_EINVAL with a message that names the limit, decided on the host before any CUDA call."""
    lib = P.load_library()
    buf = (C.c_double * 8)()
    p = C.cast(buf, C.c_void_p)
    assert lib.rchfsi_residual_static(None, p, p, 4, 2, p, p, None) == P.EINVAL
    assert b"null input" in lib.rchfsi_static_last_error()
    assert lib.rchfsi_residual_static(p, p, p, 4, 2, None, None, None) == P.EINVAL
    assert lib.rchfsi_residual_static(p, p, p, 0, 2, p, p, None) == P.EINVAL
    assert lib.rchfsi_residual_static(p, p, p, 4, P.STATIC_MAX_N + 1, p, p, None) == P.EINVAL
    msg = lib.rchfsi_static_last_error()
    assert b"RCHFSI_STATIC_MAX_N" in msg and str(P.STATIC_MAX_N + 1).encode() in msg
    hdr = open(os.path.join(ROOT, "include", "rchfsi.h")).read()
    assert "#define RCHFSI_STATIC_MAX_N %d" % P.STATIC_MAX_N in hdr
    assert "#define RCHFSI_STATIC_SCRATCH_BYTES %d" % (32 * 8 + 148 * P.STATIC_MAX_N * 8) in hdr
