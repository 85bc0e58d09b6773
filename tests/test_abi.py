"""CPU-only checks of the boundary: liblgf.so builds, loads without a GPU, exports every symbol
include/lgf.h declares, and its host-side argument validation works.  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1210_8018_b200 import build, lgf

    build.build()
    return lgf.lib()


def header_symbols():
    src = open(os.path.join(ROOT, "include", "lgf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lgf_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(L):
    from paper_1210_8018_b200 import lgf

    syms = header_symbols()
    assert len(syms) >= 15
    assert sorted(lgf.SYMBOLS) == syms          # the binding names exactly what the header declares
    for s in syms:
        assert hasattr(L, s), s


def test_create_validates_extents_and_precision(L):
    from paper_1210_8018_b200 import lgf

    ctx = ctypes.c_void_p()
    for bad in [(7, 8, 8, 8), (8, 8, 8, 2), (8, 8, 10, 8), (8, 8, 8, 128), (8, 14, 8, 8)]:
        assert L.lgf_create(*bad, lgf.PREC_FP64, ctypes.byref(ctx)) == lgf.ERR_UNSUPPORTED_SIZE
        assert not ctx.value
        assert b"extent" in L.lgf_last_error(None)
    assert L.lgf_create(8, 8, 8, 8, 7, ctypes.byref(ctx)) == lgf.ERR_INVALID_ARG
    assert L.lgf_create(8, 8, 8, 8, 0, None) == lgf.ERR_INVALID_ARG
    for good in [(8, 8, 8, 8), (4, 6, 12, 48), (32, 32, 32, 64), (16, 18, 24, 36)]:
        assert L.lgf_create(*good, lgf.PREC_FP32, ctypes.byref(ctx)) == lgf.OK
        assert L.lgf_destroy(ctx) == lgf.OK
    assert L.lgf_destroy(None) == lgf.OK


def test_options_and_workspace_size(L):
    from paper_1210_8018_b200 import lgf

    ctx = ctypes.c_void_p()
    assert L.lgf_create(32, 32, 32, 32, lgf.PREC_FP64, ctypes.byref(ctx)) == lgf.OK
    V = 32 ** 4
    bfused = L.lgf_workspace_bytes(ctx)
    assert L.lgf_set_option(ctx, lgf.OPT_FUSION, 2) == lgf.ERR_INVALID_ARG
    assert L.lgf_set_option(ctx, lgf.OPT_FUSION, 0) == lgf.OK
    b18 = L.lgf_workspace_bytes(ctx)
    assert bfused - b18 == (4 * 9 + 6) * V * 16          # fusion: second link buffer + rows 0, 1 of g
    assert L.lgf_set_option(ctx, lgf.OPT_RECON, 12) == lgf.OK
    b12 = L.lgf_workspace_bytes(ctx)
    assert b18 - b12 == 4 * 3 * V * 16                   # row 2 of every link is not stored
    assert b12 >= (4 * 6 + 4) * V * 16                   # links + 4 packed fields
    assert L.lgf_set_option(ctx, lgf.OPT_FFT_BATCH, 9) == lgf.OK
    assert L.lgf_workspace_bytes(ctx) - b12 == 5 * V * 16
    assert L.lgf_set_option(ctx, lgf.OPT_RECON, 13) == lgf.ERR_INVALID_ARG
    assert b"RECON" in L.lgf_last_error(ctx)
    assert L.lgf_set_option(ctx, lgf.OPT_FFT_BATCH, 6) == lgf.ERR_INVALID_ARG
    assert L.lgf_set_option(ctx, 99, 0) == lgf.ERR_INVALID_ARG
    assert L.lgf_set_option(ctx, lgf.OPT_CHECK_INTERVAL, 0) == lgf.ERR_INVALID_ARG
    assert L.lgf_set_option(ctx, lgf.OPT_MAX_ITER, 10) == lgf.OK
    assert L.lgf_set_option(ctx, lgf.OPT_GMAP, 2) == lgf.ERR_INVALID_ARG
    assert L.lgf_set_option(ctx, lgf.OPT_GMAP, lgf.GMAP_EXP) == lgf.OK
    assert L.lgf_set_option(ctx, lgf.OPT_ACCUM_G, -1) == lgf.ERR_INVALID_ARG
    assert L.lgf_set_option(ctx, lgf.OPT_ACCUM_G, 1) == lgf.OK
    assert L.lgf_bind(ctx, 256, 1 << 40, None) == lgf.ERR_INVALID_ARG   # FUSION = 0, FFT_BATCH = 9 here
    assert b"ACCUM_G" in L.lgf_last_error(ctx)
    assert L.lgf_set_option(ctx, lgf.OPT_ACCUM_G, 0) == lgf.OK
    assert L.lgf_sync_links(ctx) == lgf.ERR_NOT_BOUND
    assert L.lgf_workspace_bytes(None) == 0
    # nothing can run before bind / load
    r = lgf.lgf_result()
    assert L.lgf_fix(ctx, 0.08, 1e-15, ctypes.byref(r)) == lgf.ERR_NOT_BOUND
    assert L.lgf_iterate(ctx, 0.08, 1, None) == lgf.ERR_NOT_BOUND
    assert L.lgf_measure(ctx, None, None) == lgf.ERR_NOT_BOUND
    assert L.lgf_bind(ctx, None, 0, None) == lgf.ERR_INVALID_ARG
    assert L.lgf_bind(ctx, 256, 16, None) == lgf.ERR_WORKSPACE_TOO_SMALL
    assert L.lgf_bind(ctx, 257, 1 << 40, None) == lgf.ERR_INVALID_ARG   # not 256-byte aligned
    assert L.lgf_launch_count(ctx) == 0
    assert L.lgf_destroy(ctx) == lgf.OK
    # ACCUM_G: one link buffer instead of two, everything else as in the fused layout
    assert L.lgf_create(32, 32, 32, 32, lgf.PREC_FP64, ctypes.byref(ctx)) == lgf.OK
    assert L.lgf_set_option(ctx, lgf.OPT_ACCUM_G, 1) == lgf.OK
    assert bfused - L.lgf_workspace_bytes(ctx) == 4 * 9 * V * 16
    assert L.lgf_destroy(ctx) == lgf.OK


def test_product_path_does_not_touch_the_oracle():
    """The package must not import, link or read oracle/ or gen/ (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1210_8018_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+(oracle|gen)\b", src, flags=re.M), f
                assert "lgf_oracle" not in src and "orc_" not in src, f


def header_enums():
    """NAME = value pairs of every enum of include/lgf.h."""
    src = open(os.path.join(ROOT, "include", "lgf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return {m.group(1): int(m.group(2)) for m in re.finditer(r"\b(LGF_[A-Z0-9_]+)\s*=\s*(-?\d+)", src)}


def test_binding_constants_equal_the_header_enums():
    from paper_1210_8018_b200 import lgf

    enums = header_enums()
    assert len(enums) >= 60
    checked = 0
    for name, value in enums.items():
        short = name[len("LGF_"):]
        if hasattr(lgf, short):
            assert getattr(lgf, short) == value, name
            checked += 1
    # every option, shard step and region the binding offers is one the header declares, with the same value
    assert checked >= 45
    for short in dir(lgf):
        if short.startswith(("OPT_", "SHARD_", "REGION_", "ERR_", "STAGE_", "FIELD_", "LAYOUT_", "PREC_")):
            assert "LGF_" + short in enums, short
    assert len(lgf.KERNEL_NAMES) == enums["LGF_KERNEL_KINDS"]


def test_round_2_options_validate_on_the_host(L):
    from paper_1210_8018_b200 import lgf

    ctx = ctypes.c_void_p()
    assert L.lgf_create(16, 16, 12, 24, lgf.PREC_FP64, ctypes.byref(ctx)) == lgf.OK
    for key, good, bad in [(lgf.OPT_ZBLOCK, [0, 1, 3, 12], [-1, 5, 24]), (lgf.OPT_ZT_PIPE, [0, 1], [2]),
                           (lgf.OPT_FFT_PASSES, [3, 4, 8], [0, 2, 5]), (lgf.OPT_TMARCH, [0, 1, 2, 4], [3, 8]), (lgf.OPT_LINK_TILE, [0, 1, 128, 256, 512], [-1, 2, 64, 1024]), (lgf.OPT_LINK_STREAM, [0, 1], [-1, 2]),
                           (lgf.OPT_SHARD_WORLD, [0, 1, 2, 4, 8], [5, 3, 16])]:
        for v in bad:
            assert L.lgf_set_option(ctx, key, v) == lgf.ERR_INVALID_ARG, (key, v)
        for v in good:
            assert L.lgf_set_option(ctx, key, v) == lgf.OK, (key, v)
    assert L.lgf_set_option(ctx, lgf.OPT_SHARD_WORLD, 4) == lgf.OK
    assert L.lgf_set_option(ctx, lgf.OPT_SHARD_RANK, 4) == lgf.ERR_INVALID_ARG
    assert L.lgf_set_option(ctx, lgf.OPT_SHARD_RANK, 3) == lgf.OK
    # a sharded context stores Nt / R + 2 time slices of every array plus the two exchange buffers
    sharded = L.lgf_workspace_bytes(ctx)
    assert L.lgf_set_option(ctx, lgf.OPT_SHARD_WORLD, 0) == lgf.OK
    whole = L.lgf_workspace_bytes(ctx)
    assert whole / 4 < sharded < whole / 2
    # the shard calls refuse a context that is not bound / not sharded, without touching a GPU
    off, nb = ctypes.c_size_t(), ctypes.c_size_t()
    assert L.lgf_shard_region(ctx, lgf.REGION_G, ctypes.byref(off), ctypes.byref(nb)) == lgf.ERR_INVALID_ARG
    assert L.lgf_shard_step(ctx, lgf.SHARD_ZT, 0.0, 0.0) == lgf.ERR_NOT_BOUND
    assert L.lgf_destroy(ctx) == lgf.OK
