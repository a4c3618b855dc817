"""CPU-side checks of the boundary: libspd.so loads, exports every symbol include/spd.h declares, and rejects
bad arguments before touching the device (no compute calls without a GPU)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1611_09704_b200 import build as B
    B.build()
    import paper_1611_09704_b200 as P
    return P.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "spd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(spd_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(L):
    syms = declared_symbols()
    assert {"spd_stats", "spd_boxcar_snr", "spd_candidates", "spd_stats_merge", "spd_search_fused", "spd_search_host",
            "spd_workspace_bytes", "spd_search_host_arena_bytes", "spd_status_string"} <= set(syms)
    for s in syms:
        assert hasattr(L, s), s


def test_struct_layouts_match_the_header():
    import paper_1611_09704_b200 as P
    assert P.STATS_DTYPE.itemsize == 80 and P.CAND_DTYPE.itemsize == 16
    assert P.STATS_DTYPE.fields["n"][1] == 56 and P.STATS_DTYPE.fields["nmax_of_sigma"][1] == 72


def test_status_strings(L):
    assert L.spd_status_string(0) == b"SPD_OK" and L.spd_status_string(1) == b"SPD_ERR_INVALID_ARG"
    assert L.spd_status_string(2) == b"SPD_ERR_CUDA" and L.spd_status_string(3) == b"SPD_ERR_WORKSPACE"


def test_workspace_sizes(L):
    assert L.spd_workspace_bytes(64, 16384, 32) >= 2 * 2048 * 24
    assert L.spd_workspace_bytes(0, 16384, 32) == 0 and L.spd_workspace_bytes(1, 1, 5000) == 0
    n = 6000 * 262144
    assert L.spd_search_host_arena_bytes(6000, 262144, 128, 1 << 20) >= n * 4 + (16 << 20)      # x + records (+ stats, count, workspace)


def test_argument_validation_needs_no_device(L):
    fake = C.c_void_p(4096)            # never dereferenced: every call below must fail in the argument checks
    INV, WS = 1, 3
    assert L.spd_stats(None, 1, 1, 1, 0, fake, fake, 1 << 20, None) == INV
    assert L.spd_stats(fake, 0, 10, 10, 0, fake, fake, 1 << 20, None) == INV
    assert L.spd_stats(fake, 2, 10, 9, 0, fake, fake, 1 << 20, None) == INV          # row_stride < n_t
    assert L.spd_stats(fake, 2, 10, 10, 11, fake, fake, 1 << 20, None) == INV        # nmax_for_sigma > n_t
    assert L.spd_stats(fake, 2, 10, 10, 0, fake, fake, 16, None) == WS
    assert L.spd_boxcar_snr(fake, 2, 10, 10, fake, 0, 0, fake, fake, fake, 1 << 20, None) == INV
    assert L.spd_boxcar_snr(fake, 2, 10, 10, fake, 11, 0, fake, fake, fake, 1 << 20, None) == INV
    assert L.spd_boxcar_snr(fake, 2, 10000, 10000, fake, 4097, 0, fake, fake, fake, 1 << 20, None) == INV
    assert L.spd_boxcar_snr(fake, 2, 10, 10, fake, 4, 7, fake, fake, fake, 1 << 20, None) == INV   # bad mode
    assert L.spd_boxcar_snr(fake, 2, 10, 10, fake, 4, 0, None, fake, fake, 1 << 20, None) == INV
    assert L.spd_boxcar_snr(fake, 2, 10, 10, fake, 4, 0, fake, fake, fake, 4, None) == WS
    assert L.spd_candidates(None, fake, 2, 10, 10, 6.0, fake, 10, fake, None) == INV
    assert L.spd_candidates(fake, fake, 2, 10, 10, float("nan"), fake, 10, fake, None) == INV
    assert L.spd_candidates(fake, fake, 2, 10, 10, 6.0, None, 10, fake, None) == INV
    assert L.spd_stats_merge(fake, 0, fake, None) == INV
    assert L.spd_search_fused(fake, 2, 10, 10, fake, 4, 0, 6.0, fake, 10, None, fake, 1 << 20, None) == INV
    assert L.spd_search_host(None, 2, 10, 4, 0, 6.0, fake, 10, fake, None, fake, 1 << 30, None) == INV


def test_product_path_has_no_cpu_fallback():
    import torch
    import paper_1611_09704_b200 as P
    with pytest.raises(P.SpdError):
        P.spd_stats(torch.zeros((2, 10)))                 # CPU tensor is refused, not computed
    # and nothing in the package imports the oracle
    pkg = os.path.join(ROOT, "paper_1611_09704_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert "oracle" not in open(os.path.join(dirpath, f)).read(), f


def test_round2_entry_points_validate_arguments(L):
    """spd_stats_rows / spd_boxcar_snr_rows / spd_search_fused_rows / spd_boxcar_snr_decimated / spd_candidates_decimated /
    spd_search_fused_decimated."""
    fake = C.c_void_p(4096)
    INV, WS = 1, 3
    L.spd_decimated_level_offset.restype = C.c_int64
    L.spd_decimated_level_offset.argtypes = [C.c_int64, C.c_int]
    L.spd_decimated_workspace_bytes.restype = C.c_size_t
    assert [L.spd_decimated_level_offset(1003, l) for l in range(5)] == [0, 1008, 1512, 1768, 1896]     # rows of 1003, 501, 250, 125 padded to 8
    assert L.spd_decimated_level_offset(0, 1) == -1
    assert L.spd_decimated_workspace_bytes(C.c_int64(2), C.c_int64(4096), 16, 4) >= 2 * (2048 + 1024) * 4
    assert L.spd_decimated_workspace_bytes(C.c_int64(2), C.c_int64(4096), 24, 4) == 0                      # w0 must be 16 or 32
    assert L.spd_decimated_workspace_bytes(C.c_int64(2), C.c_int64(4096), 32, 9) == 0                      # 32 * 2^8 > 4096
    a = [C.c_int64(2), C.c_int64(4096), C.c_int64(4096)]
    assert L.spd_boxcar_snr_decimated(fake, *a, fake, 8, 2, 0, fake, fake, C.c_int64(8192), fake, C.c_size_t(1 << 30), None) == INV
    assert L.spd_boxcar_snr_decimated(fake, *a, fake, 16, 2, 0, fake, fake, C.c_int64(100), fake, C.c_size_t(1 << 30), None) == INV   # plane_stride too short
    assert L.spd_boxcar_snr_decimated(fake, *a, fake, 16, 2, 0, fake, fake, C.c_int64(8192), fake, C.c_size_t(64), None) == WS
    assert L.spd_candidates_decimated(fake, fake, C.c_int64(2), C.c_int64(4096), C.c_int64(100), 2, C.c_float(5.0), fake, C.c_uint64(10), fake, None) == INV
    assert L.spd_search_fused_decimated(fake, *a, fake, 8, 2, 0, C.c_float(5.0), fake, C.c_uint64(4), fake, fake, C.c_size_t(1 << 30), None) == INV
    assert L.spd_search_fused_decimated(fake, *a, fake, 16, 2, 0, C.c_float(float("nan")), fake, C.c_uint64(4), fake, fake, C.c_size_t(1 << 30), None) == INV
    assert L.spd_search_fused_decimated(fake, *a, fake, 16, 2, 0, C.c_float(5.0), fake, C.c_uint64(4), fake, fake, C.c_size_t(64), None) == WS
    L.spd_workspace_bytes_rows.restype = C.c_size_t
    assert L.spd_workspace_bytes_rows(C.c_int64(100), C.c_int64(4096), 64) >= 100 * 80 * 4
    assert L.spd_stats_rows(fake, C.c_int64(0), C.c_int64(10), C.c_int64(10), 0, fake, fake, C.c_size_t(1 << 20), None) == INV
    assert L.spd_stats_rows(fake, C.c_int64(4), C.c_int64(10), C.c_int64(10), 0, fake, fake, C.c_size_t(16), None) == WS
    assert L.spd_boxcar_snr_rows(fake, C.c_int64(4), C.c_int64(100), C.c_int64(100), fake, 101, 0, fake, fake, fake, C.c_size_t(1 << 20), None) == INV
    assert L.spd_boxcar_snr_rows(fake, C.c_int64(4), C.c_int64(100), C.c_int64(100), fake, 40, 1, fake, fake, fake, C.c_size_t(64), None) == WS
    assert L.spd_search_fused_rows(fake, C.c_int64(4), C.c_int64(100), C.c_int64(100), fake, 40, 0, C.c_float(float("nan")), fake, C.c_uint64(4), fake,
                                   fake, C.c_size_t(1 << 20), None) == INV


def test_search_host_decimated_validates_arguments(L):
    fake = C.c_void_p(4096)
    INV, WS = 1, 3
    ab = L.spd_search_host_decimated_arena_bytes
    assert ab(64, 16384, 16, 3, 1 << 12) >= 64 * 16384 * 4 + (16 << 12) + L.spd_decimated_workspace_bytes(C.c_int64(64), C.c_int64(16384), 16, 3)
    assert ab(64, 16384, 24, 3, 1 << 12) == 0 and ab(64, 16384, 32, 9, 1 << 12) == 0 and ab(0, 16384, 16, 3, 16) == 0
    f = L.spd_search_host_decimated
    assert f(None, 2, 4096, 16, 2, 0, 6.0, fake, 10, fake, None, fake, 1 << 30, None) == INV
    assert f(fake, 2, 4096, 16, 2, 0, 6.0, fake, 10, None, None, fake, 1 << 30, None) == INV
    assert f(fake, 2, 4096, 16, 2, 0, 6.0, None, 10, fake, None, fake, 1 << 30, None) == INV
    assert f(fake, 2, 4096, 24, 2, 0, 6.0, fake, 10, fake, None, fake, 1 << 30, None) == INV       # w0 must be 16 or 32
    assert f(fake, 2, 4096, 16, 2, 5, 6.0, fake, 10, fake, None, fake, 1 << 30, None) == INV       # bad mode
    assert f(fake, 2, 4096, 16, 2, 0, 6.0, fake, 10, fake, None, C.c_void_p(4097), 1 << 30, None) == INV   # arena alignment
    assert f(fake, 2, 4096, 16, 2, 0, 6.0, fake, 10, fake, None, fake, 1024, None) == WS
