"""CPU-only checks of the C-ABI boundary: the library builds/loads, exports every symbol
include/iqa_tiles.h declares, and validates arguments BEFORE touching the device (so these
calls are safe without a GPU: nothing is enqueued when the status is not IQA_OK)."""
import ctypes
import math
import os
import re

import pytest

from paper_2501_10653_b200 import binding as B

ROOT = os.path.abspath(os.path.join(os.path.dirname(__file__), ".."))
HEADER = os.path.join(ROOT, "include", "iqa_tiles.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(iqa_[a-z_0-9]+)\s*\(", src)))


def test_library_is_in_tree_and_exports_every_declared_symbol():
    assert os.path.dirname(B.LIB_PATH) == os.path.join(ROOT, "paper_2501_10653_b200")
    names = _declared()
    assert set(names) == set(B.EXPORTS), names
    raw = ctypes.CDLL(B.LIB_PATH)
    for n in names:
        assert getattr(raw, n) is not None


def test_status_strings_and_version():
    seen = {B.iqa_status_string(s) for s in range(7)}
    assert len(seen) == 7 and "unknown status" not in seen
    assert B.iqa_status_string(99) == "unknown status"
    assert re.fullmatch(r"\d+\.\d+\.\d+", B.iqa_version())


def test_workspace_bytes():
    # tiles of side <= 64 are always finished inside one CTA: no second pass, no workspace
    for N, N_T in [(256, 16), (2048, 8), (2048, 64), (8192, 64), (10, 5), (192, 48)]:
        assert B.iqa_workspace_bytes(N, N_T) == 0
    # split tiles: 16 B per piece; the worst case over the kernels a call may take: tma_kernel cuts pieces of 128 x 64
    # pixels, any_kernel (unaligned bases, other pixel types) pieces of at most 112 x 64
    assert B.iqa_workspace_bytes(2048, 128) == 256 * 2 * 2 * 16
    assert B.iqa_workspace_bytes(2048, 512) == 16 * 5 * 8 * 16
    assert B.iqa_workspace_bytes(16384, 128) == 16384 * 4 * 16
    assert B.iqa_workspace_bytes(16384, 16384) == 147 * 256 * 16
    assert B.iqa_batch_workspace_bytes(16, 16384, 128) == 16 * 16384 * 4 * 16
    assert B.iqa_workspace_bytes(900, 300) == 9 * 3 * 5 * 16      # any_kernel: 3 x 5 pieces of 112 x 64
    assert B.iqa_batch_workspace_bytes(5, 2048, 64) == 0
    assert B.iqa_batch_workspace_bytes(0, 2048, 128) == 0
    assert B.iqa_workspace_bytes(200, 100) == 4 * 2 * 16          # generic: ceil(100/64) pieces
    # invalid shapes report 0 here; the entry points return the error
    for N, N_T in [(0, 8), (100, 0), (100, 7), (-4, 2), (64, 128), ((1 << 20) + 8, 8)]:
        assert B.iqa_workspace_bytes(N, N_T) == 0
        assert B.iqa_host_scratch_bytes(N, N_T) == 0
    assert B.iqa_host_scratch_bytes(256, 16) >= 2 * 256 * 256 * 4 + 4 * 256 * 4 + 8


FAKE = 0x1000   # a non-NULL, 16-byte aligned address that is never dereferenced on the host


def _fused(x=FAKE, y=FAKE, N=256, N_T=16, C1=1e-6, C2=1e-6, C=1e-6, D=5e-7,
           lisi=FAKE, aug=FAKE, sx=FAKE, sy=FAKE, ws=None, wsb=0):
    return B.iqa_fused_tiles(x, y, N, N_T, C1, C2, C, D, lisi, aug, sx, sy, None, None, ws, wsb, None)


def test_fused_argument_validation():
    assert _fused(x=None) == B.IQA_ERR_NULL
    assert _fused(y=None) == B.IQA_ERR_NULL
    assert _fused(lisi=None) == B.IQA_ERR_NULL
    assert _fused(aug=None) == B.IQA_ERR_NULL
    assert _fused(sx=None) == B.IQA_ERR_NULL
    assert _fused(sy=None) == B.IQA_ERR_NULL
    assert _fused(N=0) == B.IQA_ERR_SHAPE
    assert _fused(N=-256) == B.IQA_ERR_SHAPE
    assert _fused(N_T=0) == B.IQA_ERR_SHAPE
    assert _fused(N=100, N_T=16) == B.IQA_ERR_SHAPE          # P:64 presumes N % N_T == 0
    assert _fused(N=16, N_T=32) == B.IQA_ERR_SHAPE
    assert _fused(N=(1 << 20) + 16, N_T=16) == B.IQA_ERR_SHAPE
    assert _fused(N=1 << 20, N_T=1) == B.IQA_ERR_SHAPE       # 2^40 tiles do not fit an int index
    assert _fused(C1=1e-40) == B.IQA_ERR_PARAM               # subnormal C1: |x - y| + C1 would be flushed to zero
    assert _fused(C2=1e-40, C=1e-40, N=256, N_T=128) == B.IQA_ERR_WORKSPACE   # subnormal C2 / C are fine
    for bad in (0.0, -1e-6, math.inf, math.nan):
        assert _fused(C1=bad) == B.IQA_ERR_PARAM
        assert _fused(C2=bad) == B.IQA_ERR_PARAM
        assert _fused(C=bad) == B.IQA_ERR_PARAM
    assert _fused(D=math.nan) == B.IQA_ERR_PARAM
    assert _fused(D=math.inf) == B.IQA_ERR_PARAM
    assert _fused(x=FAKE + 2) == B.IQA_ERR_ALIGN
    assert _fused(y=FAKE + 1) == B.IQA_ERR_ALIGN
    assert _fused(N=256, N_T=128) == B.IQA_ERR_WORKSPACE     # split tiles need the workspace
    assert _fused(N=256, N_T=128, ws=FAKE, wsb=8) == B.IQA_ERR_WORKSPACE
    assert _fused(N=256, N_T=128, ws=FAKE + 4, wsb=1 << 20) == B.IQA_ERR_ALIGN


def test_standalone_and_aggregate_validation():
    assert B.iqa_lisi_tiles(None, FAKE, 256, 16, 1e-6, 1e-6, 5e-7, FAKE) == B.IQA_ERR_NULL
    assert B.iqa_lisi_tiles(FAKE, FAKE, 256, 16, 1e-6, 1e-6, 5e-7, None) == B.IQA_ERR_NULL
    assert B.iqa_lisi_tiles(FAKE, FAKE, 256, 24, 1e-6, 1e-6, 5e-7, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_lisi_tiles(FAKE, FAKE, 256, 16, 0.0, 1e-6, 5e-7, FAKE) == B.IQA_ERR_PARAM
    assert B.iqa_auglisi_tiles(FAKE, None, 256, 16, 1e-6, FAKE) == B.IQA_ERR_NULL
    assert B.iqa_auglisi_tiles(FAKE, FAKE, 256, 16, 1e-6, None) == B.IQA_ERR_NULL
    assert B.iqa_auglisi_tiles(FAKE, FAKE, 256, 16, -1.0, FAKE) == B.IQA_ERR_PARAM
    assert B.iqa_auglisi_tiles(FAKE, FAKE, 255, 16, 1e-6, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_aggregate(None, FAKE, FAKE, FAKE, 4, 1e-6, 1e-6, FAKE) == B.IQA_ERR_NULL
    assert B.iqa_aggregate(FAKE, FAKE, FAKE, FAKE, 4, 1e-6, 1e-6, None) == B.IQA_ERR_NULL
    assert B.iqa_aggregate(FAKE, FAKE, FAKE, FAKE, 0, 1e-6, 1e-6, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_aggregate(FAKE, FAKE, FAKE, FAKE, 4, 0.0, 1e-6, FAKE) == B.IQA_ERR_PARAM
    assert B.iqa_merge_tiles(FAKE, FAKE, FAKE, None, 8, 2, 1e-6, 1e-6, FAKE, FAKE, FAKE, FAKE) == B.IQA_ERR_NULL
    assert B.iqa_merge_tiles(FAKE, FAKE, FAKE, FAKE, 8, 3, 1e-6, 1e-6, FAKE, FAKE, FAKE, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_merge_tiles(FAKE, FAKE, FAKE, FAKE, 8, 0, 1e-6, 1e-6, FAKE, FAKE, FAKE, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_merge_tiles(FAKE, FAKE, FAKE, FAKE, 8, 2, 1e-6, math.nan, FAKE, FAKE, FAKE, FAKE) == B.IQA_ERR_PARAM
    assert B.iqa_merge_tiles_batch(FAKE, FAKE, FAKE, FAKE, 8, 2, 0, 1e-6, 1e-6, FAKE, FAKE, FAKE, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_merge_tiles_batch(FAKE, FAKE, FAKE, FAKE, 8, 2, 3, 1e-6, 1e-6, FAKE, None, FAKE, FAKE) == B.IQA_ERR_NULL
    assert B.iqa_fused_host(None, FAKE, 256, 16, 1e-6, 1e-6, 1e-6, 5e-7, None, None, None, None, None,
                            FAKE, 1 << 30) == B.IQA_ERR_NULL
    assert B.iqa_fused_host(FAKE, FAKE, 256, 16, 1e-6, 1e-6, 1e-6, 5e-7, None, None, None, None, None,
                            0x1000, 16) == B.IQA_ERR_WORKSPACE
    assert B.iqa_fused_host(FAKE, FAKE, 256, 16, 1e-6, 1e-6, 1e-6, 5e-7, None, None, None, None, None,
                            0x1010, 1 << 30) == B.IQA_ERR_ALIGN


def test_typed_host_validation():
    args = (1e-6, 1e-6, 1e-6, 5e-7, None, None, None, None, None)
    I16 = B.IQA_PIXEL_I16
    assert B.iqa_host_scratch_bytes_typed(256, 16, I16) >= 2 * 256 * 256 * 2 + 4 * 256 * 4 + 8
    assert B.iqa_host_scratch_bytes_typed(256, 16, I16) < B.iqa_host_scratch_bytes(256, 16)
    assert B.iqa_host_scratch_bytes_typed(256, 16, B.IQA_PIXEL_F32) == B.iqa_host_scratch_bytes(256, 16)
    assert B.iqa_host_scratch_bytes_typed(256, 16, 99) == 0 and B.iqa_host_scratch_bytes_typed(256, 24, I16) == 0
    for fn in (B.iqa_fused_host_typed, B.iqa_fused_host_typed_async):
        assert fn(None, FAKE, I16, 256, 16, *args, FAKE, 1 << 30) == B.IQA_ERR_NULL
        assert fn(FAKE, FAKE, I16, 256, 16, *args, None, 1 << 30) == B.IQA_ERR_NULL
        assert fn(FAKE, FAKE, 99, 256, 16, *args, FAKE, 1 << 30) == B.IQA_ERR_SHAPE
        assert fn(FAKE, FAKE, I16, 256, 24, *args, FAKE, 1 << 30) == B.IQA_ERR_SHAPE
        assert fn(FAKE, FAKE, I16, 256, 16, 0.0, *args[1:], FAKE, 1 << 30) == B.IQA_ERR_PARAM
        assert fn(FAKE, FAKE, I16, 256, 16, *args, FAKE, 16) == B.IQA_ERR_WORKSPACE
        assert fn(FAKE, FAKE, I16, 256, 16, *args, 0x1010, 1 << 30) == B.IQA_ERR_ALIGN


def test_batch_validation():
    tbl = (ctypes.c_void_p * 3)(FAKE, FAKE, FAKE)
    bad = (ctypes.c_void_p * 3)(FAKE, 0, FAKE)
    odd = (ctypes.c_void_p * 3)(FAKE, FAKE + 2, FAKE)

    def call(xs=tbl, ys=tbl, P=3, N=256, N_T=16, C=1e-6, lisi=FAKE, out2=None, ws=None, wsb=0):
        return B.iqa_fused_batch(xs, ys, P, N, N_T, 1e-6, 1e-6, C, 5e-7, lisi, FAKE, FAKE, FAKE,
                                 None, None, out2, ws, wsb, None)

    assert call(xs=None) == B.IQA_ERR_NULL
    assert call(ys=bad) == B.IQA_ERR_NULL                   # a NULL entry in the pointer table
    assert call(lisi=None) == B.IQA_ERR_NULL
    assert call(P=0) == B.IQA_ERR_SHAPE
    assert call(P=-1) == B.IQA_ERR_SHAPE
    assert call(N=100) == B.IQA_ERR_SHAPE
    assert call(N=1 << 20, N_T=32, P=3) == B.IQA_ERR_SHAPE  # 3 * 2^30 tiles do not fit an int index
    assert call(C=0.0) == B.IQA_ERR_PARAM
    assert call(xs=odd) == B.IQA_ERR_ALIGN
    assert call(N_T=128) == B.IQA_ERR_WORKSPACE
    need = B.iqa_batch_workspace_bytes(3, 256, 128)
    assert need == 3 * B.iqa_workspace_bytes(256, 128) > 0
    assert call(N_T=128, ws=FAKE, wsb=need - 1) == B.IQA_ERR_WORKSPACE


def test_series_and_candidate_validation():
    """Error paths of iqa_series_tiles / iqa_tiles_below / iqa_tiles_bottom_k: nothing is enqueued."""
    tbl = (ctypes.c_void_p * 3)(FAKE, FAKE, FAKE)
    bad = (ctypes.c_void_p * 3)(FAKE, 0, FAKE)
    odd = (ctypes.c_void_p * 3)(FAKE, FAKE + 2, FAKE)

    def call(imgs=tbl, M=3, mode=B.IQA_SERIES_REFERENCE, N=256, N_T=16, C=1e-6, lisi=FAKE, ws=None, wsb=0):
        return B.iqa_series_tiles(imgs, M, mode, N, N_T, 1e-6, 1e-6, C, 5e-7, lisi, FAKE, FAKE, FAKE,
                                  None, None, None, ws, wsb, None)

    assert call(imgs=None) == B.IQA_ERR_NULL
    assert call(imgs=bad) == B.IQA_ERR_NULL
    assert call(lisi=None) == B.IQA_ERR_NULL
    assert call(M=1) == B.IQA_ERR_SHAPE
    assert call(mode=2) == B.IQA_ERR_SHAPE
    assert call(N=100) == B.IQA_ERR_SHAPE
    assert call(C=0.0) == B.IQA_ERR_PARAM
    assert call(imgs=odd) == B.IQA_ERR_ALIGN
    assert call(N_T=128) == B.IQA_ERR_WORKSPACE
    assert B.iqa_series_workspace_bytes(3, 256, 128) == 2 * B.iqa_workspace_bytes(256, 128) > 0
    assert B.iqa_series_workspace_bytes(3, 256, 16) == 0 and B.iqa_series_workspace_bytes(1, 256, 128) == 0
    assert B.iqa_tiles_bottom_k(None, 16, 1, 4, FAKE) == B.IQA_ERR_NULL
    assert B.iqa_tiles_bottom_k(FAKE, 16, 1, 4, None) == B.IQA_ERR_NULL
    assert B.iqa_tiles_bottom_k(FAKE, 16, 1, 0, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_tiles_bottom_k(FAKE, 16, 1, 1025, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_tiles_bottom_k(FAKE, 0, 1, 4, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_tiles_below(None, 16, 1, 0.5, FAKE, 16, FAKE) == B.IQA_ERR_NULL
    assert B.iqa_tiles_below(FAKE, 16, 1, 0.5, FAKE, 16, None) == B.IQA_ERR_NULL
    assert B.iqa_tiles_below(FAKE, 16, 1, 0.5, None, 16, FAKE) == B.IQA_ERR_NULL
    assert B.iqa_tiles_below(FAKE, 16, 0, 0.5, FAKE, 16, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_tiles_below(FAKE, 16, 1, 0.5, FAKE, -1, FAKE) == B.IQA_ERR_SHAPE
    assert B.iqa_tiles_below(FAKE, 16, 1, math.nan, FAKE, 16, FAKE) == B.IQA_ERR_PARAM

    def find(imgs=tbl, M=3, N=256, N_T=16, index=B.IQA_FIND_AUGLISI, k=4, bi=FAKE, thr=0.5, li=FAKE, cap=8, cnt=FAKE):
        return B.iqa_series_find(imgs, M, B.IQA_SERIES_REFERENCE, N, N_T, 1e-6, 1e-6, 1e-6, 5e-7, FAKE, FAKE, FAKE, FAKE,
                                 None, None, None, None, 0, index, k, bi, None, thr, li, cap, cnt, None)

    # the candidate arguments are checked BEFORE the series is enqueued, then the series' own validation applies
    assert find(index=2) == B.IQA_ERR_SHAPE
    assert find(k=-1) == B.IQA_ERR_SHAPE and find(k=1025) == B.IQA_ERR_SHAPE and find(cap=-1) == B.IQA_ERR_SHAPE
    assert find(k=0, cnt=None) == B.IQA_ERR_NULL               # neither list asked for
    assert find(bi=None) == B.IQA_ERR_NULL
    assert find(li=None) == B.IQA_ERR_NULL
    assert find(thr=math.nan) == B.IQA_ERR_PARAM
    assert find(imgs=bad) == B.IQA_ERR_NULL
    assert find(N=100) == B.IQA_ERR_SHAPE
    assert find(N_T=128) == B.IQA_ERR_WORKSPACE
    tb = B.iqa_series_find_2d_typed(tbl, 3, B.IQA_SERIES_REFERENCE, B.IQA_PIXEL_I16, 64, 80, 80, 8, 1e-6, 1e-6, 1e-6, 5e-7,
                                    FAKE, FAKE, FAKE, FAKE, None, None, None, None, 0, 5, 4, FAKE, None, 0.5, FAKE, 8, FAKE)
    assert tb == B.IQA_ERR_SHAPE                                # index 5: rejected before anything else
    tb = B.iqa_series_find_2d_typed(tbl, 3, B.IQA_SERIES_REFERENCE, 9, 64, 80, 80, 8, 1e-6, 1e-6, 1e-6, 5e-7,
                                    FAKE, FAKE, FAKE, FAKE, None, None, None, None, 0, 1, 4, FAKE, None, 0.5, FAKE, 8, FAKE)
    assert tb == B.IQA_ERR_SHAPE                                # unknown pixel type: the series' own validation


def test_2d_validation():
    a = (1e-6, 1e-6, 1e-6, 5e-7)
    o = (FAKE, FAKE, FAKE, FAKE)
    assert B.iqa_fused_tiles_2d(None, FAKE, 64, 64, 64, 64, 8, *a, *o) == B.IQA_ERR_NULL
    assert B.iqa_fused_tiles_2d(FAKE, FAKE, 64, 64, 64, 64, 8, *a, FAKE, FAKE, FAKE, None) == B.IQA_ERR_NULL
    assert B.iqa_fused_tiles_2d(FAKE, FAKE, 64, 64, 63, 64, 8, *a, *o) == B.IQA_ERR_SHAPE      # pitch < W
    assert B.iqa_fused_tiles_2d(FAKE, FAKE, 64, 0, 64, 64, 8, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_fused_tiles_2d(FAKE, FAKE, 64, 64, 64, 64, 0, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_fused_tiles_2d(FAKE, FAKE, 64, 64, 64, 64, 8, 1e-6, -1.0, 1e-6, 5e-7, *o) == B.IQA_ERR_PARAM
    assert B.iqa_fused_tiles_2d(FAKE + 2, FAKE, 64, 64, 64, 64, 8, *a, *o) == B.IQA_ERR_ALIGN
    assert B.iqa_fused_tiles_2d(FAKE, FAKE, 100, 300, 300, 300, 128, *a, *o) == B.IQA_ERR_WORKSPACE
    assert B.iqa_workspace_bytes_2d(100, 300, 128) == 1 * 3 * 4 * 16
    assert B.iqa_workspace_bytes_2d(100, 300, 64) == 0 and B.iqa_workspace_bytes_2d(0, 300, 128) == 0
    tbl = (ctypes.c_void_p * 3)(FAKE, FAKE, FAKE)
    bad = (ctypes.c_void_p * 3)(FAKE, 0, FAKE)
    assert B.iqa_fused_batch_2d(tbl, bad, 3, 64, 80, 80, 8, *a, *o) == B.IQA_ERR_NULL
    assert B.iqa_fused_batch_2d(tbl, tbl, 3, 64, 80, 79, 8, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_fused_batch_2d(tbl, tbl, 3, 100, 300, 300, 128, *a, *o) == B.IQA_ERR_WORKSPACE
    assert B.iqa_series_tiles_2d(tbl, 3, 0, 64, 80, 80, 8, *a, FAKE, FAKE, FAKE, None) == B.IQA_ERR_NULL
    assert B.iqa_series_tiles_2d(tbl, 3, 5, 64, 80, 80, 8, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_series_tiles_2d(tbl, 1, 0, 64, 80, 80, 8, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_series_tiles_2d(bad, 3, 0, 64, 80, 80, 8, *a, *o) == B.IQA_ERR_NULL
    assert B.iqa_series_tiles_2d(tbl, 3, 0, 64, 80, 80, 8, 1e-6, 1e-6, 0.0, 5e-7, *o) == B.IQA_ERR_PARAM
    assert B.iqa_fused_tiles_2d_typed(FAKE, FAKE, 9, 64, 64, 64, 64, 8, *a, *o) == B.IQA_ERR_SHAPE          # unknown type
    assert B.iqa_fused_tiles_2d_typed(FAKE, None, B.IQA_PIXEL_I16, 64, 64, 64, 64, 8, *a, *o) == B.IQA_ERR_NULL
    assert B.iqa_fused_tiles_2d_typed(FAKE + 4, FAKE, B.IQA_PIXEL_F64, 64, 64, 64, 64, 8, *a, *o) == B.IQA_ERR_ALIGN
    assert B.iqa_fused_tiles_2d_typed(FAKE, FAKE, B.IQA_PIXEL_F16, 64, 64, 60, 64, 8, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_fused_tiles_2d_typed(FAKE, FAKE, B.IQA_PIXEL_F32, 64, 0, 64, 64, 8, *a, *o) == B.IQA_ERR_SHAPE
    F32, F64, U8 = B.IQA_PIXEL_F32, B.IQA_PIXEL_F64, B.IQA_PIXEL_U8
    assert B.iqa_query_plan(None, F32, 64, 64, 64, 8) == -1 and B.iqa_query_plan(FAKE, F32, 64, 64, 60, 8) == -1
    assert B.iqa_query_plan(FAKE, 17, 64, 64, 64, 8) == -1 and B.iqa_query_plan(FAKE + 4, F64, 64, 64, 64, 8) == -1
    assert B.iqa_query_plan(FAKE, F32, 64, 64, 64, 7) == B.IQA_PLAN_TMA_ANY       # tile side not a power of two
    assert B.iqa_query_plan(FAKE, F32, 64, 64, 64, 3) == B.IQA_PLAN_GENERIC       # N_T < 4
    assert B.iqa_query_plan(FAKE + 4, F32, 64, 64, 64, 8) == B.IQA_PLAN_TMA_ANY   # 4-byte aligned base: any_kernel
    assert B.iqa_query_plan(FAKE, F32, 64, 64, 64, 8) == B.IQA_PLAN_TMA + 1 and B.iqa_query_plan(FAKE, F32, 64, 64, 64, 8, 1) == B.IQA_PLAN_TMA
    assert B.iqa_query_plan(FAKE, F32, 64, 63, 63, 8) == B.IQA_PLAN_GENERIC       # pitch not a multiple of 16 bytes
    assert B.iqa_query_plan(FAKE, U8, 64, 60, 64, 8) == B.IQA_PLAN_TMA_ANY and B.iqa_query_plan(FAKE, U8, 64, 60, 60, 8) == B.IQA_PLAN_GENERIC
    assert B.iqa_query_plan(FAKE, F64, 64, 64, 66, 100) == B.IQA_PLAN_TMA_ANY
    # the square entry points keep the paper's divisibility requirement
    assert B.iqa_fused_tiles(FAKE, FAKE, 100, 64, *a, *o) == B.IQA_ERR_SHAPE


def test_pyramid_geometry_and_validation():
    assert B.iqa_pyramid_levels(1, 1) == 0 and B.iqa_pyramid_tiles(1, 1) == 0
    assert B.iqa_pyramid_levels(32, 32) == 5 and B.iqa_pyramid_tiles(32, 32) == 256 + 64 + 16 + 4 + 1
    assert B.iqa_pyramid_levels(16, 24) == 5            # 8x12, 4x6, 2x3, 1x2, 1x1
    assert B.iqa_pyramid_tiles(16, 24) == 96 + 24 + 6 + 2 + 1
    assert B.iqa_pyramid_levels(3, 1) == 2 and B.iqa_pyramid_tiles(3, 1) == 2 + 1
    assert B.iqa_pyramid_levels(0, 4) == 0 and B.iqa_pyramid_tiles(-1, 4) == 0
    o = (FAKE, FAKE, FAKE, FAKE)
    assert B.iqa_pyramid(None, FAKE, FAKE, FAKE, 4, 4, 1, 1e-6, 1e-6, *o) == B.IQA_ERR_NULL
    assert B.iqa_pyramid(FAKE, FAKE, FAKE, FAKE, 4, 4, 1, 1e-6, 1e-6, FAKE, FAKE, None, FAKE) == B.IQA_ERR_NULL
    assert B.iqa_pyramid(FAKE, FAKE, FAKE, FAKE, 0, 4, 1, 1e-6, 1e-6, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_pyramid(FAKE, FAKE, FAKE, FAKE, 4, 4, 0, 1e-6, 1e-6, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_pyramid(FAKE, FAKE, FAKE, FAKE, 4, 4, 1, 0.0, 1e-6, *o) == B.IQA_ERR_PARAM
    assert B.iqa_pyramid(FAKE, FAKE, FAKE, FAKE, 1, 1, 3, 1e-6, 1e-6, None, None, None, None) == B.IQA_OK   # nothing to emit


def test_typed_batch_series_validation_and_knobs():
    a = (1e-6, 1e-6, 1e-6, 5e-7)
    o = (FAKE, FAKE, FAKE, FAKE)
    tbl = (ctypes.c_void_p * 3)(FAKE, FAKE, FAKE)
    odd = (ctypes.c_void_p * 3)(FAKE, FAKE + 4, FAKE)
    I16, F64 = B.IQA_PIXEL_I16, B.IQA_PIXEL_F64
    assert B.iqa_fused_batch_2d_typed(tbl, None, 3, I16, 64, 80, 80, 8, *a, *o) == B.IQA_ERR_NULL
    assert B.iqa_fused_batch_2d_typed(tbl, tbl, 3, 11, 64, 80, 80, 8, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_fused_batch_2d_typed(tbl, tbl, 0, I16, 64, 80, 80, 8, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_fused_batch_2d_typed(tbl, odd, 3, F64, 64, 80, 80, 8, *a, *o) == B.IQA_ERR_ALIGN
    assert B.iqa_fused_batch_2d_typed(tbl, odd, 3, I16, 100, 300, 300, 128, *a, *o) == B.IQA_ERR_WORKSPACE
    assert B.iqa_series_tiles_2d_typed(tbl, 3, 7, I16, 64, 80, 80, 8, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_series_tiles_2d_typed(odd, 3, 0, F64, 64, 80, 80, 8, *a, *o) == B.IQA_ERR_ALIGN
    assert B.iqa_series_tiles_2d_typed(tbl, 3, 0, F64, 64, 80, 80, 8, 0.0, 1e-6, 1e-6, 5e-7, *o) == B.IQA_ERR_PARAM
    # knobs: unknown names are refused, known ones return the previous value and change the plan
    assert B.iqa_debug_knob("IQA_NO_SUCH_KNOB", 1) == -1
    assert B.iqa_query_plan(FAKE, B.IQA_PIXEL_F32, 64, 64, 64, 8) == B.IQA_PLAN_TMA + 1
    with B.knob("IQA_FORCE_ANY", 1):
        assert B.iqa_query_plan(FAKE, B.IQA_PIXEL_F32, 64, 64, 64, 8) == B.IQA_PLAN_TMA_ANY
        with B.knob("IQA_FORCE_GENERIC", 1):
            assert B.iqa_query_plan(FAKE, B.IQA_PIXEL_F32, 64, 64, 64, 8) == B.IQA_PLAN_GENERIC
    with B.knob("IQA_TMA_CONFIG", 3):
        assert B.iqa_query_plan(FAKE, B.IQA_PIXEL_F32, 64, 64, 64, 8) == B.IQA_PLAN_TMA + 3
    assert B.iqa_query_plan(FAKE, B.IQA_PIXEL_F32, 64, 64, 64, 8) == B.IQA_PLAN_TMA + 1
    # plan rule of any_kernel (no GPU needed): shapes that would fill few of its lanes go to the 128-bit generic kernel
    F32, U8 = B.IQA_PIXEL_F32, B.IQA_PIXEL_U8
    q = lambda ptr, pt, nt: B.iqa_query_plan(ptr, pt, 4096, 4096, 4096, nt)
    assert q(FAKE, F32, 100) == B.IQA_PLAN_TMA_ANY and q(FAKE, F32, 330) == B.IQA_PLAN_TMA_ANY
    assert q(FAKE, F32, 120) == B.IQA_PLAN_GENERIC and q(FAKE, F32, 200) == B.IQA_PLAN_GENERIC       # split, fill < 0.8
    assert q(FAKE + 4, F32, 64) == B.IQA_PLAN_GENERIC and q(FAKE + 4, F32, 100) == B.IQA_PLAN_TMA_ANY
    assert q(FAKE, I16, 200) == B.IQA_PLAN_GENERIC and q(FAKE, I16, 64) == B.IQA_PLAN_TMA_ANY        # 2-byte split tiles
    assert q(FAKE, F64, 330) == B.IQA_PLAN_TMA_ANY and q(FAKE, F64, 170) == B.IQA_PLAN_GENERIC
    assert q(FAKE, U8, 16) == B.IQA_PLAN_TMA_ANY                                                   # small tiles stay
    with B.knob("IQA_FORCE_ANY", 1):
        assert q(FAKE, F32, 120) == B.IQA_PLAN_TMA_ANY
    assert not B.STALE                                       # the library under test was built from the sources in the tree


def test_convenience_wrappers_refuse_cpu_tensors():
    """No CPU fallback: the product path fails loudly on host tensors."""
    torch = pytest.importorskip("torch")
    x = torch.zeros((16, 16))
    with pytest.raises(ValueError):
        B.fused_tiles(x, x, 8, 1e-6, 1e-6, 1e-6, 5e-7)


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2501_10653_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), fn
                assert "liboracle" not in src and "iqa_oracle" not in src, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".cpp")):
            src = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_2501_10653_b200." not in src and "import paper_2501_10653_b200" not in src, fn
