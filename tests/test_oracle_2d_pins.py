"""Pins for the general H x W / pitched / edge-tile oracle (oracle.tiles_2d; SURVEY.md 8(f)-4,
DESIGN.md reading R18) -- CPU only.

  G1  zero padding: padding both images with zeros (or with negatives, which the clamp removes)
      up to a square multiple of N_T and calling the pinned SQUARE oracle gives the same sums bit for bit
  G2  exact-rational brute force (oracle/exact_rational.py) of every tile incl. the edge tiles
  G3  a pitched view (column / row slice of a wider array) equals its contiguous copy
  G4  on square divisible images tiles_2d == tiles; Eqs. 3-4 over the edge-tiled matrix == one big tile
  G5  hand-checked 3 x 5 example with N_T = 2 (edge tiles of 2x1, 1x2 and 1x1 pixels)
"""
import numpy as np
import pytest

import oracle
from oracle import exact_rational as er

K = dict(C1=1e-3, C2=1e-4, C=1e-5, D=5e-4)
NAMES = ("lisi", "auglisi", "X", "Y", "L", "A")


def _pair(H, W, seed):
    rng = np.random.default_rng(seed)
    x = rng.normal(0.2, 0.5, (H, W)).astype(np.float32)
    y = rng.normal(0.2, 0.5, (H, W)).astype(np.float32)
    m = rng.random((H, W)) < 0.25
    y[m] = x[m]
    return x, y


@pytest.mark.parametrize("H,W,N_T", [(5, 7, 2), (10, 10, 4), (9, 33, 8), (40, 17, 16), (3, 3, 8), (16, 24, 8)])
@pytest.mark.parametrize("fill", [0.0, -3.5])
def test_zero_padding_equals_the_square_oracle(H, W, N_T, fill):
    x, y = _pair(H, W, H * 100 + W)
    side = -(-max(H, W) // N_T) * N_T
    xp = np.full((side, side), fill, dtype=np.float32)
    yp = np.full((side, side), fill, dtype=np.float32)
    xp[:H, :W], yp[:H, :W] = x, y
    got = oracle.tiles_2d(x, y, N_T, **K)
    ref = oracle.tiles(xp, yp, N_T, **K)
    nty, ntx = -(-H // N_T), -(-W // N_T)
    assert got["lisi"].shape == (nty, ntx)
    for n in NAMES:
        assert np.array_equal(got[n], ref[n][:nty, :ntx]), n


@pytest.mark.parametrize("H,W,N_T", [(5, 7, 2), (6, 4, 4), (7, 9, 3)])
def test_edge_tiles_vs_exact_rational(H, W, N_T):
    x, y = _pair(H, W, 7 * H + W)
    got = oracle.tiles_2d(x, y, N_T, **K)
    kk = {n: np.float32(v) for n, v in K.items()}
    for ty in range(-(-H // N_T)):
        for tx in range(-(-W // N_T)):
            xs = x[ty * N_T:(ty + 1) * N_T, tx * N_T:(tx + 1) * N_T].tolist()
            ys = y[ty * N_T:(ty + 1) * N_T, tx * N_T:(tx + 1) * N_T].tolist()
            ref = er.lisi_auglisi(xs, ys, **kk)
            for n, v in zip(NAMES, ref):
                f = float(v)
                assert abs(got[n][ty, tx] - f) <= 1e-12 * max(abs(f), 1e-30) + 1e-15, (ty, tx, n)


def test_pitched_views_equal_contiguous_copies():
    rng = np.random.default_rng(5)
    big_x = rng.random((40, 64)).astype(np.float32)
    big_y = rng.random((48, 80)).astype(np.float32)
    xv, yv = big_x[3:33, 8:45], big_y[10:40, 20:57]            # 30 x 37 views, different pitches
    assert not xv.flags.c_contiguous and xv.strides[0] == 64 * 4 and yv.strides[0] == 80 * 4
    a = oracle.tiles_2d(xv, yv, 8, **K)
    b = oracle.tiles_2d(xv.copy(), yv.copy(), 8, **K)
    for n in NAMES:
        assert np.array_equal(a[n], b[n]), n


def test_square_divisible_case_and_aggregation():
    x, y = _pair(32, 32, 1)
    a, b = oracle.tiles_2d(x, y, 8, **K), oracle.tiles(x, y, 8, **K)
    for n in NAMES:
        assert np.array_equal(a[n], b[n]), n
    x, y = _pair(37, 53, 2)
    t = oracle.tiles_2d(x, y, 16, **K)                        # 3 x 4 tiles, edge tiles on both borders
    whole = oracle.tiles_2d(x, y, 64, **K)                    # one tile = the whole image
    agg = oracle.aggregate(t["lisi"], t["auglisi"], t["X"], t["Y"], K["C2"], K["C"])
    assert abs(agg[0] - whole["lisi"][0, 0]) <= 1e-12 * abs(whole["lisi"][0, 0])
    assert abs(agg[1] - whole["auglisi"][0, 0]) <= 1e-12 * abs(whole["auglisi"][0, 0])


def test_hand_checked_3x5():
    """N_T = 2 on 3 x 5: tiles (ty, tx) hold 2x2, 2x2, 2x1 / 1x2, 1x2, 1x1 pixels.
    x = all ones, y = all zeros except y[2, 4] = 1 (and a negative pixel that the clamp removes):
    every pixel with y = 0 has s = d = 1 -> L term 1/(1+C1), A term 1; the pixel (2, 4) has s = 2, d = 0."""
    x = np.ones((3, 5), dtype=np.float32)
    y = np.zeros((3, 5), dtype=np.float32)
    y[2, 4] = 1.0
    y[0, 0] = -7.0
    k = dict(C1=0.25, C2=0.5, C=0.125, D=2.0)
    t = oracle.tiles_2d(x, y, 2, **k)
    pix = np.array([[4, 4, 2], [2, 2, 1]], dtype=np.float64)
    assert np.array_equal(t["X"], pix)
    assert np.array_equal(t["Y"], np.array([[0, 0, 0], [0, 0, 1.0]]))
    assert np.array_equal(t["A"], np.array([[4, 4, 2], [2, 2, 0.0]]))
    expL = pix / 1.25
    expL[1, 2] = 2.0 / 0.25
    assert np.allclose(t["L"], expL, rtol=1e-15)
    assert np.allclose(t["lisi"], 2.0 * expL / (pix + 0.5), rtol=1e-15)
    expA = 1.0 - np.array([[4, 4, 2], [2, 2, 0.0]]) / (pix + np.array([[0, 0, 0], [0, 0, 1.0]]) + 0.125)
    assert np.allclose(t["auglisi"], expA, rtol=1e-15)
    with pytest.raises(ValueError):
        oracle.tiles_2d(x, y[:2], 2, **k)


# ----------------------------------------------------------------------------- other pixel types
def test_any_dtype_reduces_to_the_fp32_oracle_on_fp32_values():
    """T1: fp32 images through the double-input oracle == tiles_2d bit for bit (the fp32 routine is pinned above);
    fp16 / int16 / uint8 / int32 images == the same values stored as fp32 (all exactly representable)."""
    x, y = _pair(37, 53, 11)
    a, b = oracle.tiles_2d_any(x, y, 16, **K), oracle.tiles_2d(x, y, 16, **K)
    for n in NAMES:
        assert np.array_equal(a[n], b[n]), n
    rng = np.random.default_rng(3)
    for dt, lo, hi in ((np.int16, -300, 3000), (np.uint8, 0, 255), (np.int32, -1000, 1 << 20), (np.float16, -2, 8)):
        xi = rng.uniform(lo, hi, (20, 28)).astype(dt)
        yi = rng.uniform(lo, hi, (20, 28)).astype(dt)
        yi[:10] = xi[:10]
        a = oracle.tiles_2d_any(xi, yi, 8, **K)
        b = oracle.tiles_2d(xi.astype(np.float32), yi.astype(np.float32), 8, **K)
        for n in NAMES:
            assert np.array_equal(a[n], b[n]), (dt, n)
    with pytest.raises(ValueError):
        oracle.tiles_2d_any(x, y.astype(np.float64), 16, **K)


def test_fp64_pixels_vs_exact_rational_incl_ill_conditioned_differences():
    """T2: doubles whose differences (|x - y| ~ 3e-7) are of the order of C1 and only a few fp32 ulps of the
    values: the Eq. 1 term 2x/(|x-y|+C1) depends on that difference, so rounding the INPUTS to fp32 first
    (|x - y| off by up to an ulp, 6e-8) would be wrong by percents; exact rationals decide."""
    rng = np.random.default_rng(4)
    x = rng.normal(0.5, 0.5, (6, 8))
    y = x + rng.normal(0.0, 3e-7, (6, 8))
    y[0, :4] = rng.normal(0.5, 0.5, 4)
    x[5, 5] = -0.25
    k = dict(C1=1e-6, C2=1e-6, C=1e-6, D=5e-7)
    got = oracle.tiles_2d_any(x, y, 4, **k)
    kk = {n: np.float32(v) for n, v in k.items()}
    for ty in range(2):
        for tx in range(2):
            ref = er.lisi_auglisi(x[ty * 4:ty * 4 + 4, tx * 4:tx * 4 + 4].tolist(),
                                  y[ty * 4:ty * 4 + 4, tx * 4:tx * 4 + 4].tolist(), **kk)
            for n, v in zip(NAMES, ref):
                f = float(v)
                assert abs(got[n][ty, tx] - f) <= 1e-11 * max(abs(f), 1e-30) + 1e-15, (ty, tx, n)
    # and the fp32-rounded inputs give a visibly different LISI (the reason the kernel subtracts in fp64)
    lo = oracle.tiles_2d(x.astype(np.float32), y.astype(np.float32), 4, **k)
    assert np.max(np.abs(lo["L"] - got["L"]) / got["L"]) > 1e-3
