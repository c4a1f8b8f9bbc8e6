"""-m gpu parity tests of iqa_fused_tiles_2d (H x W, row pitch, edge tiles) against
oracle.tiles_2d, element by element on the same seeded buffers, through the C ABI.  Tolerance: that of
the square path (tests/gpu_util.py)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2501_10653_b200 import binding
    return binding


@pytest.fixture(scope="module")
def U():
    import gpu_util
    return gpu_util


K = dict(C1=1e-6, C2=1e-6, C=1e-6, D=5e-7)


def _pair(H, W, seed):
    rng = np.random.default_rng(seed)
    x = rng.normal(0.05, 0.2, (H, W)).astype(np.float32)
    y = rng.normal(0.05, 0.2, (H, W)).astype(np.float32)
    m = rng.random((H, W)) < 0.3
    y[m] = x[m]
    return x, y


def _window(a, pitch, off):
    """Device copy of `a` as a window of a wider buffer: row pitch `pitch` elements, first element `off`
    elements into the allocation (controls the alignment of the base pointer)."""
    import torch
    H, W = a.shape
    buf = torch.full((H * pitch + off + 16,), float("nan"), dtype=torch.float32, device="cuda")   # NaN around the window
    view = torch.as_strided(buf, (H, W), (pitch, 1), off)
    view.copy_(torch.from_numpy(a))
    return view


def _check(B, U, x, y, xd, yd, N_T, what):
    import torch
    import oracle
    got = B.fused_tiles_2d(xd, yd, N_T, K["C1"], K["C2"], K["C"], K["D"], numerators=True)
    torch.cuda.synchronize()
    g = {n: v.cpu().numpy().astype(np.float64) for n, v in got.items()}
    ref = oracle.tiles_2d(x, y, N_T, **K)
    U.assert_parity(g, ref, K["C"], what)
    # Eqs. 3-4 over the edge-tiled matrices == the oracle's aggregate
    agg = B.aggregate(got["lisi"], got["auglisi"], got["X"], got["Y"], K["C2"], K["C"]).cpu().numpy()
    exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], K["C2"], K["C"])
    assert abs(agg[0] - exp[0]) <= 1e-5 * abs(exp[0]) and abs(agg[1] - exp[1]) <= 1e-5 * abs(exp[1]) + 1e-6
    return g


@pytest.mark.parametrize("H,W,N_T,pitch", [
    (100, 130, 16, 132), (257, 513, 64, 516), (64, 64, 8, 64), (300, 300, 256, 300), (1000, 40, 32, 40),
    (513, 1027, 128, 1028), (33, 1500, 8, 1504), (700, 129, 512, 132), (2048, 2048, 64, 2048),
    (31, 31, 32, 32), (1, 4, 8, 4), (200, 1234, 64, 1236)])
def test_tma_path_shapes(B, U, H, W, N_T, pitch):
    """16-byte aligned windows, pitch % 4 == 0, power-of-two N_T: the TMA kernel; W need not be a multiple of 4;
    edge tiles right and bottom; split tiles with pieces wholly outside the image (700 x 129, N_T = 512)."""
    x, y = _pair(H, W, H + W)
    xd, yd = _window(x, pitch, 0), _window(y, pitch + 4, 8)          # different pitches for x and y
    assert xd.data_ptr() % 16 == 0 and yd.data_ptr() % 16 == 0
    _check(B, U, x, y, xd, yd, N_T, f"tma {H}x{W} N_T={N_T}")


@pytest.mark.parametrize("H,W,N_T,pitch,off", [
    (100, 130, 16, 131, 0), (257, 300, 64, 300, 1), (90, 70, 20, 72, 0), (300, 200, 150, 200, 0),
    (64, 64, 7, 67, 3)])
def test_generic_path_shapes(B, U, H, W, N_T, pitch, off):
    """Odd pitches, unaligned bases, tile sides that are not powers of two: the generic kernel."""
    x, y = _pair(H, W, H * 3 + W)
    xd, yd = _window(x, pitch, off), _window(y, pitch, off + 1)
    _check(B, U, x, y, xd, yd, N_T, f"generic {H}x{W} N_T={N_T}")


def test_2d_equals_square_entry_point_bitwise(B, U):
    """On a square, contiguous, divisible image the 2-D entry point runs the same kernel: bit-identical."""
    import torch
    x, y = _pair(512, 512, 9)
    xd, yd = U.to_dev(x), U.to_dev(y)
    for N_T in (16, 64, 256):
        a = B.fused_tiles(xd, yd, N_T, K["C1"], K["C2"], K["C"], K["D"], numerators=True)
        b = B.fused_tiles_2d(xd, yd, N_T, K["C1"], K["C2"], K["C"], K["D"], numerators=True)
        torch.cuda.synchronize()
        for n in a:
            assert torch.equal(a[n], b[n]), (N_T, n)


def test_window_of_a_config1_sky(B, U):
    """A 1000 x 1500 window cut out of a BASELINE.json config [1] sky (row pitch 2048), N_T = 64."""
    from paper_2501_10653_b200 import synth
    cfg = synth.CONFIGS[1]
    x, y, _ = synth.make_pair(cfg)
    xd, yd = U.to_dev(x), U.to_dev(y)
    r0, c0 = 512, 256                                          # 16-byte aligned window origin
    _check(B, U, x[r0:r0 + 1000, c0:c0 + 1500], y[r0:r0 + 1000, c0:c0 + 1500],
           xd[r0:r0 + 1000, c0:c0 + 1500], yd[r0:r0 + 1000, c0:c0 + 1500], 64, "cfg1 window")


def test_2d_error_codes(B):
    import torch
    x = torch.zeros((64, 64), dtype=torch.float32, device="cuda")
    o = [torch.zeros(64, dtype=torch.float32, device="cuda") for _ in range(4)]
    a = (K["C1"], K["C2"], K["C"], K["D"])
    assert B.iqa_fused_tiles_2d(x, x, 64, 64, 64, 64, 8, *a, *o) == B.IQA_OK
    assert B.iqa_fused_tiles_2d(x, x, 64, 64, 63, 64, 8, *a, *o) == B.IQA_ERR_SHAPE      # pitch < W
    assert B.iqa_fused_tiles_2d(x, x, 0, 64, 64, 64, 8, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_fused_tiles_2d(x, None, 64, 64, 64, 64, 8, *a, *o) == B.IQA_ERR_NULL
    assert B.iqa_fused_tiles_2d(x, x, 64, 64, 64, 64, 8, 0.0, K["C2"], K["C"], K["D"], *o) == B.IQA_ERR_PARAM
    assert B.iqa_fused_tiles_2d(x, x, 64, 64, 64, 64, 128, *a, *o) == B.IQA_ERR_WORKSPACE
    assert B.iqa_workspace_bytes_2d(65, 130, 128) == 2 * 4 * 16 and B.iqa_workspace_bytes_2d(65, 130, 64) == 0
    torch.cuda.synchronize()


@pytest.mark.parametrize("world", [1, 2, 3, 5])
def test_one_pair_sharded_by_bands_of_tile_rows(B, U, world):
    """`world` ranks each take a band of tile rows of ONE pair (run one after the other on
    this GPU -- no kernel waits on another), reduce it with iqa_aggregate_partial, the partial sums are
    added (the all-reduce), iqa_aggregate_finish gives the whole-image pair; bands stacked == the full matrices."""
    import torch
    import oracle
    from paper_2501_10653_b200 import shard
    H, W, N_T = 1000, 1536, 64
    x, y = _pair(H, W, 77)
    xd, yd = U.to_dev(x), U.to_dev(y)
    ref = oracle.tiles_2d(x, y, N_T, **K)
    n_total = ref["lisi"].size
    total = torch.zeros(4, dtype=torch.float64, device="cuda")
    stacked = {n: [] for n in ("lisi", "auglisi", "X", "Y")}
    for rank in range(world):
        r0, r1 = shard.band_rows(H, N_T, rank, world)
        out = shard.banded_pair(B, xd[r0:r1], yd[r0:r1], n_total, N_T, K["C1"], K["C2"], K["C"], K["D"], dist=None)
        part = B.aggregate_partial(out["lisi"], out["auglisi"], out["X"], out["Y"], K["C2"], K["C"])
        total += part
        for n in stacked:
            stacked[n].append(out[n])
    whole = B.aggregate_finish(total, n_total, K["C2"], K["C"]).cpu().numpy().astype(np.float64)
    got = {n: torch.cat(v, dim=0).cpu().numpy().astype(np.float64) for n, v in stacked.items()}
    U.assert_parity(got, ref, K["C"], f"bands world={world}")
    exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], K["C2"], K["C"])
    assert abs(whole[0] - exp[0]) <= 1e-5 * abs(exp[0]) and abs(whole[1] - exp[1]) <= 1e-5 * abs(exp[1]) + 1e-6
    # the partial sums themselves: against the oracle's per-tile values (double)
    c2, c = float(np.float32(K["C2"])), float(np.float32(K["C"]))
    e4 = np.array([np.sum(ref["lisi"] * (np.maximum(ref["X"], ref["Y"]) + c2)),
                   np.sum(ref["auglisi"] * (ref["X"] + ref["Y"] + c)), np.sum(ref["X"]), np.sum(ref["Y"])])
    assert np.all(np.abs(total.cpu().numpy() - e4) <= 1e-5 * np.abs(e4))


@pytest.mark.parametrize("H,W,N_T,pitch,off", [(300, 500, 64, 512, 0), (513, 260, 128, 260, 0), (100, 130, 16, 131, 1),
                                               (90, 70, 20, 72, 0)])
def test_batch_and_series_2d(B, U, H, W, N_T, pitch, off):
    """iqa_fused_batch_2d / iqa_series_tiles_2d (common pitch; TMA and generic paths) against oracle.tiles_2d."""
    import torch
    import oracle
    rng = np.random.default_rng(H + W)
    imgs = [rng.normal(0.05, 0.2, (H, W)).astype(np.float32) for _ in range(4)]
    imgs[2][: H // 2] = imgs[1][: H // 2]
    dev = [_window(a, pitch, off) for a in imgs]
    xs, ys = [dev[0], dev[2]], [dev[1], dev[3]]
    out = B.fused_batch_2d(xs, ys, N_T, K["C1"], K["C2"], K["C"], K["D"], numerators=True)
    torch.cuda.synchronize()
    for p, (ix, iy) in enumerate(((0, 1), (2, 3))):
        ref = oracle.tiles_2d(imgs[ix], imgs[iy], N_T, **K)
        got = {n: out[n][p].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(got, ref, K["C"], f"batch_2d pair {p}")
        exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], K["C2"], K["C"])
        w = out["whole"][p].cpu().numpy()
        assert abs(w[0] - exp[0]) <= 1e-5 * abs(exp[0]) and abs(w[1] - exp[1]) <= 1e-5 * abs(exp[1]) + 1e-6
    for mode in ("reference", "consecutive"):
        so = B.series_tiles_2d(dev, mode, N_T, K["C1"], K["C2"], K["C"], K["D"], numerators=True)
        torch.cuda.synchronize()
        for c, (ix, iy) in enumerate(oracle.comparison_indices(4, mode)):
            ref = oracle.tiles_2d(imgs[ix], imgs[iy], N_T, **K)
            got = {n: so[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
            U.assert_parity(got, ref, K["C"], f"series_2d {mode} {c}")


@pytest.mark.parametrize("dtype,lo,hi", [("float64", -0.2, 1.0), ("float16", -2.0, 8.0), ("int16", -300, 3000),
                                         ("int32", -1000, 1 << 20), ("uint8", 0, 255)])
@pytest.mark.parametrize("H,W,N_T", [(100, 130, 16), (257, 300, 64), (300, 200, 150), (64, 64, 8)])
def test_other_pixel_types(B, U, dtype, lo, hi, H, W, N_T):
    """iqa_fused_tiles_2d_typed against oracle.tiles_2d_any (pixels -> double exactly, Eqs. 1-2 in double)."""
    import torch
    import oracle
    rng = np.random.default_rng(H + W + N_T)
    dt = np.dtype(dtype)
    x = rng.uniform(lo, hi, (H, W)).astype(dt)
    y = rng.uniform(lo, hi, (H, W)).astype(dt)
    m = rng.random((H, W)) < 0.3
    y[m] = x[m]
    k = dict(C1=1e-3, C2=1e-3, C=1e-3, D=5e-4) if dt.kind in "iu" else K      # integer counts: C's of that scale
    xd, yd = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
    got = B.fused_tiles_2d(xd, yd, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    torch.cuda.synchronize()
    g = {n: v.cpu().numpy().astype(np.float64) for n, v in got.items()}
    ref = oracle.tiles_2d_any(x, y, N_T, **k)
    U.assert_parity(g, ref, k["C"], f"{dtype} {H}x{W} N_T={N_T}")


def test_fp64_pixels_keep_their_small_differences(B, U):
    """Doubles that differ by ~3e-7 (a few fp32 ulps, the order of C1): the kernel subtracts in fp64 and stays
    within 1e-5 of the oracle, where rounding the inputs to fp32 first is off by percents."""
    import torch
    import oracle
    rng = np.random.default_rng(4)
    x = rng.normal(0.5, 0.5, (128, 192))
    y = x + rng.normal(0.0, 3e-7, (128, 192))
    got = B.fused_tiles_2d(torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda(), 32, K["C1"], K["C2"], K["C"], K["D"],
                           numerators=True)
    torch.cuda.synchronize()
    g = {n: v.cpu().numpy().astype(np.float64) for n, v in got.items()}
    ref = oracle.tiles_2d_any(x, y, 32, **K)
    U.assert_parity(g, ref, K["C"], "fp64 small differences")
    rounded = oracle.tiles_2d(x.astype(np.float32), y.astype(np.float32), 32, **K)
    assert np.max(np.abs(rounded["L"] - ref["L"]) / ref["L"]) > 1e-3


def test_typed_error_codes(B):
    import torch
    x = torch.zeros((64, 64), dtype=torch.float64, device="cuda")
    o = [torch.zeros(64, dtype=torch.float32, device="cuda") for _ in range(4)]
    a = (K["C1"], K["C2"], K["C"], K["D"])
    assert B.iqa_fused_tiles_2d_typed(x, x, B.IQA_PIXEL_F64, 64, 64, 64, 64, 8, *a, *o) == B.IQA_OK
    assert B.iqa_fused_tiles_2d_typed(x, x, 9, 64, 64, 64, 64, 8, *a, *o) == B.IQA_ERR_SHAPE
    assert B.iqa_fused_tiles_2d_typed(x, None, B.IQA_PIXEL_F64, 64, 64, 64, 64, 8, *a, *o) == B.IQA_ERR_NULL
    assert B.iqa_fused_tiles_2d_typed(x.data_ptr() + 4, x, B.IQA_PIXEL_F64, 32, 32, 64, 64, 8, *a, *o) == B.IQA_ERR_ALIGN
    assert B.iqa_fused_tiles_2d_typed(x, x, B.IQA_PIXEL_F64, 64, 64, 64, 64, 128, *a, *o) == B.IQA_ERR_WORKSPACE
    torch.cuda.synchronize()


# ---------------------------------------------------------------------------------------------- any_kernel (iqa_any.cuh)
def _typed_pair(rng, H, W, dtype):
    dt = np.dtype(dtype)
    if dt.kind in "iu":
        lo, hi = (0, 255) if dt == np.uint8 else (-300, 3000) if dt == np.int16 else (-1000, 1 << 20)
        x = rng.integers(lo, hi, (H, W)).astype(dt)
        y = rng.integers(lo, hi, (H, W)).astype(dt)
        k = dict(C1=1e-3, C2=1e-3, C=1e-3, D=5e-4)
    else:
        x = rng.normal(0.05, 0.2, (H, W)).astype(dt)
        y = rng.normal(0.05, 0.2, (H, W)).astype(dt)
        k = K
    m = rng.random((H, W)) < 0.3
    y[m] = x[m]
    return x, y, k


def _typed_window(a, pitch, off):
    """Device copy of `a` (any pixel type) as a window of a wider buffer; the halo holds NaN (floats) or a large
    value (integers), so a stray read shows up in the sums."""
    import torch
    H, W = a.shape
    t = torch.from_numpy(a)
    fill = float("nan") if a.dtype.kind == "f" else (200 if a.dtype == np.uint8 else 30000)
    buf = torch.full((H * pitch + off + 64,), fill, dtype=t.dtype, device="cuda")
    view = torch.as_strided(buf, (H, W), (pitch, 1), off)
    view.copy_(t)
    return view


def _check_typed(B, U, x, y, xd, yd, N_T, k, what, plan="tma_any"):
    import torch
    import oracle
    ref = oracle.tiles_2d_any(x, y, N_T, **k)

    def run(tag):
        got = B.fused_tiles_2d(xd, yd, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
        torch.cuda.synchronize()
        g = {n: v.cpu().numpy().astype(np.float64) for n, v in got.items()}
        U.assert_parity(g, ref, k["C"], what + tag)
        return got

    if plan == "tma_any" and B.plan_name(xd, N_T) == "generic":
        # the plan sends shapes that fill few lanes of any_kernel to the 128-bit generic kernel: check that path as
        # the library takes it, then any_kernel itself on the same shape (IQA_FORCE_ANY)
        run(" (default plan: generic)")
        with B.knob("IQA_FORCE_ANY", 1):
            assert B.plan_name(xd, N_T) == "tma_any", what
            return run(" (forced any_kernel)"), ref
    if plan is not None:
        assert B.plan_name(xd, N_T) == plan, (what, B.plan_name(xd, N_T))
    return run(""), ref


ANY_SHAPES = [
    # H, W, N_T, pitch (elements), off (elements)       -- geometry of any_geometry() in the comment
    (480, 960, 48, 960, 0),        # kx = 2, one box per item
    (500, 700, 100, 704, 0),       # kx = 1, two boxes of 50 rows
    (500, 700, 100, 704, 3),       # base aligned to 4 bytes only: shifted tensor map
    (333, 777, 50, 780, 1),        # N_T % 4 != 0: lanes straddle two tiles
    (200, 300, 7, 304, 0),         # kx = 18, ky = 4: several tile rows per box, straddling lanes
    (64, 64, 4, 64, 0),            # smallest tile side: kx = 32, ky = 8
    (130, 130, 5, 132, 2),
    (257, 513, 12, 516, 0),        # kx = 10, ky = 2
    (300, 300, 20, 300, 0), (300, 300, 36, 300, 0), (200, 650, 65, 652, 0), (400, 400, 97, 400, 0),
    (260, 390, 127, 392, 0),       # three boxes, a ragged last one that overlaps its predecessor
    (300, 400, 129, 400, 0),       # split tiles: px = 2, py = 3 with ragged last pieces
    (450, 310, 150, 312, 0), (700, 900, 300, 900, 1), (1100, 1300, 1000, 1300, 0),
    (33, 1500, 24, 1500, 0), (1000, 40, 33, 40, 0), (1, 4, 6, 4, 0), (3, 1000, 100, 1000, 0),
]


@pytest.mark.parametrize("H,W,N_T,pitch,off", ANY_SHAPES)
def test_any_kernel_fp32_shapes(B, U, H, W, N_T, pitch, off):
    """fp32, tile sides that are not powers of two, bases aligned to 4 bytes only: any_kernel against oracle.tiles_2d."""
    rng = np.random.default_rng(H * 7 + W + N_T)
    x, y, k = _typed_pair(rng, H, W, "float32")
    xd, yd = _typed_window(x, pitch, off), _typed_window(y, pitch + 4, off)        # same offset inside the 16-byte line
    got, ref = _check_typed(B, U, x, y, xd, yd, N_T, k, f"any fp32 {H}x{W} N_T={N_T} off={off}")
    agg = B.aggregate(got["lisi"], got["auglisi"], got["X"], got["Y"], k["C2"], k["C"]).cpu().numpy()
    import oracle
    exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], k["C2"], k["C"])
    assert abs(agg[0] - exp[0]) <= 1e-5 * abs(exp[0]) and abs(agg[1] - exp[1]) <= 1e-5 * abs(exp[1]) + 1e-6


@pytest.mark.parametrize("dtype", ["float64", "float16", "int16", "int32", "uint8"])
@pytest.mark.parametrize("H,W,N_T", [(300, 500, 64), (257, 300, 48), (300, 333, 100), (200, 210, 50), (150, 200, 7),
                                     (400, 600, 256), (500, 300, 150), (64, 64, 8), (90, 1000, 16)])
def test_any_kernel_pixel_types(B, U, dtype, H, W, N_T):
    """Every pixel type through the TMA-fed any_kernel (row pitch a multiple of 16 bytes, base aligned to the element
    only) against oracle.tiles_2d_any."""
    rng = np.random.default_rng(H + 3 * W + N_T)
    x, y, k = _typed_pair(rng, H, W, dtype)
    per16 = 16 // x.dtype.itemsize
    pitch = -(-(W + 5) // per16) * per16
    for off in (0, 1, per16 - 1) if per16 > 2 else (0, 1):
        xd, yd = _typed_window(x, pitch, off), _typed_window(y, pitch + per16, off)
        _check_typed(B, U, x, y, xd, yd, N_T, k, f"any {dtype} {H}x{W} N_T={N_T} off={off}")
    with B.knob("IQA_ANY_NO_WIDE", 1):          # four columns per lane also where eight would fit (N_T % 8 == 0, aligned)
        xd, yd = _typed_window(x, pitch, 0), _typed_window(y, pitch + per16, 0)
        _check_typed(B, U, x, y, xd, yd, N_T, k, f"any {dtype} {H}x{W} N_T={N_T} narrow lanes")


@pytest.mark.parametrize("dtype", ["float32", "float64", "float16", "int16", "int32", "uint8"])
@pytest.mark.parametrize("H,W,N_T", [(257, 301, 64), (200, 333, 32), (130, 515, 150), (90, 77, 7), (64, 1001, 300),
                                     (300, 63, 16), (65, 129, 2), (40, 50, 3), (1, 5, 8), (100, 3, 64)])
def test_generic_vector_kernels(B, U, dtype, H, W, N_T):
    """Row pitches that are not multiples of 16 bytes (no tensor map), x and y aligned alike: the generic kernels with
    128-bit loads (iqa_generic_vec.cuh) -- a CTA per tile piece (split tiles included) or a warp per small tile,
    every base offset inside a 16-byte line, every pixel type -- and the scalar-load kernels on the same inputs
    (IQA_GENERIC_NO_VEC) against oracle.tiles_2d_any.  The halo of the windows holds NaN / large values."""
    import torch
    rng = np.random.default_rng(H * 5 + W + N_T)
    x, y, k = _typed_pair(rng, H, W, dtype)
    per16 = 16 // x.dtype.itemsize
    pitch = W + (1 if (W + 1) % per16 else 2)                       # never a multiple of 16 bytes
    assert pitch % per16 != 0 or N_T < 4
    for off in sorted({0, 1, per16 - 1, per16 + 1}):
        xd, yd = _typed_window(x, pitch, off), _typed_window(y, pitch + per16, off)   # equal pitches modulo 16 bytes
        got, _ = _check_typed(B, U, x, y, xd, yd, N_T, k, f"generic vec {dtype} {H}x{W} N_T={N_T} off={off}", plan="generic")
    with B.knob("IQA_GENERIC_NO_VEC", 1):
        sc, _ = _check_typed(B, U, x, y, xd, yd, N_T, k, f"generic scalar {dtype} {H}x{W} N_T={N_T}", plan="generic")
    for n in got:                                                    # same arithmetic, another summation order
        assert torch.all((got[n] - sc[n]).abs() <= 4e-6 * sc[n].abs() + 1e-30), n


def test_any_kernel_matches_tma_kernel_on_power_of_two_tiles(B, U):
    """IQA_FORCE_ANY sends a power-of-two shape through any_kernel: the same per-pixel arithmetic in another
    summation order, so the two kernels agree to a few ulps (and both with the oracle)."""
    import torch
    rng = np.random.default_rng(11)
    x, y, k = _typed_pair(rng, 1024, 1536, "float32")
    xd, yd = U.to_dev(x), U.to_dev(y)
    for N_T in (8, 16, 64, 128, 512):
        a = B.fused_tiles_2d(xd, yd, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
        with B.knob("IQA_FORCE_ANY", 1):
            assert B.plan_name(xd, N_T) == "tma_any"
            b, _ = _check_typed(B, U, x, y, xd, yd, N_T, k, f"forced any N_T={N_T}")          # eight columns per lane
            with B.knob("IQA_ANY_NO_WIDE", 1):
                c, _ = _check_typed(B, U, x, y, xd, yd, N_T, k, f"forced any, narrow lanes, N_T={N_T}")
        for n in a:
            assert torch.all((a[n] - b[n]).abs() <= 2e-6 * a[n].abs() + 1e-30), (N_T, n)
            assert torch.all((a[n] - c[n]).abs() <= 2e-6 * a[n].abs() + 1e-30), (N_T, n)


@pytest.mark.parametrize("dtype,N_T", [("float32", 100), ("int16", 64), ("float64", 48), ("uint8", 150)])
def test_typed_batch_and_series(B, U, dtype, N_T):
    """iqa_fused_batch_2d_typed (40 pairs: two launches of any_kernel) and iqa_series_tiles_2d_typed (pair by pair)."""
    import torch
    import oracle
    rng = np.random.default_rng(N_T)
    H, W = 210, 330
    per16 = 16 // np.dtype(dtype).itemsize
    pitch = -(-W // per16) * per16
    imgs, k = [], None
    for _ in range(6):
        a, _, k = _typed_pair(rng, H, W, dtype)
        imgs.append(a)
    dev = [_typed_window(a, pitch, 0) for a in imgs]
    order = [(i % 6, (i * 5 + 1) % 6) for i in range(40)]
    out = B.fused_batch_2d([dev[i] for i, _ in order], [dev[j] for _, j in order], N_T, k["C1"], k["C2"], k["C"], k["D"],
                           numerators=True)
    torch.cuda.synchronize()
    refs = {}
    for p, (i, j) in enumerate(order):
        if (i, j) not in refs:
            refs[(i, j)] = oracle.tiles_2d_any(imgs[i], imgs[j], N_T, **k)
        ref = refs[(i, j)]
        got = {n: out[n][p].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(got, ref, k["C"], f"typed batch {dtype} pair {p}")
        exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], k["C2"], k["C"])
        w = out["whole"][p].cpu().numpy()
        assert abs(w[0] - exp[0]) <= 1e-5 * abs(exp[0]) and abs(w[1] - exp[1]) <= 1e-5 * abs(exp[1]) + 1e-6
    for mode in ("reference", "consecutive"):
        so = B.series_tiles_2d(dev[:4], mode, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
        torch.cuda.synchronize()
        for c, (ix, iy) in enumerate(oracle.comparison_indices(4, mode)):
            ref = oracle.tiles_2d_any(imgs[ix], imgs[iy], N_T, **k)
            got = {n: so[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
            U.assert_parity(got, ref, k["C"], f"typed series {dtype} {mode} {c}")


@pytest.mark.parametrize("dtype,N_T", [("float32", 48), ("float32", 150), ("int32", 64), ("float64", 20)])
def test_typed_series_item_order(B, U, dtype, N_T):
    """A typed / odd-N_T series is ONE any_kernel launch per 32 comparisons in pair-minor item order (the comparisons of an
    image location on neighbouring CTAs, shared images from L2).  The order is scheduling only: bit-identical to the
    pair-major order, for 35 comparisons (two launches), split tiles included; first, 32nd and last comparison against
    the oracle in both modes."""
    import torch
    import oracle
    rng = np.random.default_rng(N_T + 1)
    H, W, M = 190, 330, 36
    per16 = 16 // np.dtype(dtype).itemsize
    pitch = -(-W // per16) * per16
    imgs, k = [], None
    for _ in range(M):
        a, _, k = _typed_pair(rng, H, W, dtype)
        imgs.append(a)
    dev = [_typed_window(a, pitch, 0) for a in imgs]
    for mode in ("reference", "consecutive"):
        with B.knob("IQA_FORCE_ANY", 1):                 # (the plan would send the split N_T = 150 to the generic kernel)
            assert B.plan_name(dev[0], N_T) == "tma_any"
            so = B.series_tiles_2d(dev, mode, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
            with B.knob("IQA_SERIES_PAIR_MAJOR", 1):
                pm = B.series_tiles_2d(dev, mode, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
        torch.cuda.synchronize()
        for n in so:
            assert torch.equal(so[n], pm[n]), (mode, n)
        idx = oracle.comparison_indices(M, mode)
        for c in (0, 31, 32, M - 2):
            ix, iy = idx[c]
            ref = oracle.tiles_2d_any(imgs[ix], imgs[iy], N_T, **k)
            got = {n: so[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
            U.assert_parity(got, ref, k["C"], f"series order {dtype} N_T={N_T} {mode} {c}")


@pytest.mark.parametrize("dtype,N,N_T", [(np.int16, 512, 64), (np.uint8, 500, 100), (np.float16, 384, 48), (np.int32, 256, 128),
                                         (np.float64, 256, 16)])
def test_typed_host_entry_points(B, U, dtype, N, N_T):
    """iqa_fused_host_typed / _async (FITS planes as stored): raw pixels uploaded and computed on as they are; the
    four per-tile arrays and Eqs. 3-4 against the oracle, through the blocking call and through a two-stream pipeline."""
    import torch
    import oracle
    rng = np.random.default_rng(int(N_T) + 5)
    pairs = [_typed_pair(rng, N, N, dtype) for _ in range(3)]
    k = pairs[0][2]
    names = ("lisi", "auglisi", "X", "Y")

    def check(out, out2, x, y, what):
        ref = oracle.tiles_2d_any(x, y, N_T, **k)
        U.assert_parity({n: out[n].numpy().astype(np.float64) for n in names}, {**{n: ref[n] for n in names}, "A": ref["A"]},
                        k["C"], what)
        exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], k["C2"], k["C"])
        assert abs(out2[0].item() - exp[0]) <= 1e-5 * abs(exp[0]) and abs(out2[1].item() - exp[1]) <= 1e-5 * abs(exp[1]) + 1e-7

    out, out2 = B.fused_host(pairs[0][0], pairs[0][1], N_T, **k)                     # pageable numpy input, blocking call
    check(out, out2, pairs[0][0], pairs[0][1], f"fused_host {np.dtype(dtype).name}")
    ptype = B._pixel_types()[torch.from_numpy(pairs[0][0]).dtype]
    pipe = B.HostPipeline(N, N_T, "cuda:0", depth=2, pixel_type=ptype)
    assert pipe.runners[0].h2d_bytes == 2 * np.dtype(dtype).itemsize * N * N
    pinned = [(torch.from_numpy(x).pin_memory(), torch.from_numpy(y).pin_memory()) for x, y, _ in pairs]
    for (xp, yp), (x, y, _) in zip(pinned, pairs):
        slot = pipe.submit(xp, yp, k["C1"], k["C2"], k["C"], k["D"])
        o, o2 = pipe.wait(slot)
        check(o, o2, x, y, f"host pipeline {np.dtype(dtype).name}")
    pipe.drain()


def test_small_jobs_keep_any_kernel(B, U):
    """The generic kernel runs one warp per piece of a tile, so it needs several pieces per SM to beat any_kernel's idle
    lanes: one pair of a 600 x 600 image with 150-pixel tiles is 16 tiles x 3 pieces = 48 warps for 148 SMs and stays on
    any_kernel (iqa_query_plan_n), a batch of 64 such pairs (3072 pieces) takes the generic kernel.  Both against the oracle."""
    import torch
    import oracle
    rng = np.random.default_rng(78)
    H, W, N_T = 600, 600, 150
    a, b, k = _typed_pair(rng, H, W, np.float32)
    da, db = _typed_window(a, W, 0), _typed_window(b, W, 0)
    ref = oracle.tiles_2d_any(a, b, N_T, **k)
    names = ("lisi", "auglisi", "X", "Y", "L", "A")
    with B.knob("IQA_PLAN_LARGE_JOB", 0):
        assert B.plan_name(da, N_T) == "generic"                       # a job that fills the GPU
        assert B.plan_name(da, N_T, n=1) == "tma_any" and B.plan_name(da, N_T, n=64) == "generic"
        one = B.fused_tiles_2d(da, db, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
        many = B.fused_batch_2d([da] * 64, [db] * 64, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    with B.knob("IQA_FORCE_ANY", 1):
        forced_any = B.fused_tiles_2d(da, db, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    with B.knob("IQA_FORCE_GENERIC", 1):
        forced_gen = B.fused_tiles_2d(da, db, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    for n in names:
        assert torch.equal(one[n], forced_any[n]), n                   # the single pair took any_kernel ...
        assert torch.equal(many[n][63], forced_gen[n]), n              # ... the batch the generic kernel
    for res, what in ((one, "one pair"), ({n: many[n][0] for n in names}, "batch of 64")):
        got = {n: res[n].cpu().numpy().astype(np.float64) for n in names}
        U.assert_parity(got, ref, k["C"], f"small-job rule, {what}")


def test_series_of_two_images_is_planned_like_the_pair_it_is(B, U):
    """A series of two snapshots shares nothing through L2, so its plan is the pair's plan: N_T = 150 (split tiles filling
    0.59 of any_kernel's lanes) takes the 128-bit generic kernel in both calls and the results agree bit for bit; three
    snapshots keep any_kernel's pair-minor order."""
    import torch
    rng = np.random.default_rng(77)
    H, W, N_T = 600, 600, 150
    a, b, k = _typed_pair(rng, H, W, np.float32)
    c, _, _ = _typed_pair(rng, H, W, np.float32)
    da, db, dc = (_typed_window(v, W, 0) for v in (a, b, c))
    assert B.plan_name(da, N_T) == "generic" and B.plan_name(da, N_T, series=True) == "tma_any"
    two = B.series_tiles_2d([da, db], "consecutive", N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    pair = B.fused_tiles_2d(da, db, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    for n in pair:
        assert torch.equal(two[n][0], pair[n]), n
    three = B.series_tiles_2d([da, db, dc], "consecutive", N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    import oracle
    for cmp_i, (u, v) in enumerate([(a, b), (b, c)]):
        ref = oracle.tiles_2d_any(u, v, N_T, **k)
        for res, what in ((three, "three"),) + (((two, "two"),) if cmp_i == 0 else ()):
            got = {n: res[n][cmp_i].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
            U.assert_parity(got, ref, k["C"], f"{what}-image series, comparison {cmp_i}")


@pytest.mark.parametrize("dtype,N_T", [("float32", 50), ("float32", 125), ("int16", 64), ("float64", 7)])
def test_generic_vector_kernel_batches_and_series(B, U, dtype, N_T):
    """The 128-bit generic kernel takes 32 pairs per launch: a batch of 40 pairs on a pitch no tensor map can describe
    (two launches; split tiles at N_T = 125: workspace [pair][tile][piece]) equals the pairs one by one bit for bit and the
    oracle; a series of 36 snapshots in pair-minor unit order equals the pair-major order bit for bit."""
    import torch
    import oracle
    rng = np.random.default_rng(N_T + 17)
    H, W = 250, 251
    per16 = 16 // np.dtype(dtype).itemsize
    pitch = W + (1 if (W + 1) % per16 else 2)
    imgs, k = [], None
    for _ in range(6):
        a, _, k = _typed_pair(rng, H, W, dtype)
        imgs.append(a)
    dev = [_typed_window(a, pitch, 0) for a in imgs]
    assert B.plan_name(dev[0], N_T) == "generic"
    order = [(i % 6, (i * 5 + 1) % 6) for i in range(40)]
    out = B.fused_batch_2d([dev[i] for i, _ in order], [dev[j] for _, j in order], N_T, k["C1"], k["C2"], k["C"], k["D"],
                           numerators=True)
    torch.cuda.synchronize()
    for p_, (i, j) in enumerate(order):
        if p_ in (0, 31, 32, 39):
            one = B.fused_tiles_2d(dev[i], dev[j], N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
            for n in one:
                assert torch.equal(one[n], out[n][p_]), (p_, n)
            ref = oracle.tiles_2d_any(imgs[i], imgs[j], N_T, **k)
            got = {n: out[n][p_].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
            U.assert_parity(got, ref, k["C"], f"generic batch {dtype} N_T={N_T} pair {p_}")
    series = [dev[i % 6] for i in range(36)]
    for mode in ("reference", "consecutive"):
        so = B.series_tiles_2d(series, mode, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
        with B.knob("IQA_SERIES_PAIR_MAJOR", 1):
            pm = B.series_tiles_2d(series, mode, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
        torch.cuda.synchronize()
        for n in so:
            assert torch.equal(so[n], pm[n]), (mode, n)
        for c, (ix, iy) in enumerate(oracle.comparison_indices(36, mode)):
            if c in (0, 33, 34):
                ref = oracle.tiles_2d_any(imgs[ix % 6], imgs[iy % 6], N_T, **k)
                got = {n: so[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
                U.assert_parity(got, ref, k["C"], f"generic series {dtype} N_T={N_T} {mode} {c}")


def test_paper_named_entry_points_with_odd_tile_sides(B, U):
    """iqa_lisi_tiles / iqa_auglisi_tiles / iqa_fused_tiles with N_T = 48 and 100 (N % N_T == 0): the three modes of
    any_kernel; the standalone results equal the fused ones bit for bit."""
    import torch
    rng = np.random.default_rng(5)
    for N, N_T in ((960, 48), (1200, 100), (1000, 250)):
        x, y, k = _typed_pair(rng, N, N, "float32")
        xd, yd = U.to_dev(x), U.to_dev(y)
        for force in (0, 1):                             # the library's plan (N_T = 250: generic kernel), then any_kernel
            with B.knob("IQA_FORCE_ANY", force):
                assert B.plan_name(xd, N_T) == ("generic" if N_T == 250 and not force else "tma_any")
                f, _, _ = U.check_pair(x, y, N_T, k, f"square any N_T={N_T} force={force}", xd=xd, yd=yd)
                fo = B.fused_tiles(xd, yd, N_T, **k)
                li = B.lisi_tiles(xd, yd, N_T, k["C1"], k["C2"], k["D"])
                au = B.auglisi_tiles(xd, yd, N_T, k["C"])
                assert torch.equal(li, fo["lisi"]) and torch.equal(au, fo["auglisi"])


def test_unaligned_bases(B, U):
    """Windows that start 1..3 elements into a 16-byte line.  Same offset for x and y (two windows cut at the same
    column): any_kernel loads from the 16-byte boundary below and shifts the column -> tile assignment.  Different
    offsets: no common column grid for the boxes, the generic kernel.  Both against the oracle, for a power-of-two
    and an odd tile side."""
    rng = np.random.default_rng(8)
    x, y, k = _typed_pair(rng, 512, 768, "float32")
    for N_T in (64, 100, 256):
        for off in (1, 2, 3):
            xd, yd = _typed_window(x, 768, off), _typed_window(y, 772, off)
            assert xd.data_ptr() % 16 == 4 * off
            _check_typed(B, U, x, y, xd, yd, N_T, k, f"shift {off} N_T={N_T}", plan="tma_any")
            yd2 = _typed_window(y, 772, (off + 1) % 4)
            _check_typed(B, U, x, y, xd, yd2, N_T, k, f"offsets {off}/{(off + 1) % 4} N_T={N_T}", plan=None)


@pytest.mark.parametrize("H,W,N_T", [(1000, 1536, 64), (1000, 1536, 48), (333, 2000, 8), (700, 129, 16), (64, 64, 64)])
def test_pyramid_of_a_rectangle_every_level(B, U, H, W, N_T):
    """iqa_pyramid on a rectangular nty x ntx tile matrix with edge tiles: level j merges 2^j x 2^j blocks, blocks over
    the border merge only the tiles that exist (Eq. 4's n is that count) -- so level j must equal
    oracle.tiles_2d at tile size 2^j N_T, for EVERY level up to the 1 x 1 top."""
    import torch
    import oracle
    x, y = _pair(H, W, H + N_T)
    xd, yd = U.to_dev(x), U.to_dev(y)
    base = B.fused_tiles_2d(xd, yd, N_T, K["C1"], K["C2"], K["C"], K["D"])
    levels = B.pyramid(base, K["C2"], K["C"])
    torch.cuda.synchronize()
    nty, ntx = -(-H // N_T), -(-W // N_T)
    assert len(levels) == 1 + B.iqa_pyramid_levels(nty, ntx)
    assert sum(l["lisi"].numel() for l in levels[1:]) == B.iqa_pyramid_tiles(nty, ntx)
    for j, level in enumerate(levels):
        ref = oracle.tiles_2d(x, y, N_T << j, **K)
        got = {n: level[n].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y")}
        U.assert_parity(got, ref, K["C"], f"pyramid {H}x{W} N_T={N_T} level {j}")
    assert tuple(levels[-1]["lisi"].shape) == (1, 1)
