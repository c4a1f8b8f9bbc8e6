"""-m gpu seeded fuzz: random shapes, pitches, alignments, tile sizes, pixel types and series lengths through
the C ABI against the oracle (the same tolerance as everywhere else).  Every case is reproducible from its index."""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

K = dict(C1=1e-6, C2=1e-6, C=1e-6, D=5e-7)
EXTRA = int(os.environ.get("IQA_FUZZ_EXTRA", "0"))      # soak runs: IQA_FUZZ_EXTRA=600 adds that many cases to every test


@pytest.fixture(scope="module")
def B():
    from paper_2501_10653_b200 import binding
    return binding


@pytest.fixture(scope="module")
def U():
    import gpu_util
    return gpu_util


def _window(a, pitch, off):
    import torch
    H, W = a.shape
    buf = torch.full((H * pitch + off + 16,), float("nan") if a.dtype.kind == "f" else 0, dtype=torch.from_numpy(a).dtype,
                     device="cuda")
    view = torch.as_strided(buf, (H, W), (pitch, 1), off)
    view.copy_(torch.from_numpy(a))
    return view


@pytest.mark.parametrize("case", range(48 + EXTRA))
def test_random_2d_cases(B, U, case):
    import torch
    import oracle
    rng = np.random.default_rng(1000 + case)
    H, W = int(rng.integers(1, 700)), int(rng.integers(1, 900))
    N_T = int(rng.choice([8, 16, 32, 64, 128, 256, 512, 5, 12, 24, 100]))
    aligned = rng.random() < 0.6
    pitch = W + int(rng.integers(0, 9))
    if aligned:
        pitch = -(-pitch // 4) * 4
    off = 0 if aligned else int(rng.integers(1, 4))
    dtype = np.dtype(rng.choice(["float32", "float32", "float32", "float64", "float16", "int16"]))
    if dtype.kind == "i":
        x = rng.integers(-50, 500, (H, W)).astype(dtype)
        y = rng.integers(-50, 500, (H, W)).astype(dtype)
        k = dict(C1=1e-3, C2=1e-3, C=1e-3, D=5e-4)
    else:
        x = rng.normal(0.05, 0.2, (H, W)).astype(dtype)
        y = rng.normal(0.05, 0.2, (H, W)).astype(dtype)
        k = K
    m = rng.random((H, W)) < 0.3
    y[m] = x[m]
    xd, yd = _window(x, pitch, off), _window(y, pitch, off)
    got = B.fused_tiles_2d(xd, yd, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    torch.cuda.synchronize()
    g = {n: v.cpu().numpy().astype(np.float64) for n, v in got.items()}
    ref = oracle.tiles_2d_any(x, y, N_T, **k)
    U.assert_parity(g, ref, k["C"], f"case {case}: {H}x{W} N_T={N_T} pitch={pitch} off={off} {dtype}")


@pytest.mark.parametrize("case", range(16 + EXTRA))
def test_random_series_cases(B, U, case):
    import torch
    import oracle
    rng = np.random.default_rng(2000 + case)
    H, W = int(rng.integers(8, 500)), int(rng.integers(8, 600))
    N_T = int(rng.choice([8, 16, 32, 64, 128, 256, 20]))
    M = int(rng.integers(2, 7))
    pitch = -(-(W + int(rng.integers(0, 9))) // 4) * 4
    mode = ["reference", "consecutive"][case % 2]
    imgs = [rng.normal(0.05, 0.2, (H, W)).astype(np.float32) for _ in range(M)]
    for j in range(1, M):
        m = rng.random((H, W)) < 0.3
        imgs[j][m] = imgs[j - 1][m]
    dev = [_window(a, pitch, 0) for a in imgs]
    got = B.series_tiles_2d(dev, mode, N_T, K["C1"], K["C2"], K["C"], K["D"], numerators=True)
    torch.cuda.synchronize()
    for c, (ix, iy) in enumerate(oracle.comparison_indices(M, mode)):
        ref = oracle.tiles_2d(imgs[ix], imgs[iy], N_T, **K)
        g = {n: got[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(g, ref, K["C"], f"series case {case}: {H}x{W} N_T={N_T} M={M} {mode} cmp {c}")
        exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], K["C2"], K["C"])
        w = got["whole"][c].cpu().numpy()
        assert abs(w[0] - exp[0]) <= 1e-5 * abs(exp[0]) and abs(w[1] - exp[1]) <= 1e-5 * abs(exp[1]) + 1e-6


@pytest.mark.parametrize("case", range(24 + EXTRA))
def test_random_typed_series_find_cases(B, U, case):
    """iqa_series_find_2d_typed on random windows: every pixel type, tile sides of any kind, row pitches with and
    without a tensor map (any_kernel in series item order / tma_kernel series modes / generic kernels pair by pair),
    then the candidate lists -- matrices against the oracle, lists against the oracle's selection on the device matrices."""
    import torch
    import oracle
    rng = np.random.default_rng(3000 + case)
    H, W = int(rng.integers(8, 400)), int(rng.integers(8, 500))
    N_T = int(rng.choice([8, 16, 64, 128, 4, 7, 20, 48, 100, 150]))
    M = int(rng.integers(2, 6))
    dtype = np.dtype(["float32", "float64", "float16", "int16", "int32", "uint8"][case % 6])
    per16 = 16 // dtype.itemsize
    pitch = W + int(rng.integers(0, 9))
    if rng.random() < 0.7:
        pitch = -(-pitch // per16) * per16
    off = int(rng.integers(0, per16)) if rng.random() < 0.4 else 0
    mode = ["reference", "consecutive"][(case // 6) % 2]
    if dtype.kind in "iu":
        lo = 0 if dtype == np.uint8 else -50
        imgs = [rng.integers(lo, 250, (H, W)).astype(dtype) for _ in range(M)]
        k = dict(C1=1e-3, C2=1e-3, C=1e-3, D=5e-4)
    else:
        imgs = [rng.normal(0.05, 0.2, (H, W)).astype(dtype) for _ in range(M)]
        k = K
    for j in range(1, M):
        m = rng.random((H, W)) < 0.5
        imgs[j][m] = imgs[j - 1][m]
    dev = [_window(a, pitch, off) for a in imgs]
    nty, ntx = -(-H // N_T), -(-W // N_T)
    kk = int(rng.integers(1, 40))
    index = ["auglisi", "lisi"][case % 2]
    plain = B.series_tiles_2d(dev, mode, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    thr = float(np.quantile(plain[index].cpu().numpy(), 0.3))
    out = B.find_transients_2d(dev, mode, N_T, k["C1"], k["C2"], k["C"], k["D"], k=kk, index=index, threshold=thr)
    torch.cuda.synchronize()
    what = f"find case {case}: {H}x{W} N_T={N_T} M={M} {mode} {dtype} pitch={pitch} off={off} k={kk}"
    for c, (ix, iy) in enumerate(oracle.comparison_indices(M, mode)):
        ref = oracle.tiles_2d_any(imgs[ix], imgs[iy], N_T, **k)
        g = {n: plain[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(g, ref, k["C"], what + f" cmp {c}")
        assert torch.equal(out[index][c], plain[index][c]), what
        mat = out[index][c].cpu().numpy()
        ei, ev = oracle.bottom_k(mat, kk)
        n_real = ei.size
        assert np.array_equal(out["candidates"][c].cpu().numpy()[:n_real], ei), what
        assert np.array_equal(out["candidate_values"][c].cpu().numpy()[:n_real], ev), what
        eb = oracle.below_threshold(mat, thr)
        assert int(out["below_counts"][c]) == eb.size, what
        assert np.array_equal(out["below"][c].cpu().numpy()[:eb.size], eb), what
