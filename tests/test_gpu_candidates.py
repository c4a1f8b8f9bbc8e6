"""-m gpu parity tests of candidate extraction (iqa_tiles_below, iqa_tiles_bottom_k)
against oracle/series.py: index work, so the bar is BIT-EXACT indices and values.

Inputs are seeded and never come from the CUDA path: random fp32 matrices with many ties, and the
ORACLE's augLISI / LISI matrices (cast to fp32) of BASELINE.json skies.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2501_10653_b200 import binding
    return binding


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def _check_bottom_k(B, maps, k):
    import torch
    import oracle
    idx, val = B.tiles_bottom_k(_dev(maps), k)
    torch.cuda.synchronize()
    idx, val = idx.cpu().numpy(), val.cpu().numpy()
    for m in range(maps.shape[0]):
        ei, ev = oracle.bottom_k(maps[m], k)
        kk = ei.size
        assert np.array_equal(idx[m, :kk], ei), (m, k)
        assert np.array_equal(val[m, :kk], ev), (m, k)
        assert np.all(idx[m, kk:] == -1) and np.all(np.isposinf(val[m, kk:]))


def _check_below(B, maps, thr, capacity=None):
    import torch
    import oracle
    idx, cnt = B.tiles_below(_dev(maps), thr, capacity)
    torch.cuda.synchronize()
    idx, cnt = idx.cpu().numpy(), cnt.cpu().numpy()
    cap = idx.shape[1]
    for m in range(maps.shape[0]):
        e = oracle.below_threshold(maps[m], thr)
        assert cnt[m] == e.size, (m, thr)
        w = min(cap, e.size)
        assert np.array_equal(idx[m, :w], e[:w])
        assert np.all(idx[m, w:] == -1)          # untouched entries keep the wrapper's fill


@pytest.mark.parametrize("nt,n_maps,k", [(4, 1, 3), (16, 3, 16), (16, 2, 256), (32, 4, 1), (64, 2, 100),
                                         (128, 2, 1024), (256, 1, 777), (5, 2, 64), (33, 3, 1000)])
def test_bottom_k_random_with_ties(B, nt, n_maps, k):
    rng = np.random.default_rng(nt * 1000 + k)
    maps = np.round(rng.random((n_maps, nt, nt)), 2).astype(np.float32)      # two decimals: many ties
    maps[0].ravel()[:: 7] = -0.0
    maps[-1].ravel()[1:: 5] = 0.0
    maps[0].ravel()[3] = -1.5
    _check_bottom_k(B, maps, k)


@pytest.mark.parametrize("nt,n_maps,k", [(150, 2, 40), (181, 1, 1024), (300, 2, 7), (362, 1, 500), (363, 1, 100), (256, 3, 64)])
def test_bottom_k_large_matrices(B, nt, n_maps, k):
    """More than 16384 tiles: a thread-block cluster of 2..8 CTAs per matrix (n <= 131072), the single-CTA loop above
    that (nt = 363) and when IQA_CAND_NO_CLUSTER is set -- all three must give the oracle's list, ties included."""
    rng = np.random.default_rng(nt + k)
    maps = (0.99 + 0.01 * np.round(rng.random((n_maps, nt, nt)), 3)).astype(np.float32)     # clustered values, many ties
    maps[0].ravel()[:: 1013] = 0.5
    maps[-1].ravel()[-1] = 0.25                                                             # the very last tile
    _check_bottom_k(B, maps, k)
    for thr, cap in ((0.9925, None), (0.6, 10), (2.0, 1000)):
        _check_below(B, maps, thr, cap)
    with B.knob("IQA_CAND_NO_CLUSTER", 1):
        _check_bottom_k(B, maps, k)
        _check_below(B, maps, 0.9925)


def test_bottom_k_all_equal_and_sorted_inputs(B):
    maps = np.stack([np.full((16, 16), 0.25, np.float32),
                     np.arange(256, dtype=np.float32).reshape(16, 16),
                     np.arange(256, dtype=np.float32)[::-1].reshape(16, 16).copy(),
                     -np.arange(256, dtype=np.float32).reshape(16, 16)])
    for k in (1, 5, 255, 256, 300):
        _check_bottom_k(B, maps, k)


@pytest.mark.parametrize("nt,n_maps,k", [(128, 3, 32), (128, 2, 17), (127, 2, 32), (5, 3, 7), (100, 2, 1), (64, 4, 16),
                                         (90, 2, 31), (23, 5, 32)])
def test_bottom_k_small_k_path(B, nt, n_maps, k):
    """k <= 32 on a matrix of at most 16384 tiles takes the threshold-by-thread-minima path (no radix passes): random
    values with ties, map bases that are not 16-byte aligned (odd nt), and the adversarial layouts of that path -- all
    the lowest values inside ONE thread's run of 16 tiles, sorted and reversed matrices, all-equal matrices, NaN."""
    rng = np.random.default_rng(7 * nt + k)
    maps = np.round(rng.random((n_maps, nt, nt)), 3).astype(np.float32)
    maps[0].ravel()[:: 11] = -0.0
    if nt * nt >= 48:
        maps[-1].ravel()[32:48] = np.linspace(-2.0, -1.0, 16, dtype=np.float32)     # the lowest 16 in one thread's run
    _check_bottom_k(B, maps, k)
    n = nt * nt
    ramp = np.arange(n, dtype=np.float32)
    special = np.stack([ramp.reshape(nt, nt), ramp[::-1].reshape(nt, nt).copy(),
                        np.full((nt, nt), 0.5, np.float32), (ramp % 3).reshape(nt, nt)])
    _check_bottom_k(B, special, k)
    withnan = maps.copy()
    withnan[0].ravel()[1::4] = np.nan                      # NaN sorts last (never produced by the kernels: C2, C > 0)
    import torch
    idx, _ = B.tiles_bottom_k(_dev(withnan), k)
    torch.cuda.synchronize()
    got = idx.cpu().numpy()[0]
    flat = withnan[0].ravel()
    order = np.lexsort((np.arange(n), np.where(np.isnan(flat), np.inf, flat + 0.0)))
    finite = order[~np.isnan(flat[order])]
    kk = min(k, finite.size)
    assert np.array_equal(got[:kk], finite[:kk])


@pytest.mark.parametrize("thr", [-1.0, 0.0, 0.25, 0.5, 0.99, 2.0])
def test_below_threshold_random(B, thr):
    rng = np.random.default_rng(3)
    maps = np.round(rng.random((3, 40, 40)), 2).astype(np.float32)
    maps[1].ravel()[::9] = -0.0
    _check_below(B, maps, thr)
    _check_below(B, maps, thr, capacity=10)
    _check_below(B, maps, thr, capacity=0)


def test_candidates_on_oracle_matrices_of_config1(B):
    """The matrices of BASELINE.json config [1] (computed by the ORACLE, cast to fp32) and of the N_T = 8
    sweep point (65 536 tiles): bottom-k and thresholds as a finder would use them."""
    import oracle
    from paper_2501_10653_b200 import synth
    cfg = synth.CONFIGS[1]
    x, y, _ = synth.make_pair(cfg)
    for N_T in (64, 8):
        t = oracle.tiles(x, y, N_T, cfg.C1, cfg.C2, cfg.C, cfg.D)
        maps = np.stack([t["auglisi"], t["lisi"]]).astype(np.float32)
        for k in (5, 64, 1024):
            _check_bottom_k(B, maps, k)
        for thr in (float(np.quantile(maps[0], 0.01)), 0.999, 1.0):
            _check_below(B, maps, thr)


@pytest.mark.parametrize("mode,index", [("reference", "auglisi"), ("consecutive", "lisi")])
def test_find_transients_end_to_end(B, mode, index):
    """iqa_series_find: series -> bottom-k and threshold list inside ONE call.  The lists are exactly the oracle's
    selection on the device matrix of each comparison, the matrices are those of iqa_series_tiles, and the switched-off
    transients of a config-[0] series are among the flagged tiles."""
    import torch
    import oracle
    from paper_2501_10653_b200 import synth
    cfg = synth.CONFIGS[0]
    imgs, meta = synth.make_series(cfg, 4)
    dev = [torch.from_numpy(a).cuda() for a in imgs]
    plain = B.series_tiles(dev, mode, cfg.N_T, cfg.C1, cfg.C2, cfg.C, cfg.D)
    thr = float(np.quantile(plain[index].cpu().numpy(), 0.02))
    out = B.find_transients(dev, mode, cfg.N_T, cfg.C1, cfg.C2, cfg.C, cfg.D, k=12, index=index, threshold=thr,
                            capacity=20)
    torch.cuda.synchronize()
    for nm in ("lisi", "auglisi", "X", "Y", "whole"):
        assert torch.equal(out[nm], plain[nm]), nm
    cand = out["candidates"].cpu().numpy()
    mats = out[index].cpu().numpy()
    below, counts = out["below"].cpu().numpy(), out["below_counts"].cpu().numpy()
    nt = cfg.N // cfg.N_T
    src, ch = meta["sources"], meta["changed"]
    for c in range(3):
        ei, ev = oracle.bottom_k(mats[c], 12)            # selection is exact on the same fp32 matrix
        assert np.array_equal(cand[c], ei)
        assert np.array_equal(out["candidate_values"][c].cpu().numpy(), ev)
        eb = oracle.below_threshold(mats[c], thr)
        assert counts[c] == eb.size
        w = min(eb.size, 20)
        assert np.array_equal(below[c, :w], eb[:w]) and np.all(below[c, w:] == -1)
        if mode == "reference" and index == "auglisi":
            off = [i for i, s in zip(ch, meta["state_y"][c + 1]) if s and src["amp_x"][i] > 10 * cfg.noise_sigma]
            tiles = {int(src["cy"][i]) // cfg.N_T * nt + int(src["cx"][i]) // cfg.N_T for i in off}
            assert tiles <= set(cand[c].tolist()), (c, tiles, cand[c])
    only_k = B.find_transients(dev, mode, cfg.N_T, cfg.C1, cfg.C2, cfg.C, cfg.D, k=5, index=index)
    assert "below" not in only_k and torch.equal(only_k["candidates"], out["candidates"][:, :5])


@pytest.mark.parametrize("N,N_T,k", [(2048, 16, 16), (2048, 16, 40), (2048, 8, 16), (1024, 64, 32)])
def test_series_find_lists_match_oracle_selection(B, N, N_T, k):
    """iqa_series_find on 16384-tile matrices (both lists from ONE launch of the candidate kernel, small-k and radix
    paths), on 65536-tile matrices (cluster kernels, two launches) and on 256-tile matrices: the lists are the
    oracle's selection on the device matrices, which are those of iqa_series_tiles."""
    import torch
    import oracle
    g = torch.Generator(device="cuda").manual_seed(N + N_T + k)
    imgs = [torch.rand((N, N), generator=g, device="cuda") - 0.3 for _ in range(3)]
    imgs[2][: N // 2] = imgs[1][: N // 2]                      # half of the tiles of comparison 1 are identical: ties at 1.0
    kw = dict(C1=1e-3, C2=1e-3, C=1e-3, D=5e-4)
    plain = B.series_tiles(imgs, "consecutive", N_T, **kw)
    mats = plain["auglisi"].cpu().numpy()
    thr = float(np.quantile(mats[0], 0.003))
    out = B.find_transients(imgs, "consecutive", N_T, k=k, threshold=thr, capacity=64, **kw)
    torch.cuda.synchronize()
    assert torch.equal(out["auglisi"], plain["auglisi"]) and torch.equal(out["whole"], plain["whole"])
    for c in range(2):
        ei, ev = oracle.bottom_k(mats[c], k)
        assert np.array_equal(out["candidates"][c].cpu().numpy(), ei), c
        assert np.array_equal(out["candidate_values"][c].cpu().numpy(), ev), c
        eb = oracle.below_threshold(mats[c], thr)
        assert int(out["below_counts"][c]) == eb.size
        w = min(eb.size, 64)
        assert np.array_equal(out["below"][c].cpu().numpy()[:w], eb[:w])


@pytest.mark.parametrize("dtype,N_T", [("int16", 64), ("float32", 48), ("uint8", 20)])
def test_series_find_2d_typed(B, dtype, N_T):
    """iqa_series_find_2d_typed on H x W windows of other pixel types (any_kernel in series item order, then the candidate
    kernel): matrices equal to iqa_series_tiles_2d_typed, lists equal to the oracle's selection on them."""
    import torch
    import oracle
    rng = np.random.default_rng(N_T)
    H, W, M = 700, 1000, 5
    dt = np.dtype(dtype)
    per16 = 16 // dt.itemsize
    pitch = -(-W // per16) * per16
    base = rng.integers(0, 200, (H, W)) if dt.kind in "iu" else rng.normal(0.05, 0.2, (H, W))
    dev = []
    for m in range(M):
        a = base.copy()
        a[100 * m:100 * m + 40, 150 * m:150 * m + 40] = 0          # a source switched off somewhere else in every snapshot
        buf = torch.zeros((H, pitch), dtype=getattr(torch, dtype), device="cuda")
        buf[:, :W].copy_(torch.from_numpy(a.astype(dt)))
        dev.append(buf[:, :W])
    kw = dict(C1=1e-3, C2=1e-3, C=1e-3, D=5e-4)
    plain = B.series_tiles_2d(dev, "consecutive", N_T, **kw)
    mats = plain["auglisi"].cpu().numpy()
    thr = float(np.quantile(mats[0], 0.05))
    out = B.find_transients_2d(dev, "consecutive", N_T, k=9, threshold=thr, capacity=30, **kw)
    torch.cuda.synchronize()
    assert torch.equal(out["auglisi"], plain["auglisi"]) and torch.equal(out["whole"], plain["whole"])
    for c in range(M - 1):
        ei, ev = oracle.bottom_k(mats[c], 9)
        assert np.array_equal(out["candidates"][c].cpu().numpy(), ei), c
        assert np.array_equal(out["candidate_values"][c].cpu().numpy(), ev), c
        eb = oracle.below_threshold(mats[c], thr)
        assert int(out["below_counts"][c]) == eb.size
        w = min(eb.size, 30)
        assert np.array_equal(out["below"][c].cpu().numpy()[:w], eb[:w])


def test_candidate_error_codes(B):
    import torch
    v = torch.zeros((4, 4), dtype=torch.float32, device="cuda")
    i = torch.zeros(16, dtype=torch.int32, device="cuda")
    c = torch.zeros(1, dtype=torch.int32, device="cuda")
    assert B.iqa_tiles_bottom_k(v, 16, 1, 4, i) == B.IQA_OK
    assert B.iqa_tiles_bottom_k(v, 16, 1, 0, i) == B.IQA_ERR_SHAPE
    assert B.iqa_tiles_bottom_k(v, 16, 1, 1025, i) == B.IQA_ERR_SHAPE
    assert B.iqa_tiles_bottom_k(None, 16, 1, 4, i) == B.IQA_ERR_NULL
    assert B.iqa_tiles_below(v, 16, 1, 0.5, i, 16, c) == B.IQA_OK
    assert B.iqa_tiles_below(v, 16, 1, float("nan"), i, 16, c) == B.IQA_ERR_PARAM
    assert B.iqa_tiles_below(v, 16, 1, 0.5, None, 16, c) == B.IQA_ERR_NULL
    assert B.iqa_tiles_below(v, 16, 1, 0.5, None, 0, c) == B.IQA_OK
    assert B.iqa_tiles_below(v, 0, 1, 0.5, i, 16, c) == B.IQA_ERR_SHAPE
    torch.cuda.synchronize()
