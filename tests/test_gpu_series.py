"""-m gpu parity tests of the time-series mode (iqa_series_tiles) against the CPU
oracle (oracle/series.py), element by element on the same seeded snapshots, through the C ABI.

Tolerance: that of the pair path (tests/gpu_util.py): 1e-5 relative per tile on
lisi, X, Y, L, A; auglisi 1e-5 |ref| + 1e-6 r; whole-image pair 1e-5 relative.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

MODES = ["reference", "consecutive"]


@pytest.fixture(scope="module")
def B():
    from paper_2501_10653_b200 import binding
    return binding


@pytest.fixture(scope="module")
def U():
    import gpu_util
    return gpu_util


def _consts():
    return dict(C1=1e-6, C2=1e-6, C=1e-6, D=5e-7)


def _run_and_check(B, U, imgs, mode, N_T, k, what=""):
    import torch
    import oracle
    dev = [U.to_dev(a) for a in imgs]
    got = B.series_tiles(dev, mode, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    torch.cuda.synchronize()
    ref = oracle.series(imgs, mode, N_T, **k)
    K = len(imgs) - 1
    for c in range(K):
        g = {n: got[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
        r = {n: ref[n][c] for n in g}
        U.assert_parity(g, r, k["C"], f"{what} {mode} cmp {c}")
    whole = got["whole"].cpu().numpy().astype(np.float64)
    err = np.abs(whole - ref["whole"])
    tol = 1e-5 * np.abs(ref["whole"])
    tol[:, 1] += 1e-6                      # whole-image augLISI = 1 - r, r <= ~1
    assert np.all(err <= tol), (what, mode, whole, ref["whole"])
    return got, ref


def _rand_series(N, M, seed, frac_equal=0.3):
    rng = np.random.default_rng(seed)
    imgs = [rng.normal(0.05, 0.2, (N, N)).astype(np.float32) for _ in range(M)]
    for j in range(1, M):                  # shared pixels between neighbours and with the reference
        m = rng.random((N, N)) < frac_equal
        imgs[j][m] = imgs[j - 1][m]
        m = rng.random((N, N)) < 0.1
        imgs[j][m] = imgs[0][m]
    return imgs


@pytest.mark.parametrize("mode", MODES)
def test_worked_example_series(B, U, mode):
    """The hand-derived 4x4 example (tests/golden) as a 3-image series; N_T = 2 takes the generic kernel."""
    x = np.array([[1, 0.5, -1, 0], [0.25, 0, 0, 0], [0.75, 0.75, 2, -0.5], [0.125, 0.5, 0, 1]], dtype=np.float32)
    y = np.array([[1, 0.25, 3, -2], [0, 0.5, 0, 0], [0.75, 0.75, 0, 0.5], [0.125, 0.5, 1, 0]], dtype=np.float32)
    k = dict(C1=2.0 ** -20, C2=2.0 ** -20, C=2.0 ** -20, D=2.0 ** -21)
    _run_and_check(B, U, [x, y, x], mode, 2, k, "worked example")


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("N,N_T,M", [(256, 16, 4), (256, 64, 5), (512, 128, 3), (384, 8, 3), (1024, 32, 6),
                                     (2048, 64, 5), (1024, 512, 3), (392, 8, 3), (200, 40, 3), (100, 20, 4),
                                     (64, 8, 2), (32, 32, 3)])
def test_series_shapes(B, U, mode, N, N_T, M):
    """Several tiles per item, whole-tile items, split tiles, ragged right/bottom edges (384, 392, 200),
    generic-kernel shapes (N_T not a power of two), images smaller than a TMA box, M = 2."""
    _run_and_check(B, U, _rand_series(N, M, seed=N + M), mode, N_T, _consts(), f"N={N} N_T={N_T} M={M}")


@pytest.mark.parametrize("mode", MODES)
def test_series_config1_sky(B, U, mode):
    """BASELINE.json config [1] sky (N=2048, N_T=64) as a series of 5 snapshots with on/off transients."""
    from paper_2501_10653_b200 import synth
    cfg = synth.CONFIGS[1]
    imgs, _ = synth.make_series(cfg, 5)
    _run_and_check(B, U, imgs, mode, cfg.N_T, U.consts(cfg), "cfg1 series")


@pytest.mark.parametrize("mode", MODES)
def test_long_series_spans_several_launches(B, U, mode):
    """More images than tensor maps fit in one launch (128): chunks that share one image."""
    _run_and_check(B, U, _rand_series(128, 140, seed=5), mode, 16, _consts(), "M=140")


@pytest.mark.parametrize("mode", MODES)
def test_series_matches_pair_calls(B, U, mode):
    """Same arithmetic as K independent pair calls: bit-identical per-tile results."""
    import torch
    import oracle
    imgs = _rand_series(512, 4, seed=11)
    dev = [U.to_dev(a) for a in imgs]
    k = _consts()
    got = B.series_tiles(dev, mode, 64, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    for c, (ix, iy) in enumerate(oracle.comparison_indices(len(imgs), mode)):
        pair = B.fused_tiles(dev[ix], dev[iy], 64, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
        torch.cuda.synchronize()
        for n in ("lisi", "auglisi", "X", "Y", "L", "A"):
            assert torch.equal(got[n][c], pair[n]), (mode, c, n)


@pytest.mark.parametrize("mode", MODES)
def test_series_unaligned_images_take_the_pairwise_path(B, U, mode):
    import torch
    import oracle
    N, M = 256, 3
    imgs = _rand_series(N, M, seed=3)
    dev = []
    for a in imgs:                          # 4-byte aligned but not 16-byte aligned
        buf = torch.empty(N * N + 1, dtype=torch.float32, device="cuda")
        view = buf[1:].view(N, N)
        view.copy_(torch.from_numpy(a))
        assert view.data_ptr() % 16 == 4
        dev.append(view)
    k = _consts()
    got = B.series_tiles(dev, mode, 16, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    torch.cuda.synchronize()
    ref = oracle.series(imgs, mode, 16, **k)
    for c in range(M - 1):
        g = {n: got[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(g, {n: ref[n][c] for n in g}, k["C"], f"unaligned {mode} {c}")


@pytest.mark.parametrize("cfg_id", ["0", "1", "2", "3"])
@pytest.mark.parametrize("N_T", [16, 64, 256])
def test_series_ring_configurations(B, U, cfg_id, N_T):
    """Every TMA ring / box configuration (IQA_TMA_CONFIG: 6 or 4 boxes of 32 rows, 8 or 6 boxes of 16 rows)
    gives the oracle's values in both series modes."""
    imgs = _rand_series(512, 4, seed=int(cfg_id) + N_T)
    with B.knob("IQA_TMA_CONFIG", int(cfg_id)):
        for mode in MODES:
            _run_and_check(B, U, imgs, mode, N_T, _consts(), f"tma config {cfg_id} N_T={N_T}")


@pytest.mark.parametrize("mode", MODES)
def test_pyramid_of_a_series(B, U, mode):
    """P:66 on every comparison of a series in one launch per level (iqa_merge_tiles_batch): the g x g merge of the
    N_T = 16 matrices equals the oracle's series at tile size 16 g."""
    import torch
    import oracle
    imgs = _rand_series(256, 4, seed=21)
    dev = [U.to_dev(a) for a in imgs]
    k = _consts()
    base = B.series_tiles(dev, mode, 16, k["C1"], k["C2"], k["C"], k["D"])
    for g in (2, 4, 16):
        m = B.merge_tiles(base["lisi"], base["auglisi"], base["X"], base["Y"], g, k["C2"], k["C"])
        torch.cuda.synchronize()
        ref = oracle.series(imgs, mode, 16 * g, **k)
        assert m["lisi"].shape == (3, 16 // g, 16 // g)
        for c in range(3):
            got = {n: m[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y")}
            U.assert_parity(got, {n: ref[n][c] for n in list(got) + ["A"]}, k["C"], f"series merge g={g} cmp {c}")
    levels = B.pyramid(base, k["C2"], k["C"])
    assert [tuple(l["lisi"].shape) for l in levels] == [(3, 16, 16), (3, 8, 8), (3, 4, 4), (3, 2, 2), (3, 1, 1)]
    for j, level in enumerate(levels):       # every level of every comparison against the series oracle at 16 * 2^j
        ref = oracle.series(imgs, mode, 16 << j, **k)
        for c in range(3):
            got = {n: level[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y")}
            U.assert_parity(got, {n: ref[n][c] for n in list(got) + ["A"]}, k["C"], f"series pyramid level {j} cmp {c}")
    top = levels[-1]
    for c in range(3):                      # the top of the pyramid is the whole-image pair of Eqs. 3-4
        w = base["whole"][c].cpu().numpy()
        assert abs(top["lisi"][c, 0, 0].item() - w[0]) <= 1e-5 * abs(w[0])
        assert abs(top["auglisi"][c, 0, 0].item() - w[1]) <= 1e-5 * abs(w[1]) + 1e-6


def test_series_determinism(B, U):
    import torch
    imgs = [U.to_dev(a) for a in _rand_series(1024, 5, seed=2)]
    k = _consts()
    a = B.series_tiles(imgs, "consecutive", 64, k["C1"], k["C2"], k["C"], k["D"])
    b = B.series_tiles(imgs, "consecutive", 64, k["C1"], k["C2"], k["C"], k["D"])
    torch.cuda.synchronize()
    for n in a:
        assert torch.equal(a[n], b[n]), n


def test_series_error_codes(B):
    import torch
    x = torch.zeros((64, 64), dtype=torch.float32, device="cuda")
    o = [torch.zeros(64, dtype=torch.float32, device="cuda") for _ in range(4)]
    k = _consts()
    args = (64, 8, k["C1"], k["C2"], k["C"], k["D"], *o)
    assert B.iqa_series_tiles([x, x], 2, 0, *args) == B.IQA_OK
    assert B.iqa_series_tiles([x], 1, 0, *args) == B.IQA_ERR_SHAPE
    assert B.iqa_series_tiles([x, x], 2, 7, *args) == B.IQA_ERR_SHAPE
    assert B.iqa_series_tiles([x, None], 2, 0, *args) == B.IQA_ERR_NULL
    assert B.iqa_series_tiles([x, x], 2, 0, 64, 8, 0.0, k["C2"], k["C"], k["D"], *o) == B.IQA_ERR_PARAM
    assert B.iqa_series_tiles([x, x], 2, 0, 64, 7, k["C1"], k["C2"], k["C"], k["D"], *o) == B.IQA_ERR_SHAPE
    torch.cuda.synchronize()
