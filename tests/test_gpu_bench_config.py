"""-m gpu parity at BASELINE.json's FULL sizes in the launch configurations bench.py times:
iqa_fused_batch over 32 cfg1 pairs / 8 cfg3 pairs / the 16 cfg4 pairs, and iqa_series_tiles over 9 snapshots
of the N = 8192 sky.  Every pair (cfg1) or a sample of pairs / comparisons (larger configs) is checked
element by element against the oracle on the same device-drawn buffers copied to the host."""
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


def _check_batch(B, U, cfg, pairs, sample, whole_of=None):
    """`sample`: pairs checked element by element (all six per-tile arrays + the whole-image pair);
    `whole_of`: pairs whose whole-image pair (Eqs. 3-4) is checked against the oracle's."""
    import torch
    import oracle
    from paper_2501_10653_b200 import synth
    k = U.consts(cfg)
    xs, ys = [], []
    for s in range(pairs):
        xd, yd, _ = synth.make_pair(cfg, seed=s, device="cuda")
        xs.append(xd)
        ys.append(yd)
    assert B.plan_name(xs[0], cfg.N_T) == "tma:c1"
    out = B.fused_batch(xs, ys, cfg.N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True, aggregate=True)
    torch.cuda.synchronize()
    whole = out["whole"].cpu().numpy().astype(np.float64)
    for i in sorted(set(sample) | set(whole_of or ())):
        x, y = xs[i].cpu().numpy(), ys[i].cpu().numpy()
        ref = oracle.tiles(x, y, cfg.N_T, **k)
        if i in sample:
            got = {n: out[n][i].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
            U.assert_parity(got, ref, k["C"], f"{cfg.name} pair {i} of {pairs}")
        exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], k["C2"], k["C"])
        assert abs(whole[i, 0] - exp[0]) <= 1e-5 * abs(exp[0]), (i, whole[i], exp)
        assert abs(whole[i, 1] - exp[1]) <= 1e-5 * abs(exp[1]), (i, whole[i], exp)
        del x, y, ref
    del xs, ys, out
    torch.cuda.empty_cache()


def test_cfg1_batch_of_32_every_pair(B, U):
    from paper_2501_10653_b200 import synth
    _check_batch(B, U, synth.CONFIGS[1], 32, range(32))


def test_cfg3_batch_of_8_sampled_pairs(B, U):
    from paper_2501_10653_b200 import synth
    _check_batch(B, U, synth.CONFIGS[3], 8, (0, 3, 7))


def test_cfg4_throughput_loop_of_16_pairs(B, U):
    """Config [4] as BASELINE.json states it and bench.py times it: ONE iqa_fused_batch call over 16 pairs of
    N = 16384, N_T = 128 (32 GiB of images resident, a [16 pairs][16384 tiles][2 pieces] workspace, 32 tensor maps in
    one launch).  Pairs 0 and 15 are checked element by element, the whole-image pair of EVERY pair against the oracle
    (SURVEY.md 8(d))."""
    from paper_2501_10653_b200 import synth
    _check_batch(B, U, synth.CONFIGS[4], 16, (0, 15), whole_of=range(16))


@pytest.mark.parametrize("mode", ["reference", "consecutive"])
def test_series_of_9_snapshots_at_8192_sampled_comparisons(B, U, mode):
    import torch
    import oracle
    from paper_2501_10653_b200 import synth
    cfg = synth.CONFIGS[3]
    k = U.consts(cfg)
    imgs, _ = synth.make_series(cfg, 9, device="cuda")
    out = B.series_tiles(imgs, mode, cfg.N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    torch.cuda.synchronize()
    pairs = oracle.comparison_indices(9, mode)
    whole = out["whole"].cpu().numpy().astype(np.float64)
    for c in (0, 4, 7):
        ix, iy = pairs[c]
        ref = oracle.tiles(imgs[ix].cpu().numpy(), imgs[iy].cpu().numpy(), cfg.N_T, **k)
        got = {n: out[n][c].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(got, ref, k["C"], f"series {mode} comparison {c}")
        exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], k["C2"], k["C"])
        assert abs(whole[c, 0] - exp[0]) <= 1e-5 * abs(exp[0]) and abs(whole[c, 1] - exp[1]) <= 1e-5 * abs(exp[1])
    # every snapshot's tile sums must agree between the comparisons that share it (consistency at full size)
    if mode == "consecutive":
        for c in range(7):
            assert torch.equal(out["Y"][c], out["X"][c + 1]), c
    else:
        for c in range(1, 8):
            assert torch.equal(out["X"][c], out["X"][0]), c


def test_series_soak_bitwise(B, U):
    """Ten runs of a 5-snapshot series at N = 2048 (items change hands between CTAs, slots are reused
    hundreds of times): bit-identical results every time."""
    import torch
    from paper_2501_10653_b200 import synth
    cfg = synth.CONFIGS[1]
    k = U.consts(cfg)
    imgs, _ = synth.make_series(cfg, 5, device="cuda")
    for mode in ("reference", "consecutive"):
        first = B.series_tiles(imgs, mode, cfg.N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
        for _ in range(9):
            again = B.series_tiles(imgs, mode, cfg.N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
            torch.cuda.synchronize()
            for n in first:
                assert torch.equal(first[n], again[n]), (mode, n)


def test_n32768_sampled_tiles(B, U):
    """Maximum size of the suite: N = 32768 (4 GiB per image, element offsets beyond 2^30), N_T = 128.
    The oracle checks 48 sampled tiles (incl. the four corners) on crops copied to the host -- crop
    consistency is pinned for the oracle (tests/test_oracle_pins.py P9) -- plus the column sums of X and Y
    of every tile row against torch reductions of the clamped images (a property that holds at any size)."""
    import torch
    import oracle
    N, N_T = 32768, 128
    nt = N // N_T
    k = dict(C1=1e-6, C2=1e-6, C=1e-6, D=5e-7)
    g = torch.Generator(device="cuda").manual_seed(7)
    x = torch.empty((N, N), dtype=torch.float32, device="cuda").normal_(0.0, 1e-3, generator=g)
    y = torch.empty((N, N), dtype=torch.float32, device="cuda").normal_(0.0, 1e-3, generator=g)
    x[N - 100:N - 90, N - 300:N - 200] += 0.5                  # a source in the last tile row
    out = B.fused_tiles(x, y, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    torch.cuda.synchronize()
    rng = np.random.default_rng(0)
    picks = {(0, 0), (0, nt - 1), (nt - 1, 0), (nt - 1, nt - 1), (nt - 1, nt - 3)}
    while len(picks) < 48:
        picks.add((int(rng.integers(nt)), int(rng.integers(nt))))
    for ty, tx in sorted(picks):
        xc = x[ty * N_T:(ty + 1) * N_T, tx * N_T:(tx + 1) * N_T].contiguous().cpu().numpy()
        yc = y[ty * N_T:(ty + 1) * N_T, tx * N_T:(tx + 1) * N_T].contiguous().cpu().numpy()
        ref = oracle.tiles(xc, yc, N_T, **k)
        got = {n: out[n][ty:ty + 1, tx:tx + 1].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(got, ref, k["C"], f"N=32768 tile ({ty},{tx})")
    # every tile contributes: sums over tile columns == sums of the clamped image over the same row bands (fp64)
    for name, img in (("X", x), ("Y", y)):
        rows = img.clamp_min(0).view(nt, N_T * N).sum(dim=1, dtype=torch.float64)
        got = out[name].sum(dim=1, dtype=torch.float64)
        assert torch.all((got - rows).abs() <= 1e-6 * rows.abs()), name


def _path_rows():
    import bench
    return bench.PATH_ROWS


@pytest.mark.parametrize("row", _path_rows(), ids=[r[0] for r in _path_rows()])
def test_bench_path_rows_at_full_size(B, U, row):
    """The `also.paths` rows of bench.py (any_kernel on odd tile sides / other pixel types / unaligned bases, the generic
    kernels on odd pitches) at the size and in the launch configuration bench.py times -- one iqa_fused_batch_2d_typed
    call over 4 pairs of 8192 x 8192 windows -- against the oracle: EVERY tile and the whole-image pair of the first and
    the last pair, on the same seeded device buffers copied to the host."""
    import torch
    import bench
    import oracle
    name, dtype, H, W, pitch, off, N_T = row
    pairs = 4
    xs, ys = bench.make_path_inputs(torch, row, pairs, "cuda")
    # (a 64-column tile behind a base 4 bytes off fills 17 of 32 lanes of any_kernel: the plan takes the generic kernel)
    #  and split tiles that would fill few lanes take it too)
    by_lane_fill = ("f32_NT64_base4B", "f32_NT130_split", "i16_NT200_split", "f32_NT300_split")
    expect = "generic" if name.startswith("generic") or name in by_lane_fill else "tma_any"
    assert B.plan_name(xs[0], N_T) == expect, (name, B.plan_name(xs[0], N_T))
    C1, C2, C, D = bench.PATH_CONSTS
    out = B.fused_batch_2d(xs, ys, N_T, C1, C2, C, D, numerators=True, aggregate=True)
    torch.cuda.synchronize()
    whole = out["whole"].cpu().numpy().astype(np.float64)
    for i in (0, pairs - 1):
        x, y = xs[i].cpu().numpy(), ys[i].cpu().numpy()
        ref = oracle.tiles_2d_any(x, y, N_T, C1, C2, C, D)
        got = {n: out[n][i].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(got, ref, C, f"{name} pair {i}")
        exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], C2, C)
        assert abs(whole[i, 0] - exp[0]) <= 1e-5 * abs(exp[0]) and abs(whole[i, 1] - exp[1]) <= 1e-5 * abs(exp[1]), (name, i)
        del x, y, ref
    del xs, ys, out
    torch.cuda.empty_cache()
