"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by
element, on the same seeded fp32 buffers.  SURVEY.md 8(c) P11-P12 plus the edge cases.

Citations: Eq. 1, Eq. 2, clamp PAPER.md:27, Eqs. 3-4 PAPER.md:55-60.
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from paper_2501_10653_b200 import synth  # noqa: E402

K6 = dict(C1=1e-6, C2=1e-6, C=1e-6, D=float(np.float32(1e-6)) / 2)


@pytest.fixture(scope="module")
def B():
    from paper_2501_10653_b200 import binding
    return binding


@pytest.fixture(scope="module")
def U():
    import gpu_util
    return gpu_util


def _rand_pair(N, seed, frac_equal=0.2):
    rng = np.random.default_rng(seed)
    x = rng.normal(0.1, 1.0, (N, N)).astype(np.float32)
    y = rng.normal(0.1, 1.0, (N, N)).astype(np.float32)
    m = rng.random((N, N)) < frac_equal
    y[m] = x[m]                       # equal pixels: |x-y| = 0, term (x+y)/C1
    x[rng.random((N, N)) < 0.05] = 0.0
    return x, y


# ----------------------------------------------------------------------------- worked example
def test_worked_example_4x4(B, U):
    """tests/golden/worked_example_4x4.txt (derived from Eqs. 1-4 with exact rationals)."""
    from fractions import Fraction as Fr
    x = np.array([[1, 0.5, -1, 0], [0.25, 0, 0, 0], [0.75, 0.75, 2, -0.5], [0.125, 0.5, 0, 1]], np.float32)
    y = np.array([[1, 0.25, 3, -2], [0, 0.5, 0, 0], [0.75, 0.75, 0, 0.5], [0.125, 0.5, 1, 0]], np.float32)
    k = dict(C1=2.0 ** -20, C2=2.0 ** -20, C=2.0 ** -20, D=2.0 ** -21)
    golden = {}
    for ln in open(os.path.join(os.path.dirname(__file__), "golden", "worked_example_4x4.txt")):
        if ln.startswith("tile") or ln.startswith("whole"):
            parts = ln.split()
            vals = {q.split("=")[0]: float(Fr(q.split("=")[1])) for q in parts if "=" in q}
            golden[parts[1] if parts[0] == "tile" else "whole"] = vals
    got = U.run_gpu(U.to_dev(x), U.to_dev(y), 2, k)
    for t in range(4):
        for nm in ("lisi", "auglisi", "X", "Y", "L", "A"):
            exp = golden[str(t)][nm]
            assert abs(got[nm].ravel()[t] - exp) <= 1e-6 * abs(exp) + 1e-12, (t, nm)
    assert got["auglisi"].ravel()[2] == 1.0            # identical tile: exactly 1
    assert got["auglisi"].ravel()[1] < -1.99           # outputs are not clamped
    one = U.run_gpu(U.to_dev(x), U.to_dev(y), 4, k)
    for nm in ("lisi", "auglisi", "X", "Y", "L", "A"):
        exp = golden["whole"][nm]
        assert abs(one[nm][0, 0] - exp) <= 1e-6 * abs(exp), nm
    # Eqs. 3-4 on the device reproduce the whole-image values
    o = B.fused_tiles(U.to_dev(x), U.to_dev(y), 2, **k)
    agg = B.aggregate(o["lisi"], o["auglisi"], o["X"], o["Y"], k["C2"], k["C"]).cpu().numpy()
    assert abs(agg[0] - golden["whole"]["lisi"]) <= 1e-6 * golden["whole"]["lisi"]
    assert abs(agg[1] - golden["whole"]["auglisi"]) <= 1e-6


# ----------------------------------------------------------------------------- BASELINE.json configs
def test_config0(U):
    cfg = synth.CONFIGS[0]
    x, y, _ = synth.make_pair(cfg)
    U.check_pair(x, y, cfg.N_T, U.consts(cfg), "cfg0")


def test_config1_and_shared_noise(U):
    cfg = synth.CONFIGS[1]
    x, y, _ = synth.make_pair(cfg)
    got, ref, _ = U.check_pair(x, y, cfg.N_T, U.consts(cfg), "cfg1")
    # soft science echo (P10): the lowest augLISI tiles hold the dropped sources
    xs, ys, _ = synth.make_pair(cfg, shared_noise=True)
    U.check_pair(xs, ys, cfg.N_T, U.consts(cfg), "cfg1 shared noise")


@pytest.mark.parametrize("N_T", [8, 16, 32, 64, 128, 256, 512, 1024, 2048])
def test_config2_tile_sweep(U, N_T):
    cfg = synth.CONFIGS[2]
    x, y, _ = _cfg2_pair()
    U.check_pair(x, y, N_T, U.consts(cfg), f"cfg2 N_T={N_T}", *_cfg2_dev(U))


def test_config2_other_reading_of_the_generator(U):
    """BASELINE.json config [2] says "same generator as config 1, seed 1"; R13 reads that as BJ index [1].
    The other reading -- the FIRST listed config's generator (30 sources, sigma 1.5 px, log-uniform flux) on the
    2048 canvas -- is run here too, over the ends and the middle of the sweep."""
    from dataclasses import replace
    cfg = replace(synth.CONFIGS[0], name="cfg2_alt_N2048", N=2048, N_T=64, seed=1)
    x, y, _ = synth.make_pair(cfg)
    xd, yd = U.to_dev(x), U.to_dev(y)
    for N_T in (8, 64, 512):
        U.check_pair(x, y, N_T, U.consts(cfg), f"cfg2 alt N_T={N_T}", xd, yd)


_CFG2 = {}


def _cfg2_pair():
    if "host" not in _CFG2:
        _CFG2["host"] = synth.make_pair(synth.CONFIGS[2])
    return _CFG2["host"]


def _cfg2_dev(U):
    if "dev" not in _CFG2:
        x, y, _ = _cfg2_pair()
        _CFG2["dev"] = (U.to_dev(x), U.to_dev(y))
    return _CFG2["dev"]


def test_config3_full(U, B):
    cfg = synth.CONFIGS[3]
    x, y, _ = synth.make_pair(cfg)
    k = U.consts(cfg)
    xd, yd = U.to_dev(x), U.to_dev(y)
    got, ref, _ = U.check_pair(x, y, cfg.N_T, k, "cfg3", xd, yd)
    # aggregate (Eqs. 3-4) against the oracle's whole-image value computed directly
    o = B.fused_tiles(xd, yd, cfg.N_T, **k)
    agg = B.aggregate(o["lisi"], o["auglisi"], o["X"], o["Y"], k["C2"], k["C"]).cpu().numpy()
    exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], k["C2"], k["C"])
    assert abs(agg[0] - exp[0]) <= 1e-5 * abs(exp[0])
    assert abs(agg[1] - exp[1]) <= 1e-5 * abs(exp[1])


def test_config4_full_size(U, B):
    """N=16384, N_T=128, 1 GiB per image: noise drawn on the device, buffers copied back for the oracle."""
    cfg = synth.CONFIGS[4]
    k = U.consts(cfg)
    xd, yd, _ = synth.make_pair(cfg, device="cuda")
    x, y = xd.cpu().numpy(), yd.cpu().numpy()
    got, ref, _ = U.check_pair(x, y, cfg.N_T, k, "cfg4", xd, yd)
    o = B.fused_tiles(xd, yd, cfg.N_T, **k)
    agg = B.aggregate(o["lisi"], o["auglisi"], o["X"], o["Y"], k["C2"], k["C"]).cpu().numpy()
    exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], k["C2"], k["C"])
    assert abs(agg[0] - exp[0]) <= 1e-5 * abs(exp[0])
    assert abs(agg[1] - exp[1]) <= 1e-5 * abs(exp[1])
    # whole image as ONE tile (maximum tile size; 65536 pieces through the workspace)
    one = U.run_gpu(xd, yd, cfg.N, k)
    whole = oracle.tiles(x, y, cfg.N, **k)
    U.assert_parity(one, whole, k["C"], "cfg4 single tile")


# ----------------------------------------------------------------------------- shapes and edges
@pytest.mark.parametrize("N,N_T", [
    (8, 8), (16, 8), (24, 8), (136, 8), (200, 8), (264, 8), (64, 64), (192, 64), (320, 64),
    (128, 128), (384, 128), (256, 256), (768, 256), (1536, 512), (48, 16), (96, 32), (160, 32),
    (4, 2), (12, 4), (10, 5), (9, 3), (7, 1), (36, 12), (200, 100), (130, 65), (390, 130), (5, 5)])
def test_shapes(U, N, N_T):
    x, y = _rand_pair(N, seed=N * 1000 + N_T)
    U.check_pair(x, y, N_T, K6, f"N={N} N_T={N_T}")


@pytest.mark.parametrize("N,N_T", [(256, 8), (256, 64), (512, 128), (100, 20)])
def test_unaligned_pointers_take_generic_kernel(U, B, N, N_T):
    x, y = _rand_pair(N, seed=7)
    buf_x = torch.empty(N * N + 3, dtype=torch.float32, device="cuda")
    buf_y = torch.empty(N * N + 3, dtype=torch.float32, device="cuda")
    xd = buf_x[1:1 + N * N].view(N, N)
    yd = buf_y[3:3 + N * N].view(N, N)
    xd.copy_(torch.from_numpy(x))
    yd.copy_(torch.from_numpy(y))
    assert xd.data_ptr() % 16 != 0
    U.check_pair(x, y, N_T, K6, "unaligned", xd, yd)


def test_special_values(U):
    """NaN, -0, -Inf and negatives clamp to zero (reading R3); all-zero tile gives lisi 0, auglisi 1 (R7)."""
    N, N_T = 128, 16
    x, y = _rand_pair(N, seed=11)
    x[0:16, 0:16] = -1.0
    y[0:16, 0:16] = np.nan                 # tile 0: everything clamps to zero
    x[20, 20] = np.nan
    y[21, 21] = -np.inf
    x[22, 22] = -0.0
    y[22, 22] = -0.0
    got, ref, _ = U.check_pair(x, y, N_T, K6, "special")
    assert got["lisi"][0, 0] == 0.0 and got["auglisi"][0, 0] == 1.0
    assert got["X"][0, 0] == 0.0 and got["Y"][0, 0] == 0.0
    # P7: replacing the clamped pixels by zeros changes nothing, bit for bit
    xz = np.where(x > 0, x, 0).astype(np.float32)
    yz = np.where(y > 0, y, 0).astype(np.float32)
    got2 = U.run_gpu(U.to_dev(xz), U.to_dev(yz), N_T, K6)
    for nm in got:
        assert np.array_equal(got[nm], got2[nm]), nm


def test_identical_images(U):
    """P3: auglisi(x, x) = 1 exactly; lisi(x, x) = (2D/C1) X/(X+C2)."""
    cfg = synth.CONFIGS[0]
    x, _, _ = synth.make_pair(cfg)
    k = U.consts(cfg)
    got, ref, _ = U.check_pair(x, x, cfg.N_T, k, "identical")
    assert np.all(got["auglisi"] == 1.0)
    assert np.array_equal(got["X"], got["Y"])
    X = ref["X"]
    closed = X / (X + float(np.float32(cfg.C2)))
    assert np.max(np.abs(got["lisi"] - closed) / closed) <= 1e-5


def test_symmetry_bitwise(U):
    """P4: swapping x and y leaves both indices bit-identical and swaps X, Y."""
    x, y = _rand_pair(256, seed=3)
    a = U.run_gpu(U.to_dev(x), U.to_dev(y), 32, K6)
    b = U.run_gpu(U.to_dev(y), U.to_dev(x), 32, K6)
    assert np.array_equal(a["lisi"], b["lisi"]) and np.array_equal(a["auglisi"], b["auglisi"])
    assert np.array_equal(a["X"], b["Y"]) and np.array_equal(a["Y"], b["X"])


def test_determinism_and_mapping_independence(U, B):
    """P12: two runs bit-identical; every mapping (tma_kernel ring / box configurations, any_kernel, generic
    kernel, a capped grid, no PDL) agrees with the oracle and with the default mapping to 2e-6."""
    cfg = synth.CONFIGS[0]
    x, y, _ = synth.make_pair(synth.scaled(synth.CONFIGS[3], 1024))
    xd, yd = U.to_dev(x), U.to_dev(y)
    k = U.consts(cfg)
    for N_T in (8, 32, 64, 128, 512):
        base = U.run_gpu(xd, yd, N_T, k)
        again = U.run_gpu(xd, yd, N_T, k)
        for nm in base:
            assert np.array_equal(base[nm], again[nm]), (N_T, nm)
        ref = U.run_oracle(x, y, N_T, k)
        for env, val in (("IQA_FORCE_ANY", 1), ("IQA_TMA_MAX_CTAS", 37), ("IQA_NO_PDL", 1),
                         ("IQA_FORCE_GENERIC", 1), ("IQA_TMA_CONFIG", 0), ("IQA_TMA_CONFIG", 2),
                         ("IQA_TMA_CONFIG", 3), ("IQA_TMA_CONFIG", 4)):
            with B.knob(env, val):
                other = U.run_gpu(xd, yd, N_T, k)
            U.assert_parity(other, ref, k["C"], f"{env}={val} N_T={N_T}")
            for nm in base:
                assert np.max(U.rel_err(other[nm], base[nm])) <= 2e-6, (env, val, N_T, nm)


def test_standalone_entry_points_match_fused(U, B):
    cfg = synth.CONFIGS[1]
    x, y, _ = synth.make_pair(cfg)
    xd, yd = U.to_dev(x), U.to_dev(y)
    k = U.consts(cfg)
    for N_T in (16, 64, 256):        # tma_kernel<lisi> / <auglisi>: several tiles per item, whole tiles, split tiles
        f = B.fused_tiles(xd, yd, N_T, **k)
        li = B.lisi_tiles(xd, yd, N_T, k["C1"], k["C2"], k["D"])
        au = B.auglisi_tiles(xd, yd, N_T, k["C"])
        assert torch.equal(li, f["lisi"]) and torch.equal(au, f["auglisi"])
        # and against the oracle directly on the same data, not only through the fused call
        ref = U.run_oracle(x, y, N_T, k)
        got = {"lisi": li.cpu().numpy().astype(np.float64), "auglisi": au.cpu().numpy().astype(np.float64)}
        U.assert_parity(got, ref, k["C"], f"standalone entry points, N_T={N_T}")


@pytest.mark.parametrize("N,N_T,P", [(256, 16, 5), (2048, 64, 3), (1024, 8, 2), (1024, 256, 3), (392, 8, 4),
                                     (200, 100, 2), (512, 128, 40), (256, 16, 70)])
def test_fused_batch_matches_per_pair_calls_and_oracle(U, B, N, N_T, P):
    """iqa_fused_batch == P calls of iqa_fused_tiles + iqa_aggregate, bit for bit, and == the oracle."""
    cfg = synth.scaled(synth.CONFIGS[3], N, N_T)
    k = U.consts(cfg)
    hosts = [synth.make_pair(cfg, seed=s)[:2] for s in range(min(P, 6))]
    hosts = [hosts[i % len(hosts)] for i in range(P)]
    xs = [U.to_dev(h[0]) for h in hosts]
    ys = [U.to_dev(h[1]) for h in hosts]
    out = B.fused_batch(xs, ys, N_T, numerators=True, **k)
    torch.cuda.synchronize()
    nt = N // N_T
    assert out["lisi"].shape == (P, nt, nt) and out["whole"].shape == (P, 2)
    for i in range(P):
        one = B.fused_tiles(xs[i], ys[i], N_T, numerators=True, **k)
        agg = B.aggregate(one["lisi"], one["auglisi"], one["X"], one["Y"], k["C2"], k["C"])
        for nm in one:
            assert torch.equal(one[nm], out[nm][i]), (i, nm)
        assert torch.equal(agg, out["whole"][i]), i
    for i in range(min(P, 6)):
        ref = U.run_oracle(hosts[i][0], hosts[i][1], N_T, k)
        got = {nm: out[nm][i].cpu().numpy().astype(np.float64) for nm in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(got, ref, k["C"], f"batch pair {i}")
        exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], k["C2"], k["C"])
        w = out["whole"][i].cpu().numpy()
        assert abs(w[0] - exp[0]) <= 1e-5 * abs(exp[0]) and abs(w[1] - exp[1]) <= 1e-5 * abs(exp[1])


def test_fused_batch_unaligned_pair_takes_generic_kernel(U, B):
    N, N_T, P = 128, 16, 3
    hosts = [_rand_pair(N, seed=20 + s) for s in range(P)]
    buf = torch.empty(N * N + 3, dtype=torch.float32, device="cuda")
    x1 = buf[1:1 + N * N].view(N, N)
    x1.copy_(torch.from_numpy(hosts[1][0]))
    xs = [U.to_dev(hosts[0][0]), x1, U.to_dev(hosts[2][0])]
    ys = [U.to_dev(h[1]) for h in hosts]
    out = B.fused_batch(xs, ys, N_T, numerators=True, **K6)
    for i in range(P):
        ref = U.run_oracle(hosts[i][0], hosts[i][1], N_T, K6)
        got = {nm: out[nm][i].cpu().numpy().astype(np.float64) for nm in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(got, ref, K6["C"], f"unaligned batch pair {i}")


@pytest.mark.parametrize("N,N_T", [(512, 64), (512, 128)])
def test_fused_batch_of_mixed_alignment_is_planned_per_run(U, B, N, N_T):
    """One pair behind a base 4 bytes off in a 4-pair batch: every pair gets the kernel it would get alone (bit-identical
    to the single calls, which for the aligned pairs means tma_kernel and not the generic fall-back), Eqs. 3-4 included."""
    P = 4
    hosts = [_rand_pair(N, seed=40 + s) for s in range(P)]
    buf = torch.empty(N * N + 3, dtype=torch.float32, device="cuda")
    x2 = buf[1:1 + N * N].view(N, N)
    x2.copy_(torch.from_numpy(hosts[2][0]))
    xs = [U.to_dev(hosts[0][0]), U.to_dev(hosts[1][0]), x2, U.to_dev(hosts[3][0])]
    ys = [U.to_dev(h[1]) for h in hosts]
    assert B.plan_name(xs[0], N_T).startswith("tma:") and not B.plan_name(x2, N_T).startswith("tma:")
    out = B.fused_batch(xs, ys, N_T, numerators=True, **K6)
    for i in range(P):
        single = B.fused_tiles(xs[i], ys[i], N_T, numerators=True, **K6)
        whole = B.aggregate(single["lisi"], single["auglisi"], single["X"], single["Y"], K6["C2"], K6["C"])
        for nm in ("lisi", "auglisi", "X", "Y", "L", "A"):
            assert torch.equal(out[nm][i], single[nm]), (i, nm)
        assert torch.equal(out["whole"][i], whole), i
        ref = U.run_oracle(hosts[i][0], hosts[i][1], N_T, K6)
        got = {nm: out[nm][i].cpu().numpy().astype(np.float64) for nm in ("lisi", "auglisi", "X", "Y", "L", "A")}
        U.assert_parity(got, ref, K6["C"], f"mixed batch pair {i}")


def test_aggregate_equals_whole_image_and_merge(U, B):
    """P6: Eqs. 3-4 over the tiles == the index of the whole image; g x g merge == tiles at g*N_T."""
    cfg = synth.CONFIGS[1]
    x, y, _ = synth.make_pair(cfg)
    xd, yd = U.to_dev(x), U.to_dev(y)
    k = U.consts(cfg)
    whole = oracle.tiles(x, y, cfg.N, **k)
    for N_T in (8, 64, 256):
        o = B.fused_tiles(xd, yd, N_T, **k)
        agg = B.aggregate(o["lisi"], o["auglisi"], o["X"], o["Y"], k["C2"], k["C"]).cpu().numpy()
        assert abs(agg[0] - whole["lisi"][0, 0]) <= 1e-5 * whole["lisi"][0, 0], N_T
        assert abs(agg[1] - whole["auglisi"][0, 0]) <= 1e-5 * abs(whole["auglisi"][0, 0]), N_T
    o = B.fused_tiles(xd, yd, 32, **k)
    for g in (1, 2, 4, 64):
        m = B.merge_tiles(o["lisi"], o["auglisi"], o["X"], o["Y"], g, k["C2"], k["C"])
        ref = oracle.tiles(x, y, 32 * g, **k)
        got = {n: m[n].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y")}
        U.assert_parity(got, ref, k["C"], f"merge g={g}")
    # iqa_pyramid: EVERY level in one launch, each against the oracle at tile size 2^j * 32
    lv = B.pyramid(o, k["C2"], k["C"])
    assert [l["lisi"].shape[0] for l in lv] == [64, 32, 16, 8, 4, 2, 1]
    for j, level in enumerate(lv):
        ref = oracle.tiles(x, y, 32 << j, **k)
        got = {n: level[n].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y")}
        U.assert_parity(got, ref, k["C"], f"pyramid level {j}")
    agg = B.aggregate(o["lisi"], o["auglisi"], o["X"], o["Y"], k["C2"], k["C"]).cpu().numpy()
    assert abs(lv[-1]["lisi"].item() - agg[0]) <= 1e-6 * abs(agg[0]) and abs(lv[-1]["auglisi"].item() - agg[1]) <= 1e-6 * abs(agg[1])
    for N_T in (8, 64):                     # 65536 base tiles (CTA-wide units at the top) and the bench tile size
        o2 = B.fused_tiles(xd, yd, N_T, **k)
        for j, level in enumerate(B.pyramid(o2, k["C2"], k["C"])):
            if j in (0, 1, 5) or (N_T << j) >= 1024:
                ref = oracle.tiles(x, y, N_T << j, **k)
                got = {n: level[n].cpu().numpy().astype(np.float64) for n in ("lisi", "auglisi", "X", "Y")}
                U.assert_parity(got, ref, k["C"], f"pyramid N_T={N_T} level {j}")


def test_fused_host_entry_point(U, B):
    cfg = synth.CONFIGS[0]
    x, y, _ = synth.make_pair(cfg)
    k = U.consts(cfg)
    xp, yp = torch.from_numpy(x).pin_memory(), torch.from_numpy(y).pin_memory()
    out, out2 = B.fused_host(xp, yp, cfg.N_T, **k)
    ref = U.run_oracle(x, y, cfg.N_T, k)
    got = {n: out[n].numpy().astype(np.float64) for n in out}
    U.assert_parity(got, ref, k["C"], "fused_host")
    exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], k["C2"], k["C"])
    assert abs(out2[0].item() - exp[0]) <= 1e-5 * abs(exp[0])
    assert abs(out2[1].item() - exp[1]) <= 1e-5 * abs(exp[1])
    out_np, _ = B.fused_host(x, y, 128, **k)          # pageable numpy input, split-tile mapping
    ref = U.run_oracle(x, y, 128, k)
    U.assert_parity({n: out_np[n].numpy().astype(np.float64) for n in out_np}, ref, k["C"], "fused_host 128")


def test_host_pipeline_two_streams(U, B):
    """iqa_fused_host_async on two streams (binding.HostPipeline): six distinct pairs, every result against the oracle."""
    cfg = synth.scaled(synth.CONFIGS[1], 512)
    k = U.consts(cfg)
    pairs = [synth.make_pair(cfg, seed=s)[:2] for s in range(6)]
    pinned = [(torch.from_numpy(x).pin_memory(), torch.from_numpy(y).pin_memory()) for x, y in pairs]
    pipe = B.HostPipeline(cfg.N, cfg.N_T, "cuda:0", depth=2)
    results, slots = [], []

    def collect(slot):
        out, out2 = pipe.wait(slot)
        results.append(({n: v.clone() for n, v in out.items()}, out2.clone()))

    for xp, yp in pinned:
        slots.append(pipe.submit(xp, yp, k["C1"], k["C2"], k["C"], k["D"]))
        if len(slots) > 1:
            collect(slots[-2])
    collect(slots[-1])
    pipe.drain()
    assert len(results) == 6
    for (x, y), (out, out2) in zip(pairs, results):
        ref = U.run_oracle(x, y, cfg.N_T, k)
        U.assert_parity({n: out[n].numpy().astype(np.float64) for n in out}, ref, k["C"], "host pipeline")
        exp = oracle.aggregate(ref["lisi"], ref["auglisi"], ref["X"], ref["Y"], k["C2"], k["C"])
        assert abs(out2[0].item() - exp[0]) <= 1e-5 * abs(exp[0]) and abs(out2[1].item() - exp[1]) <= 1e-5 * abs(exp[1])


def test_every_baseline_configuration_takes_the_tma_kernel(B):
    """A silent fall-back to the generic kernel would keep parity and lose bandwidth: assert the plan."""
    for idx in range(5):
        cfg = synth.CONFIGS[idx]
        x = torch.empty((cfg.N, cfg.N), dtype=torch.float32, device="cuda")
        for N_T in (cfg.sweep_N_T or (cfg.N_T,)):
            assert B.plan_name(x, N_T) == "tma:c1", (cfg.name, N_T)
            assert B.plan_name(x, N_T, series=True) == "tma:c0", (cfg.name, N_T)
        del x
    x = torch.empty((300, 516), dtype=torch.float32, device="cuda")
    assert B.plan_name(x[:, :513], 64).startswith("tma")            # pitched window, W % 4 != 0
    assert B.plan_name(x[:, 1:514], 100) == "tma_any"               # base 4-byte aligned only: any_kernel shifts columns
    assert B.plan_name(x[:, 1:514], 64) == "generic"                # ... unless that leaves half of its lanes idle
    assert B.plan_name(x, 130) == "generic" and B.plan_name(x, 110) == "tma_any"   # split tiles: by lane fill
    assert B.plan_name(x, 100) == "tma_any"                         # tile side not a power of two
    assert B.plan_name(x[:, :515], 2) == "generic"                  # N_T < 4
    y = torch.empty((300, 517), dtype=torch.float32, device="cuda")
    assert B.plan_name(y, 64) == "generic"                          # row pitch not a multiple of 16 bytes
    assert B.plan_name(y.to(torch.float64)[:, :500], 64) == "generic" and B.plan_name(x.to(torch.uint8), 64) == "generic"
    assert B.plan_name(torch.empty((64, 528), dtype=torch.uint8, device="cuda"), 50) == "tma_any"


def test_many_small_tiles(U):
    """N=4096, N_T=8: 262144 tiles (16 tile segments per warp row)."""
    x, y = _rand_pair(4096, seed=5)
    U.check_pair(x, y, 8, K6, "many tiles")


def test_error_codes_on_device(B):
    N, N_T = 256, 128
    x = torch.zeros((N, N), device="cuda")
    n = (N // N_T) ** 2
    o = [torch.zeros(n, device="cuda") for _ in range(4)]
    need = B.iqa_workspace_bytes(N, N_T)
    assert need > 0
    rc = B.iqa_fused_tiles(x, x, N, N_T, 1e-6, 1e-6, 1e-6, 5e-7, *o, None, None, None, 0, None)
    assert rc == B.IQA_ERR_WORKSPACE
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    rc = B.iqa_fused_tiles(x, x, N, N_T, 1e-6, 1e-6, 1e-6, 5e-7, *o, None, None, ws, need - 1, None)
    assert rc == B.IQA_ERR_WORKSPACE
    rc = B.iqa_fused_tiles(x, x, N, N_T, 1e-6, 1e-6, 1e-6, 5e-7, *o, None, None, ws, need, None)
    assert rc == B.IQA_OK
    rc = B.iqa_fused_tiles(x.data_ptr() + 2, x, N, N_T, 1e-6, 1e-6, 1e-6, 5e-7, *o, None, None, ws, need, None)
    assert rc == B.IQA_ERR_ALIGN
    torch.cuda.synchronize()


@pytest.mark.parametrize("N,N_T", [(2048, 64), (2048, 256), (2048, 512), (512, 128), (256, 128)])
def test_one_pair_calls_and_batches_sum_in_the_same_order(U, B, N, N_T):
    """iqa_fused_batch over 1 pair, over 5 pairs, and iqa_fused_tiles + iqa_aggregate give bit-identical results: the
    second pass of split tiles is chosen by (pieces, tiles per pair) alone, never by the batch size (n = 16 tiles with
    32 pieces at N = 2048, N_T = 512 used to switch kernels between a single pair and a batch of four)."""
    dev = [tuple(U.to_dev(a) for a in _rand_pair(N, seed=N_T + i)) for i in range(5)]
    k = K6
    batch = B.fused_batch([d[0] for d in dev], [d[1] for d in dev], N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
    for i, (xd, yd) in enumerate(dev):
        one = B.fused_batch([xd], [yd], N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=True)
        t = B.fused_tiles(xd, yd, N_T, numerators=True, **k)
        agg = B.aggregate(t["lisi"], t["auglisi"], t["X"], t["Y"], k["C2"], k["C"])
        torch.cuda.synchronize()
        for n in ("lisi", "auglisi", "X", "Y", "L", "A"):
            assert torch.equal(batch[n][i], one[n][0]) and torch.equal(one[n][0], t[n]), (i, n)
        assert torch.equal(batch["whole"][i], agg) and torch.equal(one["whole"][0], agg), i
