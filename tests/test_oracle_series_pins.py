"""Pins for the time-series and candidate-extraction oracles (oracle/series.py) -- CPU only.

series (Eqs. 1-4 PAPER.md:15-21, 55-60 applied to each comparison of a series,
PAPER.md:13, :39):
  S1  the hand-derived 4x4 worked example embedded in a 3-image series: reference and consecutive
      modes must put the golden values (tests/golden/worked_example_4x4.txt) in the right slots,
      with X and Y swapped where the roles of the two images swap
  S2  exact-rational brute force (oracle/exact_rational.py) of every comparison, both modes
  S3  a repeated reference frame gives auglisi == 1 exactly in that slot only (reference mode);
      a frame repeated twice in a row does so in consecutive mode
  S4  the two modes agree on comparison 0 and differ afterwards
candidates (reading R17):
  C1  hand-written lists incl. ties, -0/+0, k = 0, k >= n
  C2  pure-Python selection loop on random matrices with many ties
  C3  soft: on a config-[0] sky the bottom-5 augLISI tiles contain the dropped sources
"""
import os
from fractions import Fraction as Fr

import numpy as np
import pytest

import oracle
from oracle import exact_rational as er
from paper_2501_10653_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "worked_example_4x4.txt")
X_ROWS = [[1, 0.5, -1, 0], [0.25, 0, 0, 0], [0.75, 0.75, 2, -0.5], [0.125, 0.5, 0, 1]]
Y_ROWS = [[1, 0.25, 3, -2], [0, 0.5, 0, 0], [0.75, 0.75, 0, 0.5], [0.125, 0.5, 1, 0]]
K = dict(C1=2.0 ** -20, C2=2.0 ** -20, C=2.0 ** -20, D=2.0 ** -21)


def _golden():
    tiles, whole = {}, None
    for ln in open(GOLDEN):
        if ln.startswith("tile") or ln.startswith("whole"):
            parts = ln.split()
            vals = {p.split("=")[0]: float(Fr(p.split("=")[1])) for p in parts if "=" in p}
            if parts[0] == "tile":
                tiles[int(parts[1])] = vals
            else:
                whole = vals
    return tiles, whole


def _close(a, b, rtol=1e-12):
    return abs(a - b) <= rtol * max(abs(b), 1e-300)


# ----------------------------------------------------------------------------- S1
@pytest.mark.parametrize("mode", ["reference", "consecutive"])
def test_worked_example_in_a_series(mode):
    tiles, whole = _golden()
    x = np.array(X_ROWS, dtype=np.float32)
    y = np.array(Y_ROWS, dtype=np.float32)
    got = oracle.series([x, y, x], mode, 2, **K)
    assert got["lisi"].shape == (2, 2, 2) and got["whole"].shape == (2, 2)
    # comparison 0 is (x, y) in both modes: the golden values as they are
    for t, g in tiles.items():
        ty, tx = divmod(t, 2)
        for name in ("lisi", "auglisi", "X", "Y", "L", "A"):
            assert _close(got[name][0, ty, tx], g[name]), (mode, t, name)
    assert _close(got["whole"][0, 0], whole["lisi"]) and _close(got["whole"][0, 1], whole["auglisi"])
    if mode == "reference":
        # comparison 1 is (x, x): identical images
        assert np.all(got["auglisi"][1] == 1.0) and np.all(got["A"][1] == 0.0)
        assert np.array_equal(got["X"][1], got["Y"][1])
        assert got["whole"][1, 1] == 1.0
    else:
        # comparison 1 is (y, x): the golden values with the roles of x and y swapped
        for t, g in tiles.items():
            ty, tx = divmod(t, 2)
            assert _close(got["X"][1, ty, tx], g["Y"]) and _close(got["Y"][1, ty, tx], g["X"])
            for name in ("lisi", "auglisi", "L", "A"):
                assert _close(got[name][1, ty, tx], g[name]), (t, name)
        assert _close(got["whole"][1, 0], whole["lisi"]) and _close(got["whole"][1, 1], whole["auglisi"])


# ----------------------------------------------------------------------------- S2
@pytest.mark.parametrize("mode", ["reference", "consecutive"])
@pytest.mark.parametrize("seed,N,N_T,M", [(0, 4, 2, 3), (1, 8, 4, 4), (2, 6, 3, 5), (3, 8, 8, 2)])
def test_series_vs_exact_rational(mode, seed, N, N_T, M):
    rng = np.random.default_rng(seed)
    imgs = []
    for _ in range(M):
        a = rng.normal(0.2, 0.5, (N, N)).astype(np.float32)
        a[rng.random((N, N)) < 0.2] = 0.0
        imgs.append(a)
    imgs[-1][: N // 2] = imgs[0][: N // 2]            # equal pixels between first and last
    k = dict(C1=1e-3, C2=1e-4, C=1e-5, D=5e-4)
    got = oracle.series(imgs, mode, N_T, **k)
    nt = N // N_T
    for c in range(M - 1):
        ix = 0 if mode == "reference" else c
        xr, yr = imgs[ix].tolist(), imgs[c + 1].tolist()
        ref = er.tiles(xr, yr, N_T, **{n: np.float32(v) for n, v in k.items()})
        for t, vals in enumerate(ref):
            ty, tx = divmod(t, nt)
            for name, v in zip(("lisi", "auglisi", "X", "Y", "L", "A"), vals):
                f = float(v)
                assert abs(got[name][c, ty, tx] - f) <= 1e-12 * max(abs(f), 1e-30) + 1e-15, (c, t, name)
        w = er.aggregate(ref, np.float32(k["C2"]), np.float32(k["C"]))
        assert abs(got["whole"][c, 0] - float(w[0])) <= 1e-11 * abs(float(w[0])) + 1e-15
        assert abs(got["whole"][c, 1] - float(w[1])) <= 1e-11 * abs(float(w[1])) + 1e-15


# ----------------------------------------------------------------------------- S3, S4
def test_repeated_frames_mark_their_slot_only():
    rng = np.random.default_rng(7)
    a, b, c = (rng.random((16, 16)).astype(np.float32) for _ in range(3))
    k = dict(C1=1e-6, C2=1e-6, C=1e-6, D=5e-7)
    ref = oracle.series([a, b, a, c], "reference", 8, **k)
    assert np.all(ref["auglisi"][1] == 1.0)
    assert np.all(ref["auglisi"][0] < 1.0) and np.all(ref["auglisi"][2] < 1.0)
    con = oracle.series([a, b, b, c], "consecutive", 8, **k)
    assert np.all(con["auglisi"][1] == 1.0)
    assert np.all(con["auglisi"][0] < 1.0) and np.all(con["auglisi"][2] < 1.0)


def test_modes_agree_on_first_comparison_and_differ_after():
    rng = np.random.default_rng(8)
    imgs = [rng.random((8, 8)).astype(np.float32) for _ in range(4)]
    k = dict(C1=1e-6, C2=1e-6, C=1e-6, D=5e-7)
    ref = oracle.series(imgs, "reference", 4, **k)
    con = oracle.series(imgs, "consecutive", 4, **k)
    for name in ("lisi", "auglisi", "X", "Y", "L", "A"):
        assert np.array_equal(ref[name][0], con[name][0])
    # X of comparison k: the reference image in one mode, the predecessor in the other
    assert np.array_equal(ref["X"][2], ref["X"][0])
    assert np.array_equal(con["X"][2], con["Y"][1])
    assert not np.array_equal(ref["X"][2], con["X"][2])
    assert oracle.comparison_indices(4, "reference") == [(0, 1), (0, 2), (0, 3)]
    assert oracle.comparison_indices(4, "consecutive") == [(0, 1), (1, 2), (2, 3)]
    with pytest.raises(ValueError):
        oracle.comparison_indices(1, "reference")
    with pytest.raises(ValueError):
        oracle.comparison_indices(3, "pairs")


# ----------------------------------------------------------------------------- C1
def test_candidates_hand_written():
    v = [0.9, 0.2, 0.5, 0.2, 1.0, -0.5, 0.2]
    idx, val = oracle.bottom_k(v, 4)
    assert idx.tolist() == [5, 1, 3, 6]                       # ties by ascending tile index
    assert val.tolist() == [np.float32(-0.5)] + [np.float32(0.2)] * 3
    assert oracle.bottom_k(v, 0)[0].size == 0
    assert oracle.bottom_k(v, 100)[0].tolist() == [5, 1, 3, 6, 2, 0, 4]
    assert oracle.bottom_k([0.0, -0.0, 0.0], 3)[0].tolist() == [0, 1, 2]     # -0 == +0: index order
    assert oracle.below_threshold(v, 0.5).tolist() == [1, 3, 5, 6]           # strict <
    assert oracle.below_threshold(v, -1.0).size == 0
    assert oracle.below_threshold(v, 2.0).tolist() == list(range(7))
    # the threshold is compared in fp32: 0.2 (double) rounds to the same fp32 as the entries
    assert oracle.below_threshold(np.float32([0.2]), 0.2).size == 0


# ----------------------------------------------------------------------------- C2
@pytest.mark.parametrize("seed,n,k", [(0, 50, 7), (1, 256, 256), (2, 1000, 33), (3, 17, 1)])
def test_candidates_vs_python_selection_loop(seed, n, k):
    rng = np.random.default_rng(seed)
    v = np.round(rng.random(n), 2).astype(np.float32)        # two decimals: many ties
    idx, val = oracle.bottom_k(v, k)
    taken, expect = set(), []
    for _ in range(min(k, n)):                                # repeated minimum search
        best = None
        for i in range(n):
            if i in taken:
                continue
            if best is None or v[i] < v[best]:
                best = i
        taken.add(best)
        expect.append(best)
    assert idx.tolist() == expect
    assert np.array_equal(val, v[expect])
    thr = np.float32(0.25)
    assert oracle.below_threshold(v, thr).tolist() == [i for i in range(n) if v[i] < thr]


# ----------------------------------------------------------------------------- C3 (soft)
def test_bottom_k_finds_the_dropped_sources():
    """Echo of PAPER.md:70: the bottom-k augLISI tiles of a config-[0] pair hold the removed sources."""
    x, y, meta = synth.make_pair(synth.CONFIGS[0])
    cfg, src = meta["cfg"], meta["sources"]
    t = oracle.tiles(x, y, cfg.N_T, cfg.C1, cfg.C2, cfg.C, cfg.D)
    dropped = np.nonzero((src["amp_y"] == 0) & (src["amp_x"] > 0))[0]
    nt = cfg.N // cfg.N_T
    tiles = {int(src["cy"][i]) // cfg.N_T * nt + int(src["cx"][i]) // cfg.N_T for i in dropped}
    idx, val = oracle.bottom_k(t["auglisi"].astype(np.float32), 3 * len(tiles))
    assert np.all(np.diff(val) >= 0) and len(set(idx.tolist())) == idx.size
    assert len(tiles & set(idx.tolist())) >= max(1, len(tiles) - 2)


# ----------------------------------------------------------------------------- series generator
def test_series_generator_is_seeded_and_switches_only_the_transients():
    cfg = synth.CONFIGS[0]
    a, ma = synth.make_series(cfg, 4)
    b, _ = synth.make_series(cfg, 4)
    assert len(a) == 4 and all(i.dtype == np.float32 and i.shape == (256, 256) for i in a)
    assert all(np.array_equal(p, q) for p, q in zip(a, b))
    assert ma["state_y"].shape == (4, cfg.n_drop) and not ma["state_y"][0].any()
    assert ma["state_y"][1:].any()
    # snapshots differ from snapshot 0 by noise everywhere and by a source where a transient is off
    src, ch = ma["sources"], ma["changed"]
    for j in range(1, 4):
        diff = np.abs(a[j] - a[0])
        assert np.median(diff) < 10 * cfg.noise_sigma
        for i, off in zip(ch, ma["state_y"][j]):
            cy, cx = int(src["cy"][i]), int(src["cx"][i])
            peak = diff[max(0, cy - 1):cy + 2, max(0, cx - 1):cx + 2].max()
            if off and src["amp_x"][i] > 20 * cfg.noise_sigma:
                assert peak > 0.5 * src["amp_x"][i]
    with pytest.raises(ValueError):
        synth.make_series(cfg, 1)
