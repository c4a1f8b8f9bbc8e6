"""CPU oracle for the TIME-SERIES mode and for candidate extraction -- TEST INFRASTRUCTURE ONLY.

Both are the plain definitions, written out step by step:

``series``  A time series of M images I_0 .. I_{M-1} of one field ("intensity variations between
    observations of the same section of the sky"; "the rest of the image remains
    largely stable with slight variations over time") gives K = M - 1 comparisons,
    each of them exactly the pair computation of Eqs. 1-4 (clamp PAPER.md:27):
        reference   comparison k is (x, y) = (I_0, I_{k+1})   -- every snapshot against one reference
        consecutive comparison k is (x, y) = (I_k, I_{k+1})   -- every snapshot against its predecessor
    The oracle literally calls the pair oracle K times; nothing is shared between comparisons.

``below_threshold`` / ``bottom_k``  The paper gives no decision rule (it shows the matrices and
    says the finders localise "transients to tiles"), so the rule is the plainest one
    (reading R17): flag the tiles whose value is below a user threshold (listed in
    ascending tile index), or the k tiles of lowest value (ordered by ascending value, ties by
    ascending tile index).  Values are compared as the fp32 numbers they are.

Pins (tests/test_oracle_series_pins.py): the worked example embedded in a series, exact-rational
brute force per comparison, mode-distinguishing sequences, hand-written candidate lists and a
pure-Python selection loop -- nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

MODES = ("reference", "consecutive")


def comparison_indices(n_images: int, mode: str) -> list:
    """[(index of x, index of y)] for the K = n_images - 1 comparisons of a series."""
    if mode not in MODES:
        raise ValueError(f"mode must be one of {MODES}")
    if n_images < 2:
        raise ValueError("a series needs at least two images")
    if mode == "reference":
        return [(0, k + 1) for k in range(n_images - 1)]
    return [(k, k + 1) for k in range(n_images - 1)]


def series(images, mode: str, N_T: int, C1, C2, C, D, threads: int = 0) -> dict:
    """Per-tile Eqs. 1-2 and whole-image Eqs. 3-4 for every comparison of a series.

    Returns float64 arrays lisi, auglisi, X, Y, L, A of shape (K, nt, nt) and ``whole`` (K, 2).
    """
    from . import aggregate, tiles          # the pair oracle (iqa_oracle.cpp)
    pairs = comparison_indices(len(images), mode)
    per = []
    whole = []
    for ix, iy in pairs:
        t = tiles(images[ix], images[iy], N_T, C1, C2, C, D, threads=threads)
        per.append(t)
        whole.append(aggregate(t["lisi"], t["auglisi"], t["X"], t["Y"], C2, C))
    out = {k: np.stack([t[k] for t in per]) for k in ("lisi", "auglisi", "X", "Y", "L", "A")}
    out["whole"] = np.asarray(whole, dtype=np.float64)
    return out


def below_threshold(values, threshold) -> np.ndarray:
    """Indices (ascending) of the tiles whose fp32 value is < the fp32 threshold. int32."""
    v = np.asarray(values, dtype=np.float32).ravel()
    thr = np.float32(threshold)
    return np.flatnonzero(v < thr).astype(np.int32)


def bottom_k(values, k: int):
    """The k tiles of lowest fp32 value, ascending by (value, tile index).

    Returns (indices int32 [k'], values float32 [k']) with k' = min(k, number of tiles).
    NaN never occurs in the matrices (C2, C > 0 keep every tile finite); it is rejected here.
    """
    v = np.asarray(values, dtype=np.float32).ravel()
    if np.isnan(v).any():
        raise ValueError("NaN in the matrix")
    if k < 0:
        raise ValueError("k must be >= 0")
    order = np.lexsort((np.arange(v.size), v))          # primary key v, ties by index
    idx = order[: min(k, v.size)].astype(np.int32)
    return idx, v[idx]
