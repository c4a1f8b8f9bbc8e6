"""Helpers for the -m gpu parity tests: run the CUDA path through the binding, run the oracle
on the same fp32 buffers, compare element by element with the tolerance DESIGN.md derives.

Tolerance (BASELINE.json north_star: relative error <= 1e-5 per tile):
  X, Y, L, A, lisi : |got - ref| <= 1e-5 * |ref|            (sums of non-negative terms)
  auglisi = 1 - r  : |got - ref| <= 1e-5 * |ref| + 1e-6 * r  with r = A / (X + Y + C) from the oracle;
                     the second term only matters when auglisi is near 0 (cancellation), which
                     never happens on the BASELINE.json skies (r <= ~0.1 there).
"""
from __future__ import annotations

import numpy as np
import torch

import oracle
from paper_2501_10653_b200 import binding

RTOL = 1e-5


def consts(cfg):
    return dict(C1=cfg.C1, C2=cfg.C2, C=cfg.C, D=cfg.D)


def to_dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def run_gpu(xd, yd, N_T, k, numerators=True):
    out = binding.fused_tiles(xd, yd, N_T, k["C1"], k["C2"], k["C"], k["D"], numerators=numerators)
    torch.cuda.synchronize()
    return {n: v.cpu().numpy().astype(np.float64) for n, v in out.items()}


def run_oracle(x, y, N_T, k):
    return oracle.tiles(x, y, N_T, k["C1"], k["C2"], k["C"], k["D"])


def rel_err(got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    den = np.where(ref == 0.0, 1.0, np.abs(ref))
    return np.abs(got - ref) / den


def assert_parity(got: dict, ref: dict, C, what=""):
    """Element-by-element comparison of every array the GPU returned."""
    report = {}
    for name in got:
        g, r = got[name], ref[name]
        assert g.shape == r.shape, (what, name, g.shape, r.shape)
        assert np.all(np.isfinite(g)), (what, name, "non-finite output")
        err = np.abs(g - r)
        tol = RTOL * np.abs(r)
        if name == "auglisi":
            ratio = ref["A"] / (ref["X"] + ref["Y"] + float(np.float32(C)))
            tol = tol + 1e-6 * ratio
        bad = err > tol
        report[name] = float(np.max(rel_err(g, r))) if g.size else 0.0
        assert not bad.any(), (what, name, int(bad.sum()), "worst rel", report[name],
                               "at", np.unravel_index(np.argmax(err - tol), g.shape))
    return report


def check_pair(x, y, N_T, k, what="", xd=None, yd=None):
    """x, y: host fp32 arrays (source of truth).  Returns (gpu, oracle, report)."""
    xd = to_dev(x) if xd is None else xd
    yd = to_dev(y) if yd is None else yd
    got = run_gpu(xd, yd, N_T, k)
    ref = run_oracle(x, y, N_T, k)
    rep = assert_parity(got, ref, k["C"], what)
    return got, ref, rep
