"""CPU oracle for tile-wise LISI / augLISI -- TEST INFRASTRUCTURE ONLY.

Thin ctypes loader around ``oracle/iqa_oracle.cpp`` (the plain definition of
Eqs. 1-4 of arxiv 2501.10653, double accumulation) plus ``exact_rational`` (a
second, deliberately different brute-force implementation with exact rationals,
usable on tiny images only).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product path
(``paper_2501_10653_b200``) never does, and this package never imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

os.environ.setdefault("OMP_WAIT_POLICY", "passive")   # idle OpenMP threads sleep instead of spinning

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "iqa_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle_iqa.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the C++ oracle with g++ (-O2, OpenMP, no fast-math). Returns the .so path."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
           "-o", _LIB, _SRC]
    subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        fp = ctypes.POINTER(ctypes.c_float)
        lib.iqa_oracle_tiles.restype = ctypes.c_int
        lib.iqa_oracle_tiles.argtypes = [fp, fp, ctypes.c_long, ctypes.c_long,
                                         ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                         ctypes.c_double, dp, dp, dp, dp, dp, dp, ctypes.c_int]
        lib.iqa_oracle_tiles_2d.restype = ctypes.c_int
        lib.iqa_oracle_tiles_2d.argtypes = [fp, fp, ctypes.c_long, ctypes.c_long, ctypes.c_long, ctypes.c_long,
                                            ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                            ctypes.c_double, dp, dp, dp, dp, dp, dp, ctypes.c_int]
        lib.iqa_oracle_tiles_2d_f64.restype = ctypes.c_int
        lib.iqa_oracle_tiles_2d_f64.argtypes = [dp, dp, ctypes.c_long, ctypes.c_long, ctypes.c_long, ctypes.c_long,
                                                ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                                ctypes.c_double, dp, dp, dp, dp, dp, dp, ctypes.c_int]
        lib.iqa_oracle_aggregate.restype = ctypes.c_int
        lib.iqa_oracle_aggregate.argtypes = [dp, dp, dp, dp, ctypes.c_long,
                                             ctypes.c_double, ctypes.c_double, dp]
        lib.iqa_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _cpu_budget() -> int:
    """CPUs this process may actually use: scheduler affinity capped by the cgroup CPU quota.
    (OpenMP's own default ignores the quota; oversubscribed spinning threads are very slow.)"""
    n = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    for path in ("/sys/fs/cgroup/cpu.max", "/sys/fs/cgroup/cpu/cpu.cfs_quota_us"):
        try:
            with open(path) as f:
                parts = f.read().split()
            if path.endswith("cpu.max"):
                if parts[0] != "max":
                    n = min(n, max(1, int(int(parts[0]) / int(parts[1]))))
            else:
                quota = int(parts[0])
                if quota > 0:
                    with open("/sys/fs/cgroup/cpu/cpu.cfs_period_us") as g:
                        n = min(n, max(1, quota // int(g.read().split()[0])))
            break
        except (OSError, ValueError, IndexError):
            continue
    return max(1, n)


def max_threads() -> int:
    """Threads the oracle uses by default: min(OpenMP default, usable CPUs)."""
    return max(1, min(int(_load().iqa_oracle_max_threads()), _cpu_budget()))


def _f32c(a) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float32)
    if a.ndim != 2 or a.shape[0] != a.shape[1]:
        raise ValueError("oracle expects a square 2-D image")
    return a


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def tiles(x, y, N_T: int, C1, C2, C, D, threads: int = 0) -> dict:
    """Per-tile Eq. 1 / Eq. 2 of two N x N fp32 images (clamp P:27).

    Constants are first rounded to fp32 (the C ABI of the CUDA library takes ``float``),
    then promoted to double, so both sides use bit-identical constants.
    Returns a dict of (N/N_T, N/N_T) float64 arrays: lisi, auglisi, X, Y, L, A.
    """
    x = _f32c(x)
    y = _f32c(y)
    if x.shape != y.shape:
        raise ValueError("x and y must have the same shape")
    N = x.shape[0]
    if N_T <= 0 or N % N_T:
        raise ValueError("N must be a multiple of N_T (P:64)")
    nt = N // N_T
    out = {k: np.empty((nt, nt), dtype=np.float64)
           for k in ("lisi", "auglisi", "X", "Y", "L", "A")}
    fp = ctypes.POINTER(ctypes.c_float)
    rc = _load().iqa_oracle_tiles(
        x.ctypes.data_as(fp), y.ctypes.data_as(fp), N, N_T,
        float(np.float32(C1)), float(np.float32(C2)), float(np.float32(C)), float(np.float32(D)),
        _dptr(out["lisi"]), _dptr(out["auglisi"]), _dptr(out["X"]), _dptr(out["Y"]),
        _dptr(out["L"]), _dptr(out["A"]), int(threads) if threads > 0 else max_threads())
    if rc != 0:
        raise RuntimeError(f"iqa_oracle_tiles failed with code {rc}")
    return out


def tiles_2d(x, y, N_T: int, C1, C2, C, D, threads: int = 0) -> dict:
    """Per-tile Eq. 1 / Eq. 2 of two H x W fp32 images with EDGE TILES (reading R18):
    the tile grid is ceil(H/N_T) x ceil(W/N_T), cells over the border hold only the pixels that exist.
    x, y: 2-D float32 arrays whose rows are contiguous; a row stride (pitch) larger than W is allowed
    (e.g. a column slice of a wider array) and is passed through, not copied away.
    Returns (nty, ntx) float64 arrays: lisi, auglisi, X, Y, L, A."""
    def prep(a):
        a = np.asarray(a)
        if a.dtype != np.float32 or a.ndim != 2:
            raise ValueError("need 2-D float32 arrays")
        if a.strides[1] != 4 or a.strides[0] % 4 or a.strides[0] < 4 * a.shape[1]:
            a = np.ascontiguousarray(a)
        return a
    x, y = prep(x), prep(y)
    if x.shape != y.shape:
        raise ValueError("x and y must have the same shape")
    H, W = x.shape
    if N_T <= 0:
        raise ValueError("N_T must be positive")
    nty, ntx = -(-H // N_T), -(-W // N_T)
    out = {k: np.empty((nty, ntx), dtype=np.float64) for k in ("lisi", "auglisi", "X", "Y", "L", "A")}
    fp = ctypes.POINTER(ctypes.c_float)
    rc = _load().iqa_oracle_tiles_2d(
        ctypes.cast(x.ctypes.data, fp), ctypes.cast(y.ctypes.data, fp), H, W, x.strides[0] // 4, y.strides[0] // 4, N_T,
        float(np.float32(C1)), float(np.float32(C2)), float(np.float32(C)), float(np.float32(D)),
        _dptr(out["lisi"]), _dptr(out["auglisi"]), _dptr(out["X"]), _dptr(out["Y"]),
        _dptr(out["L"]), _dptr(out["A"]), int(threads) if threads > 0 else max_threads())
    if rc != 0:
        raise RuntimeError(f"iqa_oracle_tiles_2d failed with code {rc}")
    return out


PIXEL_DTYPES = (np.float32, np.float64, np.float16, np.int16, np.int32, np.uint8)   # FITS BITPIX -32, -64, (fp16), 16, 32, 8


def tiles_2d_any(x, y, N_T: int, C1, C2, C, D, threads: int = 0) -> dict:
    """``tiles_2d`` for images of any supported pixel type: the pixels are converted to
    double -- exact for every type in ``PIXEL_DTYPES`` -- and Eqs. 1-2 are evaluated in double on those values."""
    x, y = np.asarray(x), np.asarray(y)
    if x.dtype != y.dtype or x.dtype.type not in PIXEL_DTYPES:
        raise ValueError(f"x and y must share one of the pixel types {[t.__name__ for t in PIXEL_DTYPES]}")
    if x.ndim != 2 or x.shape != y.shape:
        raise ValueError("need two equally shaped 2-D images")
    xd = np.ascontiguousarray(x, dtype=np.float64)
    yd = np.ascontiguousarray(y, dtype=np.float64)
    H, W = xd.shape
    if N_T <= 0:
        raise ValueError("N_T must be positive")
    nty, ntx = -(-H // N_T), -(-W // N_T)
    out = {k: np.empty((nty, ntx), dtype=np.float64) for k in ("lisi", "auglisi", "X", "Y", "L", "A")}
    rc = _load().iqa_oracle_tiles_2d_f64(
        _dptr(xd), _dptr(yd), H, W, W, W, N_T,
        float(np.float32(C1)), float(np.float32(C2)), float(np.float32(C)), float(np.float32(D)),
        _dptr(out["lisi"]), _dptr(out["auglisi"]), _dptr(out["X"]), _dptr(out["Y"]),
        _dptr(out["L"]), _dptr(out["A"]), int(threads) if threads > 0 else max_threads())
    if rc != 0:
        raise RuntimeError(f"iqa_oracle_tiles_2d_f64 failed with code {rc}")
    return out


def aggregate(lisi, auglisi, X, Y, C2, C) -> tuple[float, float]:
    """Eqs. 3-4: merge the given tiles into one (LISI, augLISI) pair."""
    arrs = [np.ascontiguousarray(np.asarray(a, dtype=np.float64).ravel())
            for a in (lisi, auglisi, X, Y)]
    n = arrs[0].size
    if any(a.size != n for a in arrs) or n == 0:
        raise ValueError("need four equally sized, non-empty per-tile arrays")
    out2 = np.empty(2, dtype=np.float64)
    rc = _load().iqa_oracle_aggregate(_dptr(arrs[0]), _dptr(arrs[1]), _dptr(arrs[2]),
                                      _dptr(arrs[3]), n, float(np.float32(C2)),
                                      float(np.float32(C)), _dptr(out2))
    if rc != 0:
        raise RuntimeError(f"iqa_oracle_aggregate failed with code {rc}")
    return float(out2[0]), float(out2[1])


from .series import below_threshold, bottom_k, comparison_indices, series  # noqa: E402  (time series, candidates)
