"""Exact-rational brute force for Eqs. 1-4 of arxiv 2501.10653 -- TEST INFRASTRUCTURE ONLY.

A second oracle, deliberately different from ``iqa_oracle.cpp``: pure-Python loops over
``fractions.Fraction`` values built from the exact fp32 bit patterns, so there is no
rounding anywhere.  Usable on tiny images only (<= ~32 x 32).  It validates the C++
oracle (tests/test_oracle_pins.py, pin P2) and writes the worked example under
``tests/golden/`` (pin P1).  It is itself pinned by values derived by hand in that test.

Citations: Eq. 1, Eq. 2, clamp P:27, tiles P:62-64, Eqs. 3-4 P:55-60.
"""
from __future__ import annotations

import math
from fractions import Fraction


def _clamp(v: float) -> Fraction:
    # negative pixels -> 0.  NaN -> 0 as well (reading R3 in DESIGN.md).
    if v != v or v <= 0.0:
        return Fraction(0)
    if math.isinf(v):
        raise ValueError("+Inf pixels are outside the contract")
    return Fraction(v)            # exact: every finite float is a dyadic rational


def tile_sums(x_rows, y_rows):
    """Return exact (L, A, X, Y) over all pixels of the given equally shaped 2-D lists.
    C1 enters L, so L is returned as a function: call ``L(C1)``."""
    pix = []
    for xr, yr in zip(x_rows, y_rows):
        for xv, yv in zip(xr, yr):
            pix.append((_clamp(float(xv)), _clamp(float(yv))))
    X = sum((p[0] for p in pix), Fraction(0))
    Y = sum((p[1] for p in pix), Fraction(0))
    A = sum((abs(p[0] + p[1]) * abs(p[0] - p[1]) for p in pix), Fraction(0))

    def L(C1: Fraction) -> Fraction:
        return sum((abs(p[0] + p[1]) / (abs(p[0] - p[1]) + C1) for p in pix), Fraction(0))

    return L, A, X, Y


def lisi_auglisi(x_rows, y_rows, C1, C2, C, D):
    """Eq. 1 and Eq. 2 over ALL pixels of x_rows / y_rows. Returns exact Fractions
    (lisi, auglisi, X, Y, L, A)."""
    C1, C2, C, D = (Fraction(float(v)) for v in (C1, C2, C, D))
    Lf, A, X, Y = tile_sums(x_rows, y_rows)
    L = Lf(C1)
    lisi = D * L / (max(X, Y) + C2)
    auglisi = 1 - A / (X + Y + C)
    return lisi, auglisi, X, Y, L, A


def tiles(x_rows, y_rows, N_T: int, C1, C2, C, D):
    """Per-tile values, row-major list of tuples (lisi, auglisi, X, Y, L, A); t = ty*(N/N_T)+tx."""
    N = len(x_rows)
    assert N % N_T == 0 and all(len(r) == N for r in x_rows) and len(y_rows) == N
    nt = N // N_T
    out = []
    for ty in range(nt):
        for tx in range(nt):
            xs = [row[tx * N_T:(tx + 1) * N_T] for row in x_rows[ty * N_T:(ty + 1) * N_T]]
            ys = [row[tx * N_T:(tx + 1) * N_T] for row in y_rows[ty * N_T:(ty + 1) * N_T]]
            out.append(lisi_auglisi(xs, ys, C1, C2, C, D))
    return out


def aggregate(per_tile, C2, C):
    """Eqs. 3-4 over a list of per-tile tuples as returned by ``tiles``. Exact Fractions."""
    C2, C = Fraction(float(C2)), Fraction(float(C))
    n = len(per_tile)
    SX = sum((t[2] for t in per_tile), Fraction(0))
    SY = sum((t[3] for t in per_tile), Fraction(0))
    num3 = sum((t[0] * (max(t[2], t[3]) + C2) for t in per_tile), Fraction(0))
    num4 = sum((t[1] * (t[2] + t[3] + C) for t in per_tile), Fraction(0)) - (n - 1) * C
    return num3 / (max(SX, SY) + C2), num4 / (SX + SY + C)
