"""Writes tests/golden/worked_example_4x4.txt.

The paper (arxiv 2501.10653) prints no worked example, so this fixture is DERIVED from its
equations with exact rational arithmetic: Eq. 1, Eq. 2,
the clamp, the tile layout and Eqs. 3-4.
It calls only ``oracle/exact_rational.py`` (never the CUDA path, never the C++ oracle);
several of the values are re-derived by hand in tests/test_oracle_pins.py.

Run from the repo root:  python tests/golden/make_worked_example.py
"""
import os
import sys
from fractions import Fraction

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.abspath(os.path.join(HERE, "..", "..")))

from oracle import exact_rational as er  # noqa: E402

X_ROWS = [[1, 0.5, -1, 0], [0.25, 0, 0, 0], [0.75, 0.75, 2, -0.5], [0.125, 0.5, 0, 1]]
Y_ROWS = [[1, 0.25, 3, -2], [0, 0.5, 0, 0], [0.75, 0.75, 0, 0.5], [0.125, 0.5, 1, 0]]
C1 = C2 = C = 2.0 ** -20
D = 2.0 ** -21          # = C1/2 (reading R1)


def _fmt(fr: Fraction) -> str:
    return f"{fr.numerator}/{fr.denominator}"


def main():
    lines = [
        "# Worked example for tile-wise LISI / augLISI -- derived, not printed by the paper.",
        "# Source: exact rationals from Eq. 1 (PAPER.md:15-17), Eq. 2 (PAPER.md:19-21), clamp (PAPER.md:27),",
        "# tiles (PAPER.md:62-64), Eqs. 3-4 (PAPER.md:55-60).  Written by tests/golden/make_worked_example.py.",
        "# N=4, N_T=2, C1=C2=C=2^-20, D=2^-21.  Rows of x / y below; then one line per tile",
        "# (t = ty*2+tx) and a 'whole' line (N_T=4 == Eqs. 3-4 over the four tiles, equal as rationals).",
        "# Each value is 'numerator/denominator' (exact) -- convert with float(Fraction(...)).",
    ]
    for name, rows in (("x", X_ROWS), ("y", Y_ROWS)):
        for r in rows:
            lines.append(f"{name} " + " ".join(repr(float(v)) for v in r))
    per_tile = er.tiles(X_ROWS, Y_ROWS, 2, C1, C2, C, D)
    for t, (lisi, aug, X, Y, L, A) in enumerate(per_tile):
        lines.append(f"tile {t} lisi={_fmt(lisi)} auglisi={_fmt(aug)} X={_fmt(X)} Y={_fmt(Y)} "
                     f"L={_fmt(L)} A={_fmt(A)}")
    whole = er.lisi_auglisi(X_ROWS, Y_ROWS, C1, C2, C, D)
    agg = er.aggregate(per_tile, C2, C)
    assert agg[0] == whole[0] and agg[1] == whole[1], "Eqs. 3-4 must reproduce the whole image exactly"
    lisi, aug, X, Y, L, A = whole
    lines.append(f"whole lisi={_fmt(lisi)} auglisi={_fmt(aug)} X={_fmt(X)} Y={_fmt(Y)} "
                 f"L={_fmt(L)} A={_fmt(A)}")
    with open(os.path.join(HERE, "worked_example_4x4.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")
    for ln in lines[-5:]:
        print(ln[:160])


if __name__ == "__main__":
    main()
