"""Writes tests/golden/laplace_minimax.txt: minimax exponential-sum grids for 1/x on [0.4, 4.5] (the Laplace interval
of every BASELINE.json config; Eq. 11) for k = 8, 10, 12 points, computed by the CPU ORACLE ONLY
(oracle.laplace_minimax, 80-digit Remez).  The paper prints no grid (SI S4 is not available), so these values are
the oracle's; they are pinned by the equi-oscillation certificate in tests/test_oracle_laplace.py, not by a number
from the paper.

    python tests/golden/make_laplace_golden.py        (takes ~15 min)
"""
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent.parent
sys.path.insert(0, str(ROOT))
from oracle import oracle as O  # noqa: E402

XMIN, XMAX = 0.4, 4.5


def main():
    out = ["# minimax grids for 1/x on [%r, %r]; written by tests/golden/make_laplace_golden.py (oracle only)" % (XMIN, XMAX),
           "# record: k <k> delta <max abs error>; then k lines 'tau w'; then 2k+1 alternation points"]
    for k in (8, 10, 12):
        tau, w, delta, xs = O.laplace_minimax(XMIN, XMAX, k)
        out.append("k %d delta %.17e" % (k, delta))
        for t, ww in zip(tau, w):
            out.append("%.17e %.17e" % (t, ww))
        out.append(" ".join("%.17e" % x for x in xs))
    (Path(__file__).resolve().parent / "laplace_minimax.txt").write_text("\n".join(out) + "\n")


if __name__ == "__main__":
    main()
