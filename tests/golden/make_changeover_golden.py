"""Regenerates tests/golden/changeover_fig3.txt's value rows from oracle/ only (run from the repo root)."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import oracle  # noqa: E402

if __name__ == "__main__":
    lam = 9.0 / 11.0
    for x in (0.0, 0.10, 0.25, 0.50, 0.75, 0.90, 1.0):
        print(f"{x:.2f} {oracle.K(x, lam):.12f} {oracle.W(x, lam):.12f}")
