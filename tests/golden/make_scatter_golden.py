"""Writes tests/golden/scatter_fit_T200_N128_n16.txt: the oracle's (scipy L-BFGS-B) minimum loss and its prediction
at 400 sampled (t, i, j) for the 200-frame scattered-light problem of tests/test_gpu_scatter.py.  Calls only
oracle/ and the seeded problem generator in tests/helpers.py (never the CUDA path); takes about 15 minutes.
Run: python tests/golden/make_scatter_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "..", ".."))
sys.path.insert(0, os.path.join(HERE, ".."))
import oracle                          # noqa: E402
from helpers import scatter_problem    # noqa: E402


def main():
    T, N, n = 200, 128, 16
    D, jit, _, _ = scatter_problem(21, T, N, n)
    ob, oS, oL = oracle.scatter_fit(D, jit, 1.0, n, max_iter=3000)
    pred = oracle.upsample(oS, N) + np.einsum("tk,kij->tij", oracle.background_basis(jit), ob)
    rng = np.random.default_rng(0)
    t, i, j = rng.integers(T, size=400), rng.integers(N, size=400), rng.integers(N, size=400)
    out = os.path.join(HERE, "scatter_fit_T200_N128_n16.txt")
    with open(out, "w") as fh:
        fh.write("# written by tests/golden/make_scatter_golden.py (oracle/ + the seeded generator only)\n")
        fh.write("# first row: 0 0 0 minimum loss; then t i j prediction of the oracle's minimiser\n")
        fh.write("0 0 0 %.17g\n" % oL)
        for a, b, c in zip(t, i, j):
            fh.write("%d %d %d %.17g\n" % (a, b, c, pred[a, b, c]))
    print("wrote", out, "loss", oL)


if __name__ == "__main__":
    main()
