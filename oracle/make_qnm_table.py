"""Writes oracle/qnm_220_table.txt: the Kerr (2,2,0) quasi-normal mode on a grid of spins, from oracle.qnm.kerr_qnm_220
(Leaver's continued fractions).  Calls only oracle/.  Run:  python -m oracle.make_qnm_table

The grid is uniform in y = sqrt(1 - a/M) (the mode varies fastest towards the extremal hole), 401 nodes from a/M = -0.998
to +0.998; oracle.qnm.qnm_220 interpolates it with a cubic spline (interpolation error < 1e-8, tests/test_oracle_qnm.py).
"""
import numpy as np

from oracle import qnm


def main():
    y = np.linspace(np.sqrt(1.0 - 0.998), np.sqrt(1.0 + 0.998), 401)
    spins = np.sort(1.0 - y * y)
    i0 = int(np.argmin(np.abs(spins)))
    rows = {}
    # walk outwards from the node nearest to zero spin, each solve starting from its neighbour's solution
    w, sep = qnm.kerr_qnm_220(spins[i0])
    rows[i0] = (w, sep)
    for order in (range(i0 + 1, len(spins)), range(i0 - 1, -1, -1)):
        prev = i0
        for i in order:
            w0, s0 = rows[prev]
            w, sep = qnm.kerr_qnm_220(spins[i], start=(spins[prev], w0, s0))
            rows[i] = (w, sep)
            prev = i
    with open(qnm.TABLE_PATH, "w") as fh:
        fh.write("# Kerr l = m = 2, n = 0 quasi-normal mode: a/M, Re(M omega), -Im(M omega); written by oracle/make_qnm_table.py\n")
        fh.write("# from Leaver's continued fractions (oracle/qnm.py); ref. [32] of the paper (PAPER.md:344) uses this function\n")
        for i, a in enumerate(spins):
            fh.write("%.16e %.16e %.16e\n" % (a, rows[i][0].real, -rows[i][0].imag))


if __name__ == "__main__":
    main()
