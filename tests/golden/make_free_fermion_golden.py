"""Writes tests/golden/free_fermion_closed_form.txt from the theta = 0 closed form (mathematics, no oracle and no
CUDA code involved): at theta = 0 the x- and y-sweeps of Eq.22 commute, B = Bx (x) By, and on the
2-site unit cell E2(a/2) E1(a) E2(a/2) has eigenvalues exp(+-lambda(k)), cosh lambda = cosh^2(dtau) + sinh^2(dtau)
cos 2k, k = 2 pi m / L.  With M of Eq.8 (antiperiodic in tau): spec(M^+M) = {1 + b^2 - 2 b cos w_n},
w_n = (2n+1) pi / Ntau, and log det M = sum_b log(1 + b^Ntau)  (Eq.7).

    python tests/golden/make_free_fermion_golden.py
"""
import os

import numpy as np

DTAU = 0.1
CASES = [(4, 8), (6, 10), (8, 8), (12, 120)]


def closed_form(L, Nt, dtau=DTAU):
    ks = 2 * np.pi * np.arange(L // 2) / L
    lam = np.arccosh(np.maximum(1.0, np.cosh(dtau) ** 2 + np.sinh(dtau) ** 2 * np.cos(2 * ks)))
    b = np.array([np.exp(sx * lx + sy * ly) for lx in lam for ly in lam for sx in (1, -1) for sy in (1, -1)])
    w = (2 * np.arange(Nt) + 1) * np.pi / Nt
    spec = 1 + b[:, None] ** 2 - 2 * b[:, None] * np.cos(w[None, :])
    # log(1 + b^Nt) without overflow
    logdet = np.sum(np.logaddexp(0.0, Nt * np.log(b)))
    return logdet, spec.min(), spec.max(), spec.sum()


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "free_fermion_closed_form.txt")
    with open(out, "w") as f:
        f.write("# theta = 0 closed form of M (PAPER.md:155 Eq.8) with B of PAPER.md:298 Eq.22, dtau = 0.1, t = 1\n")
        f.write("# written by tests/golden/make_free_fermion_golden.py (numpy only)\n")
        f.write("# L Ntau log_det_M lambda_min(M^+M) lambda_max(M^+M) trace(M^+M)\n")
        for L, Nt in CASES:
            ld, lo, hi, tr = closed_form(L, Nt)
            f.write(f"{L} {Nt} {ld:.15e} {lo:.15e} {hi:.15e} {tr:.15e}\n")
    print(open(out).read())
