"""CPU ORACLE for the stochastic estimation of fermionic observables.  TEST INFRASTRUCTURE ONLY.

Only tests/ (and bench.py's cpu_baseline leg) may import this.  Plain numpy, complex128, written in the paper's order
and notation; it never imports the CUDA package.  Lattice vectors are arrays [N_tau][L][L] (tau, y, x), the same
layout as everywhere else in this repository.

What the paper fixes:
  * PAPER.md:226-230  unbiased estimate of M^{-1}:  sum_l [M^{-1}]_il xi_l xi_j^*,  computed in practice as
                      G xi = (M^+ M)^{-1} R,  R := M^+ xi,  with the pCG of Eq.20                       -> green_apply
  * PAPER.md:232-236  (Eq.17)  C(Delta) = (1/N) sum_i C(i, i + Delta),  N = V_s N_tau                   -> translation_average_direct
  * PAPER.md:238-244  (Eq.18, 19)  C^(i,j) = a_i b_j;  C^(Delta) = F^{-1}[F[a]_{-k} F[b]_k](Delta)       -> translation_average_fft
  * PAPER.md:240, 244 two-point estimate  G^_ij = [G xi]_i xi_j^*;  example C(i,j) = G_ij G_ij with
                      a_i = (G xi)_i (G xi')_i,  b_j = xi_j^* xi'_j^*,  every unordered pair of the N_rv
                      vectors used once: binom(N_rv, 2) samples                                        -> green_2pt, pair_correlator

Readings: C23 "i + Delta" is taken periodically in all three directions, exactly as Eq.19's FFT
does (the paper prints no boundary sign for the temporal wrap of odd-fermion-number correlators); C24 the FFT of Eq.19
is the unnormalised forward DFT with e^{-ik.x}, the inverse carries 1/N, and the 1/N of Eq.17 is applied on top.

Pins (tests/test_oracle_measure.py): Eq.17 written as an O(N^2) double loop against Eq.19 through numpy's FFT (two
different formulas); delta-function inputs (closed form); the full-basis identity -- averaging the estimator over the
N vectors sqrt(N) e_l reproduces the translation average of the dense numpy inverse of the dense M of tests/dense_ref.py
exactly; the pair correlator against Eq.18 + Eq.17 evaluated pair by pair with explicit loops.
"""
from __future__ import annotations

import itertools

import numpy as np


def translation_average_direct(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    """Eq.17 with C(i,j) = a_i b_j (Eq.18), literally: C(Delta) = (1/N) sum_i a_i b_{i+Delta}.  O(N^2): small lattices."""
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    Nt, Ly, Lx = a.shape
    N = a.size
    C = np.zeros_like(a)
    for dt in range(Nt):
        for dy in range(Ly):
            for dx in range(Lx):
                s = 0.0 + 0.0j
                for t in range(Nt):
                    for y in range(Ly):
                        for x in range(Lx):
                            s += a[t, y, x] * b[(t + dt) % Nt, (y + dy) % Ly, (x + dx) % Lx]
                C[dt, dy, dx] = s / N
    return C


def _minus_k(F: np.ndarray) -> np.ndarray:
    """F[a]_{-k}: index k -> (-k) mod n along every axis."""
    for ax in range(F.ndim):
        F = np.roll(np.flip(F, axis=ax), 1, axis=ax)
    return F


def translation_average_fft(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    """Eq.19: C^(Delta) = (1/N) sum_i a_i b_{i+Delta} = (1/N) F^{-1}[ F[a]_{-k} . F[b]_k ](Delta)   (reading C24)."""
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    Fa = np.fft.fftn(a)
    Fb = np.fft.fftn(b)
    return np.fft.ifftn(_minus_k(Fa) * Fb) / a.size


def green_apply(orc, theta, xi, tol: float = 1e-12, max_iter: int = 1000000):
    """G xi = (M^+ M)^{-1} R with R := M^+ xi, by the pCG of Eq.20.  `orc` is an oracle.Oracle.
    Returns (G xi, iterations)."""
    R = orc.apply_Mdag(theta, xi)
    g, it, _ = orc.pcg(theta, R, tol, max_iter)
    return g, it


def green_2pt(gs, xis) -> np.ndarray:
    """Translation average of the two-point estimate G^_ij = [G xi]_i xi_j^* (PAPER.md:240), mean over the vectors."""
    acc = np.zeros_like(np.asarray(gs[0], dtype=np.complex128))
    for g, xi in zip(gs, xis):
        acc += translation_average_fft(g, np.conj(xi))
    return acc / len(gs)


def pair_correlator(gs, xis) -> np.ndarray:
    """The paper's example C(i,j) = G_ij G_ij: a_i = (G xi)_i (G xi')_i, b_j = xi_j^* xi'_j^*, Eq.19 per
    pair, mean over the binom(N_rv, 2) unordered pairs (xi, xi').  Pairs in lexicographic order."""
    n = len(gs)
    acc = np.zeros_like(np.asarray(gs[0], dtype=np.complex128))
    npair = 0
    for k, kp in itertools.combinations(range(n), 2):
        a = np.asarray(gs[k]) * np.asarray(gs[kp])
        b = np.conj(xis[k]) * np.conj(xis[kp])
        acc += translation_average_fft(a, b)
        npair += 1
    return acc / npair
