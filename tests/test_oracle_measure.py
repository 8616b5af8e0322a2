"""Pins of the measurement oracle (oracle/measure_oracle.py; Eq.17-19) against facts it does not
contain: the O(N^2) definition, closed forms, and the dense inverse of the dense M of tests/dense_ref.py.  CPU only."""
import itertools

import numpy as np
import pytest

from oracle import measure_oracle as mo
from oracle import oracle as orc
from paper_2508_16298_b200 import inputs
from tests import dense_ref as dr


@pytest.mark.parametrize("shape,seed", [((3, 4, 4), 0), ((4, 2, 6), 1), ((5, 4, 2), 2)])
def test_eq19_fft_equals_eq17_double_loop(shape, seed):
    """Eq.19 (FFT) against Eq.17 + Eq.18 written as explicit loops: different formulas, same numbers."""
    a = inputs.complex_gaussian(shape, seed)
    b = inputs.complex_gaussian(shape, seed + 100)
    Cd = mo.translation_average_direct(a, b)
    Cf = mo.translation_average_fft(a, b)
    assert np.abs(Cd - Cf).max() <= 1e-13 * max(1.0, np.abs(Cd).max())
    # a transposed operand or F[a]_k instead of F[a]_{-k} gives the reflected correlation: must differ
    assert np.abs(mo.translation_average_fft(b, a) - Cd).max() > 1e-3


def test_translation_average_of_delta_functions():
    """a = delta_{i,i0}, b = delta_{j,j0}: C(Delta) = (1/N) delta_{Delta, j0 - i0} (closed form)."""
    shape = (4, 6, 4)
    i0, j0 = (1, 2, 3), (3, 1, 0)
    a = np.zeros(shape, np.complex128); a[i0] = 2.0 - 1.0j
    b = np.zeros(shape, np.complex128); b[j0] = 0.5j
    C = mo.translation_average_fft(a, b)
    want = np.zeros(shape, np.complex128)
    d = tuple((j - i) % n for i, j, n in zip(i0, j0, shape))
    want[d] = (2.0 - 1.0j) * 0.5j / a.size
    assert np.abs(C - want).max() <= 1e-15


def test_constant_vectors():
    """a = alpha, b = beta constant: every Delta gives alpha * beta."""
    shape = (3, 4, 4)
    C = mo.translation_average_fft(np.full(shape, 1.5 + 0.5j), np.full(shape, -2.0j))
    assert np.abs(C - (1.5 + 0.5j) * (-2.0j)).max() <= 1e-14


def test_full_basis_estimator_reproduces_dense_inverse():
    """averaging [G xi]_i xi_j^* over the N vectors xi = sqrt(N) e_l (which satisfy E xi_i^* xi_j =
    delta_ij exactly) gives M^{-1} itself, so the translation-averaged estimate must equal (1/N) sum_i [M^{-1}]_{i,i+Delta}
    of the dense inverse of the dense M assembled from generic matrix exponentials."""
    L, Nt, seed = 4, 4, 3
    theta = inputs.theta_uniform(L, Nt, seed)
    o = orc.Oracle(L, Nt)
    N = L * L * Nt
    Md, _ = dr.dense_M(L, Nt, theta)
    Minv = np.linalg.inv(Md)
    want = np.zeros((Nt, L, L), np.complex128)
    idx = np.arange(N).reshape(Nt, L, L)
    for dt, dy, dx in itertools.product(range(Nt), range(L), range(L)):
        j = np.roll(idx, (-dt, -dy, -dx), axis=(0, 1, 2))            # j = i + Delta
        want[dt, dy, dx] = Minv[idx.ravel(), j.ravel()].sum() / N
    gs, xis = [], []
    for l in range(N):
        xi = np.zeros(N, np.complex128); xi[l] = np.sqrt(N)
        xi = xi.reshape(Nt, L, L)
        g, it = mo.green_apply(o, theta, xi, 1e-13, 10000)
        assert np.abs(g.ravel() - Minv[:, l] * np.sqrt(N)).max() <= 1e-9 * np.sqrt(N)      # G xi = M^{-1} xi
        gs.append(g); xis.append(xi)
    got = mo.green_2pt(gs, xis)
    assert np.abs(got - want).max() <= 1e-10


def test_pair_correlator_against_explicit_pairs():
    """Eq.18 with a_i = (G xi)_i (G xi')_i, b_j = xi_j^* xi'_j^*, Eq.17 by loops, mean over the binom(n,2) pairs."""
    shape, n = (2, 4, 2), 4
    gs = [inputs.complex_gaussian(shape, 10 + k) for k in range(n)]
    xis = [inputs.complex_gaussian(shape, 20 + k) for k in range(n)]
    want = np.zeros(shape, np.complex128)
    pairs = [(k, kp) for k in range(n) for kp in range(k + 1, n)]
    assert len(pairs) == 6
    for k, kp in pairs:
        want += mo.translation_average_direct(gs[k] * gs[kp], np.conj(xis[k]) * np.conj(xis[kp]))
    want /= len(pairs)
    assert np.abs(mo.pair_correlator(gs, xis) - want).max() <= 1e-13


def test_free_fermion_green_function_is_translation_invariant():
    """theta = 0, L = 4: on a 4-site ring the even- and odd-bond hopping matrices commute, so the split B is invariant
    under ONE-site translations and the full-basis average of Eq.17 equals row 0 of M^{-1} (index/sign pin)."""
    L, Nt = 4, 3
    theta = np.zeros((Nt, 2, L, L))
    Md, _ = dr.dense_M(L, Nt, theta)
    Minv = np.linalg.inv(Md)
    N = L * L * Nt
    a_sum = np.zeros((Nt, L, L), np.complex128)
    for l in range(N):
        xi = np.zeros(N, np.complex128); xi[l] = np.sqrt(N)
        a_sum += mo.translation_average_fft((Minv @ xi).reshape(Nt, L, L), np.conj(xi).reshape(Nt, L, L))
    got = a_sum / N
    # C(Delta) = M^{-1}[0, Delta] for spatial shifts; the temporal wrap of a fermion line carries a minus sign, so only
    # the dt = 0 plane is translation-averaged without sign bookkeeping (reading C23)
    assert np.abs(got[0] - Minv[0, :L * L].reshape(L, L)).max() <= 1e-12
