"""Pins of the oracle's counter-based random numbers (oracle/hqmc_oracle.c: Philox4x32-10 + Box-Muller; PAPER.md:185 step (i),
:199 step (iii); readings C6, C25) against what is fixed OUTSIDE the oracle: the generator's published known-answer vectors,
the moments and distribution functions of U[0,1) and N(0, 1/2), E|R|^2 = 1 and Var p = 1/2.  CPU only."""
import os

import numpy as np
from scipy import stats

from oracle import oracle as orc

HERE = os.path.dirname(os.path.abspath(__file__))


def test_philox_known_answer_vectors():
    rows = [l for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for l in rows:
        ctr, key, out = [[int(w, 16) for w in part.split()] for part in l.split("|")]
        assert orc.philox4x32_10(ctr, key) == out, l


def test_counter_layout_and_streams_are_independent():
    """Element i, stream s, update k of seed S is the block at counter (i lo, i hi, s, k) under key (S lo, S hi)."""
    seed, upd = 0x1234567890ABCDEF, 7
    raw = orc.rng_raw(seed, upd, 1, 5)
    for i in range(5):
        assert list(raw[i]) == orc.philox4x32_10([i, 0, 1, upd], [seed & 0xFFFFFFFF, seed >> 32])
    a, b, c = orc.rng_raw(seed, upd, 0, 64), orc.rng_raw(seed, upd, 1, 64), orc.rng_raw(seed, upd + 1, 0, 64)
    assert not np.array_equal(a, b) and not np.array_equal(a, c)
    # 53-bit uniforms from the words: ((x0 >> 5) 2^26 + (x1 >> 6)) / 2^53
    u = orc.rng_uniform(seed, upd, 1, 5)
    want = ((raw[:, 0].astype(np.uint64) >> 5) * 67108864 + (raw[:, 1].astype(np.uint64) >> 6)) / 9007199254740992.0
    assert np.array_equal(u[:, 0], want) and (u >= 0).all() and (u < 1).all()


def test_uniforms_and_gaussians_have_the_stated_distributions():
    n = 400000
    u = orc.rng_uniform(11, 3, 2, n).ravel()
    assert abs(u.mean() - 0.5) < 4 / np.sqrt(12 * u.size) and abs(u.var() - 1 / 12) < 1e-3
    assert stats.kstest(u, "uniform").pvalue > 1e-3
    g = orc.rng_gauss(11, 3, 0, n)                       # stream 0: R = g[:, 0] + i g[:, 1]
    z = g.ravel()
    assert abs(z.mean()) < 4 * np.sqrt(0.5 / z.size) and abs(z.var() - 0.5) < 4 * 0.5 * np.sqrt(2 / z.size)   # reading C6
    assert stats.kstest(z * np.sqrt(2.0), "norm").pvalue > 1e-3
    assert abs((g[:, 0] ** 2 + g[:, 1] ** 2).mean() - 1.0) < 4 / np.sqrt(n)                                  # E|R|^2 = 1
    assert abs(np.corrcoef(g[:, 0], g[:, 1])[0, 1]) < 4 / np.sqrt(n)                                          # Re, Im independent
    p = orc.rng_gauss(11, 3, 1, n).ravel()
    assert abs(p.var() - 0.5) < 4 * 0.5 * np.sqrt(2 / p.size)                                                 # Var p = 1/2
    assert abs(stats.kurtosis(p)) < 0.05                                                                      # Gaussian tails


def test_sweep_is_the_loop_of_hqmc_steps_with_these_draws():
    """orc_hqmc_sweep = steps (i)-(iv) repeated with (R, p, u) taken from streams 0, 1, 2 of update k."""
    from paper_2508_16298_b200 import inputs
    L, Nt, seed = 4, 8, 21
    theta = inputs.theta_uniform(L, Nt, 0)
    o = orc.Oracle(L, Nt)
    sw = o.hqmc_sweep(theta, seed, 5, 3, 4, 0.1, cg_tol=1e-12)
    th = theta.copy()
    for k in range(3):
        eta = orc.rng_gauss(seed, 5 + k, 0, Nt * L * L)
        eta = (eta[:, 0] + 1j * eta[:, 1]).reshape(Nt, L, L)
        p = orc.rng_gauss(seed, 5 + k, 1, Nt * L * L).reshape(Nt, 2, L, L)
        u = orc.rng_uniform(seed, 5 + k, 2, 1)[0, 0]
        r = o.hqmc_step(th, p, eta, u, 4, 0.1, cg_tol=1e-12)
        assert r["accepted"] == sw["accepted"][k] and r["H0"] == sw["H0"][k] and r["H1"] == sw["H1"][k]
        th = r["theta"]
    assert np.array_equal(th, sw["theta"])
    assert sw["accepted"].any()                          # eps = 0.1 on this lattice accepts
