"""GPU parity of the stochastic estimator (Eq.17-19; widening row NEXT-2): libhqmc.so through the C ABI
against oracle/measure_oracle.py on the same seeded inputs.  Tolerances: 1e-12 relative for the FFT path (fp64 transforms
of <= 1.1 M points), 1e-9 for G xi (north_star's CG bound)."""
import numpy as np
import pytest
import torch

from oracle import measure_oracle as mo
from oracle import oracle as orc
from paper_2508_16298_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hq(cuda_device):
    from paper_2508_16298_b200 import hqmc
    return hqmc


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


# power-of-two, mixed-radix (3, 5, 7) and prime extents; the last one is a Bluestein size for cuFFT
@pytest.mark.parametrize("L,Nt,seed", [(4, 8, 0), (6, 10, 1), (12, 7, 2), (20, 9, 3), (14, 11, 4), (48, 6, 5)])
def test_translation_average_matches_oracle(hq, L, Nt, seed):
    a = inputs.complex_gaussian((Nt, L, L), seed, inputs.STREAM_VEC)
    b = inputs.complex_gaussian((Nt, L, L), seed + 50, inputs.STREAM_VEC)
    g = hq.HQMC(L, Nt, W=0)
    C = g.translation_average(dev(a), dev(b)).cpu().numpy()
    want = mo.translation_average_fft(a, b)
    assert rel(C, want) <= 1e-12
    if L * L * Nt <= 200:                                  # and against the O(N^2) definition itself
        assert rel(C, mo.translation_average_direct(a, b)) <= 1e-12
    # in-place forms (d_C aliasing an input) and repeatability
    da, db = dev(a), dev(b)
    g.translation_average(da, db, out=da)
    assert torch.equal(da.cpu(), torch.from_numpy(C))
    g.close()


def test_translation_average_of_a_delta_is_exact(hq):
    L, Nt = 8, 6
    a = np.zeros((Nt, L, L), np.complex128); a[1, 2, 3] = 1.0
    b = np.zeros((Nt, L, L), np.complex128); b[4, 0, 7] = 1.0
    g = hq.HQMC(L, Nt, W=0)
    C = g.translation_average(dev(a), dev(b)).cpu().numpy() * (L * L * Nt)
    want = np.zeros_like(a); want[3, 6, 4] = 1.0
    assert np.abs(C - want).max() <= 1e-14
    g.close()


@pytest.mark.parametrize("L,Nt,seed,n_rv", [(4, 8, 0, 5), (8, 12, 1, 4), (12, 10, 2, 3)])
def test_green_apply_2pt_and_pair_correlator(hq, L, Nt, seed, n_rv):
    theta = inputs.theta_uniform(L, Nt, seed)
    o = orc.Oracle(L, Nt)
    orc.set_threads(orc.max_threads())
    g = hq.HQMC(L, Nt)
    g.set_theta(dev(theta))
    xis = [inputs.complex_gaussian((Nt, L, L), seed + 10 * k, inputs.STREAM_VEC) for k in range(n_rv)]
    gs, its = zip(*[mo.green_apply(o, theta, xi, 1e-12, 200000) for xi in xis])
    d_xi = dev(np.stack(xis))
    d_g, it, ok = g.green_apply(d_xi, 1e-12, 200000)
    assert ok and abs(it - sum(its)) <= n_rv                 # same iteration counts up to a last-step rounding flip
    G = d_g.cpu().numpy()
    for k in range(n_rv):
        assert rel(G[k], gs[k]) <= 1e-9
        # G xi = M^{-1} xi: M (G xi) returns xi
        back = g.apply_M(d_g[k].contiguous()).cpu().numpy()
        assert rel(back, xis[k]) <= 1e-9
    # estimators on the ORACLE's g (isolates the FFT path from CG rounding), then end to end on the GPU's own g
    d_go = dev(np.stack(gs))
    assert rel(g.green_2pt(d_go, d_xi).cpu().numpy(), mo.green_2pt(gs, xis)) <= 1e-12
    assert rel(g.pair_correlator(d_go, d_xi).cpu().numpy(), mo.pair_correlator(gs, xis)) <= 1e-12
    assert rel(g.green_2pt(d_g, d_xi).cpu().numpy(), mo.green_2pt(gs, xis)) <= 1e-8
    assert rel(g.pair_correlator(d_g, d_xi).cpu().numpy(), mo.pair_correlator(gs, xis)) <= 1e-8
    g.close()


def test_full_basis_reproduces_the_oracle_full_basis_average(hq):
    """N vectors sqrt(N) e_l: the estimator is exact; compare with the oracle's pinned full-basis result."""
    L, Nt, seed = 4, 4, 3
    N = L * L * Nt
    theta = inputs.theta_uniform(L, Nt, seed)
    o = orc.Oracle(L, Nt, W=3)
    g = hq.HQMC(L, Nt, W=3)
    g.set_theta(dev(theta))
    xi = (np.sqrt(N) * np.eye(N, dtype=np.complex128)).reshape(N, Nt, L, L)
    d_xi = dev(xi)
    d_g, it, ok = g.green_apply(d_xi, 1e-13, 10000)
    assert ok
    gs = [mo.green_apply(o, theta, xi[l], 1e-13, 10000)[0] for l in range(N)]
    want = mo.green_2pt(gs, list(xi))
    assert rel(g.green_2pt(d_g, d_xi).cpu().numpy(), want) <= 1e-9
    g.close()


def test_full_size_config4_sampled(hq):
    """BASELINE config 4 size (L=48, N_tau=480) on a paper-regime field: Eq.19 on sampled Delta against Eq.17 evaluated one
    Delta at a time; G xi through the property M (G xi) = xi; estimator linearity in the number of vectors."""
    L, Nt, seed = 48, 480, 4
    N = L * L * Nt
    a = inputs.complex_gaussian((Nt, L, L), seed, inputs.STREAM_VEC)
    b = inputs.complex_gaussian((Nt, L, L), seed + 1, inputs.STREAM_VEC)
    g = hq.HQMC(L, Nt)
    C = g.translation_average(dev(a), dev(b)).cpu().numpy()
    rng = np.random.default_rng(7)
    scale = np.abs(C).max()
    for d in [(0, 0, 0), (1, 0, 0), (Nt - 1, L - 1, L - 1), (0, 1, 47)] + [tuple(int(rng.integers(0, n)) for n in (Nt, L, L)) for _ in range(6)]:
        want = np.vdot(np.conj(a).ravel(), np.roll(b, tuple(-x for x in d), axis=(0, 1, 2)).ravel()) / N      # sum_i a_i b_{i+d} / N
        assert abs(C[d] - want) <= 1e-12 * scale, d
    theta = inputs.theta_paper_regime(L, Nt, seed)
    g.set_theta(dev(theta))
    xi = np.stack([inputs.complex_gaussian((Nt, L, L), seed + 10 * k, inputs.STREAM_VEC) for k in range(3)])
    d_xi = dev(xi)
    d_g, it, ok = g.green_apply(d_xi, 1e-10, 20000)
    assert ok and it < 3 * 2000
    for k in range(3):
        back = g.apply_M(d_g[k].contiguous())
        assert float(torch.linalg.vector_norm(back - d_xi[k]) / torch.linalg.vector_norm(d_xi[k])) <= 1e-8
    # mean over 3 pairs = mean of the three single-pair results
    full = g.pair_correlator(d_g, d_xi).clone()
    acc = torch.zeros_like(full)
    for k, kp in ((0, 1), (0, 2), (1, 2)):
        acc += g.pair_correlator(torch.stack([d_g[k], d_g[kp]]), torch.stack([d_xi[k], d_xi[kp]]))
    assert float((full - acc / 3).abs().max() / full.abs().max()) <= 1e-12
    g.close()


def test_measure_c64_variant(hq):
    L, Nt, seed = 8, 12, 6
    a = inputs.complex_gaussian((Nt, L, L), seed, inputs.STREAM_VEC)
    b = inputs.complex_gaussian((Nt, L, L), seed + 1, inputs.STREAM_VEC)
    g = hq.HQMC(L, Nt, prec="c64", W=0)
    C = g.translation_average(dev(a.astype(np.complex64)), dev(b.astype(np.complex64))).cpu().numpy()
    assert rel(C, mo.translation_average_fft(a, b)) <= 2e-5
    g.close()


def test_measure_argument_checks(hq):
    g = hq.HQMC(4, 8)
    v = g.new_vec()
    with pytest.raises(hq.HqmcError):                       # theta not set
        g.green_apply(torch.zeros((2, 8, 4, 4), dtype=torch.complex128, device="cuda"))
    with pytest.raises(AssertionError):                     # one vector is not a pair
        g.pair_correlator(v, v)
    g.close()
