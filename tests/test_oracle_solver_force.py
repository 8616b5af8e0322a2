"""Pins of the oracle's CG, forces, actions and leapfrog against dense LU, central finite
differences, exact identities and symmetries.  CPU only."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2508_16298_b200 import inputs
from tests import dense_ref as dr

DTAU = 0.1


def _setup(L, Nt, seed, **kw):
    theta = inputs.theta_uniform(L, Nt, seed)
    o = orc.Oracle(L, Nt, **kw)
    eta = inputs.complex_gaussian((Nt, L, L), seed)
    phi = o.apply_Mdag(theta, eta)
    return o, theta, eta, phi


@pytest.mark.parametrize("W", [0, 6])
def test_pcg_vs_dense_lu_config1(W):
    """Config 1: CG to 1e-10 against a dense LU solve of M^+M built from generic expm."""
    o, theta, eta, phi = _setup(4, 8, 0, W=W)
    Md, _ = dr.dense_M(4, 8, theta, DTAU)
    Od = Md.conj().T @ Md
    x_ref = np.linalg.solve(Od, phi.ravel())
    x, it, rel = o.pcg(theta, phi, 1e-10, 10000)
    assert rel <= 1e-10 and 0 < it < 200
    true_res = np.linalg.norm(phi.ravel() - Od @ x.ravel()) / np.linalg.norm(phi)
    assert true_res < 1.05e-10
    assert np.abs(x.ravel() - x_ref).max() <= 1e-9 * np.abs(x_ref).max()
    # R = [M^+]^{-1} phi is the Gaussian: S_F(theta_0) = phi^+ x = eta^+ eta
    x13, _, _ = o.pcg(theta, phi, 1e-13, 10000)
    assert abs(np.vdot(phi, x13).real - np.vdot(eta, eta).real) < 1e-10
    assert abs(np.vdot(phi, x13).imag) < 1e-10


def test_pcg_preconditioner_cuts_iterations():
    """Regression, not parity (C10): survey probes saw 73 -> 42 on config 1 and ~3.5x on 8^2 x 80."""
    o0, theta, _, phi = _setup(4, 8, 0, W=0)
    o6 = orc.Oracle(4, 8, W=6)
    it0 = o0.pcg(theta, phi, 1e-10)[1]
    it6 = o6.pcg(theta, phi, 1e-10)[1]
    assert it6 < it0
    o0, theta, _, phi = _setup(8, 80, 7, W=0)
    o6 = orc.Oracle(8, 80, W=6)
    it0 = o0.pcg(theta, phi, 1e-10, 20000)[1]
    it6 = o6.pcg(theta, phi, 1e-10, 20000)[1]
    assert it6 * 2.5 < it0


def test_pcg_fixed_iteration_mode():
    """tol <= 0 runs exactly max_iter iterations."""
    o, theta, _, phi = _setup(4, 8, 0)
    x, it, rel = o.pcg(theta, phi, 0.0, 17)
    assert it == 17
    Md, _ = dr.dense_M(4, 8, theta, DTAU)
    true = np.linalg.norm(phi.ravel() - Md.conj().T @ (Md @ x.ravel())) / np.linalg.norm(phi)
    assert abs(true - rel) < 1e-8   # epsilon of PAPER.md:280 equals the recurrence residual


def _SF_dense(L, Nt, theta, phi):
    Md, _ = dr.dense_M(L, Nt, theta, DTAU)
    y = np.linalg.solve(Md.conj().T, phi.ravel())      # S_F = |M^{-+} phi|^2
    return np.vdot(y, y).real


def test_force_fermion_vs_finite_differences():
    """Every component on config 1 (256 bonds): central differences of S_F(theta) from dense LU (C11)."""
    L, Nt = 4, 8
    o, theta, _, phi = _setup(L, Nt, 0)
    x, _, _ = o.pcg(theta, phi, 1e-14, 10000)
    g = o.force_fermion(theta, x).ravel()
    h = 1e-5
    fd = np.zeros_like(g)
    for b in range(g.size):
        tp = theta.copy().ravel(); tp[b] += h
        tm = theta.copy().ravel(); tm[b] -= h
        fd[b] = (_SF_dense(L, Nt, tp.reshape(theta.shape), phi) - _SF_dense(L, Nt, tm.reshape(theta.shape), phi)) / (2 * h)
    assert np.abs(g).max() > 1e-2
    assert np.abs(g - fd).max() < 5e-9 * max(1.0, np.abs(g).max())


@pytest.mark.parametrize("compact", [True, False])
def test_force_boson_vs_finite_differences(compact):
    L, Nt = 4, 6
    theta = inputs.theta_uniform(L, Nt, 5)
    o = orc.Oracle(L, Nt, c_tau=1.3, K=0.7, compact=compact)
    assert abs(o.action_boson(theta) - dr.dense_SB(theta, 1.3, 0.7, compact)) < 1e-11
    g = o.force_boson(theta).ravel()
    h = 1e-4   # truncation ~ h^2/6 ~ 2e-9, round-off ~ 1e-16 * S_B / h ~ 1e-9
    for b in range(g.size):
        tp = theta.copy().ravel(); tp[b] += h
        tm = theta.copy().ravel(); tm[b] -= h
        fd = (dr.dense_SB(tp.reshape(theta.shape), 1.3, 0.7, compact) - dr.dense_SB(tm.reshape(theta.shape), 1.3, 0.7, compact)) / (2 * h)
        assert abs(g[b] - fd) < 2e-8


def test_gauge_invariance_of_solution_action_and_iteration_count():
    """theta -> theta + alpha_i - alpha_j, phi -> G phi leaves |x_i|, S_F, S_B and the CG iteration
    count invariant (BASELINE.json north_star; reading C3, C10: P is site-diagonal)."""
    L, Nt = 6, 12
    o, theta, _, phi = _setup(L, Nt, 9)
    alpha = inputs.gauge_alpha(L, 9)
    thp = inputs.gauge_transform_theta(theta, alpha)
    G = np.exp(1j * alpha)[None]
    x, it, _ = o.pcg(theta, phi, 1e-10)
    xg, itg, _ = o.pcg(thp, G * phi, 1e-10)
    assert it == itg
    assert np.abs(np.abs(x) - np.abs(xg)).max() < 1e-9 * np.abs(x).max()
    assert abs(np.vdot(phi, x).real - np.vdot(G * phi, xg).real) < 1e-9
    assert abs(o.action_boson(theta) - o.action_boson(thp)) < 1e-9
    # the force is gauge invariant too
    assert np.abs(o.force_fermion(theta, x) - o.force_fermion(thp, xg)).max() < 1e-8


def test_trajectory_H_decomposition_reversibility_and_eps2():
    L, Nt = 4, 8
    o, theta, eta, phi = _setup(L, Nt, 0)
    p = inputs.momenta(L, Nt, 0)
    r = o.trajectory(theta, p, phi, nsteps=8, eps=0.05, cg_tol=1e-13)
    # H0 = S_B + sum p^2 + eta^+ eta (Eq.12 + PAPER.md:183)
    assert abs(r["H0"] - (dr.dense_SB(theta, 1.0, 1.0) + (p * p).sum() + np.vdot(eta, eta).real)) < 1e-9
    assert abs(r["parts"][2] - np.vdot(eta, eta).real) < 1e-9
    # reversibility: flip p, integrate back
    back = o.trajectory(r["theta"], -r["p"], phi, nsteps=8, eps=0.05, cg_tol=1e-13)
    assert np.abs(back["theta"] - theta).max() < 1e-10
    assert np.abs(back["p"] + p).max() < 1e-10
    # dH ~ eps^2 at fixed trajectory length
    dH = [o.trajectory(theta, p, phi, nsteps=n, eps=0.4 / n, cg_tol=1e-13) for n in (8, 16, 32)]
    d = [q["H1"] - q["H0"] for q in dH]
    assert abs(d[0]) > 1e-4
    assert 3.5 < d[0] / d[1] < 4.5 and 3.8 < d[1] / d[2] < 4.2


def test_thread_count_does_not_change_results():
    o, theta, _, phi = _setup(6, 10, 4)
    orc.set_threads(1)
    x1, it1, _ = o.pcg(theta, phi, 1e-10)
    g1 = o.force_fermion(theta, x1)
    orc.set_threads(min(4, orc.max_threads()))
    x4, it4, _ = o.pcg(theta, phi, 1e-10)
    g4 = o.force_fermion(theta, x4)
    orc.set_threads(1)
    assert it1 == it4 and np.array_equal(x1, x4) and np.array_equal(g1, g4)


def test_heatbath_generator_plaquette():
    """<cos a_plaq> ~ 0.47-0.48 at 1/g^2 = 1 after 10 sweeps from a hot start;
    strong-coupling lower bound I1(1)/I0(1) = 0.446."""
    a = inputs.heatbath_theta(12, 120, 1, add_pi_flux=False)
    ps, pt = inputs.mean_plaquettes(a)
    assert 0.446 < ps < 0.50 and 0.446 < pt < 0.50
    th = inputs.heatbath_theta(12, 120, 1)
    assert abs(inputs.mean_plaquettes(th)[0] + ps) < 1e-12   # + A_pi flips the sign of cos(curl)


def test_hqmc_step_metropolis_rule():
    """orc_hqmc_step: H0 = S_B + sum p^2 + eta^+ eta exactly (phi = M^+ eta), the decision is
    u < min(1, e^{H0-H1}) (Eq.15), theta is restored on rejection and equals the trajectory's end point on acceptance."""
    L, Nt = 4, 8
    theta = inputs.theta_uniform(L, Nt, 0)
    p = inputs.momenta(L, Nt, 0)
    eta = inputs.complex_gaussian((Nt, L, L), 0)
    o = orc.Oracle(L, Nt, c_tau=0.0, K=0.0)     # (with c_tau = K = 1 this far-from-equilibrium field always has dH < 0)
    phi = o.apply_Mdag(theta, eta)
    t = o.trajectory(theta, p, phi, 6, 0.15)
    r_acc = min(1.0, np.exp(t["H0"] - t["H1"]))
    assert abs(t["H0"] - (o.action_boson(theta) + o.sum_p2(p) + np.vdot(eta, eta).real)) < 1e-9
    assert 0.0 < r_acc < 1.0            # dH = +0.067 here, so both branches are reachable
    for u, want in ((r_acc - 1e-9, True), (r_acc + 1e-9, False), (0.0, True)):
        s = o.hqmc_step(theta, p, eta, u, 6, 0.15)
        assert s["accepted"] is want and s["H0"] == t["H0"] and s["H1"] == t["H1"]
        assert np.array_equal(s["theta"], t["theta"] if want else theta)
        assert np.array_equal(s["p"], t["p"])
