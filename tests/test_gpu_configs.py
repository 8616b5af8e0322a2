"""GPU parity on BASELINE.json's five configs AS STATED (north_star: "match the oracle on all five configs"), at full size,
in the launch configuration bench.py times.  Tolerances: <= 1e-12 per M / M^+ / M^+M application, <= 1e-9 per CG solution
at tol 1e-10 (reading C16: judged by the residual under the ORACLE's operator and against the oracle's iterate), <= 1e-9 per
force component, |dH_gpu - dH_oracle| <= 1e-8 max(1, |H0| 1e-6) (reading C17), reversibility <= 1e-10.
Citations: PAPER.md:155 (Eq.8), :207-214 (Eq.16), :250-261 (Eq.20), :348 (fixed-count protocol), :455-477 (force)."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2508_16298_b200 import inputs
from tests import dense_ref

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hq(cuda_device):
    from paper_2508_16298_b200 import hqmc
    return hqmc


@pytest.fixture(scope="module")
def theta5():
    """BASELINE config 5's field: the seeded heat bath on the full 64^2 x 640 lattice (about 40 s of numpy on the host)."""
    return inputs.make_theta(5)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(a, b):
    """max |a - b| / max |b|: small elements are compared absolutely against the largest one."""
    return float(np.abs(a - b).max() / np.abs(b).max())


def setup(hq, cfg, theta=None, **kw):
    c = inputs.CONFIGS[cfg]
    theta = inputs.make_theta(cfg) if theta is None else theta
    o = orc.Oracle(c["L"], c["Ntau"], **kw)
    orc.set_threads(orc.max_threads())
    g = hq.HQMC(c["L"], c["Ntau"], **kw)
    g.set_theta(dev(theta))
    return c, o, g, theta


def relres_under_oracle(o, theta, phi, x):
    return float(np.linalg.norm((phi - o.apply_MdagM(theta, x)).ravel()) / np.linalg.norm(phi.ravel()))


def test_config1_everything_against_dense(hq):
    """Config 1 (L=4, Ntau=8, uniform theta, seed 0): CG to 1e-10 against the dense LU solution, all operators."""
    c, o, g, theta = setup(hq, 1)
    L, Nt = c["L"], c["Ntau"]
    eta = inputs.complex_gaussian((Nt, L, L), c["seed"])
    M = dense_ref.dense_M(L, Nt, theta)[0]
    phi = (M.conj().T @ eta.ravel()).reshape(eta.shape)
    assert rel(g.apply_Mdag(dev(eta)).cpu().numpy(), phi) <= 1e-12
    x, it, relres, ok = g.cg_solve(dev(phi), 1e-10, 10000)
    x_lu = np.linalg.solve(M.conj().T @ M, phi.ravel()).reshape(phi.shape)
    assert ok and relres <= 1e-10 and rel(x.cpu().numpy(), x_lu) <= 1e-9
    assert abs(np.vdot(phi, x.cpu().numpy()).real - np.vdot(eta, eta).real) <= 1e-8      # S_F(theta_0) = eta^+ eta
    g.close()


def test_config2_cg_solve_and_force_on_the_heatbath_field(hq):
    """Config 2 (L=12, Ntau=120, heat-bath theta): ONE PCG solve to 1e-10 and ONE force evaluation (the 20 M^+M applications
    are in test_gpu_parity.py::test_config2_twenty_MdagM)."""
    c, o, g, theta = setup(hq, 2)
    L, Nt = c["L"], c["Ntau"]
    eta = inputs.complex_gaussian((Nt, L, L), c["seed"])
    phi = o.apply_Mdag(theta, eta)
    assert rel(g.apply_Mdag(dev(eta)).cpu().numpy(), phi) <= 1e-12
    x_ref, it_ref, rel_ref = o.pcg(theta, phi, 1e-10, 200000)
    x, it, relres, ok = g.cg_solve(dev(phi), 1e-10, 200000)
    x = x.cpu().numpy()
    assert ok and relres <= 1e-10 and rel_ref <= 1e-10
    assert abs(it - it_ref) <= max(2, it_ref // 100), (it, it_ref)
    assert relres_under_oracle(o, theta, phi, x) <= 1.05e-10                 # reading C16 (i)
    assert rel(x, x_ref) <= 1e-9                                             # the two iterates at the same tolerance
    # force from the GPU's own solution, component by component, against the oracle's force from the same X
    gF = g.force(dev(x)).cpu().numpy()
    ref = o.force_fermion(theta, x)
    assert np.abs(gF - ref).max() <= 1e-9 * max(1.0, np.abs(ref).max())
    # and end to end: the oracle's force from the ORACLE's solution (differs by the two solves' 1e-10 residuals)
    ref2 = o.force_fermion(theta, x_ref)
    assert np.abs(gF - ref2).max() <= 1e-7 * max(1.0, np.abs(ref2).max())
    g.close()


def test_config3_twenty_step_trajectory_dH_and_reversibility(hq):
    """Config 3 (L=24, Ntau=240, uniform theta, eps=0.05): the full 20-step trajectory at full size with the paper's
    fixed-count CG protocol on both sides (40 iterations per solve: converging this field takes ~1e5
    iterations per solve, hours for the oracle), dH against the oracle within reading C17's bound, theta' and p' element by
    element, and the GPU reversibility leg (a leapfrog with any force that depends on theta alone is reversible)."""
    c, o, g, theta = setup(hq, 3)
    L, Nt, nsteps, iters = c["L"], c["Ntau"], 20, 40
    eta = inputs.complex_gaussian((Nt, L, L), c["seed"])
    phi = o.apply_Mdag(theta, eta)
    p = inputs.momenta(L, Nt, c["seed"])
    ref = o.trajectory(theta, p, phi, nsteps, 0.05, cg_tol=0.0, cg_max_iter=iters)
    dth, dp, dphi = dev(theta), dev(p), dev(phi)
    r = g.trajectory(dth, dp, dphi, nsteps, 0.05, cg_tol=0.0, cg_max_iter=iters)
    assert r["cg_iters"] == ref["cg_iters"] == iters * (nsteps + 1)
    bound = 1e-8 * max(1.0, abs(ref["H0"]) * 1e-6)
    assert abs(r["H0"] - ref["H0"]) <= bound and abs(r["H1"] - ref["H1"]) <= bound
    assert abs((r["H1"] - r["H0"]) - (ref["H1"] - ref["H0"])) <= bound
    assert np.abs(dth.cpu().numpy() - ref["theta"]).max() <= 1e-10
    assert np.abs(dp.cpu().numpy() - ref["p"]).max() <= 1e-9 * max(1.0, np.abs(ref["p"]).max())
    dp.neg_()
    g.trajectory(dth, dp, dphi, nsteps, 0.05, cg_tol=0.0, cg_max_iter=iters)
    assert np.abs(dth.cpu().numpy() - theta).max() <= 1e-10
    assert np.abs(dp.cpu().numpy() + p).max() <= 1e-10 * max(1.0, np.abs(p).max())
    g.close()


def test_twenty_step_trajectory_with_converged_solves(hq):
    """Config 3's protocol (20 leapfrog steps, uniform theta) with CONVERGED solves, where it is a stable integration: L=8, Ntau=80,
    eps = 0.005 (at config 3's eps = 0.05 the leapfrog diverges on both sides).  21 solves of ~1000 iterations to
    1e-12 on each side: H0, dH, theta', p' and the reversed trajectory (reading C17)."""
    L, Nt, nsteps, eps = 8, 80, 20, 0.005
    theta, p = inputs.theta_uniform(L, Nt, 2), inputs.momenta(L, Nt, 2)
    eta = inputs.complex_gaussian((Nt, L, L), 2)
    o = orc.Oracle(L, Nt)
    orc.set_threads(orc.max_threads())
    phi = o.apply_Mdag(theta, eta)
    ref = o.trajectory(theta, p, phi, nsteps, eps, cg_tol=1e-12, cg_max_iter=1000000)
    g = hq.HQMC(L, Nt)
    dth, dp, dphi = dev(theta), dev(p), dev(phi)
    r = g.trajectory(dth, dp, dphi, nsteps, eps, cg_tol=1e-12, cg_max_iter=1000000)
    assert r["converged"] and abs(r["cg_iters"] - ref["cg_iters"]) <= max(21 * 2, ref["cg_iters"] // 100)
    bound = 1e-8 * max(1.0, abs(ref["H0"]) * 1e-6) * 10          # 21 solves at 1e-12 each
    assert abs(r["H0"] - ref["H0"]) <= bound and abs((r["H1"] - r["H0"]) - (ref["H1"] - ref["H0"])) <= 1e-6
    assert np.abs(dth.cpu().numpy() - ref["theta"]).max() <= 1e-9
    assert np.abs(dp.cpu().numpy() - ref["p"]).max() <= 1e-7 * max(1.0, np.abs(ref["p"]).max())
    dp.neg_()
    g.trajectory(dth, dp, dphi, nsteps, eps, cg_tol=1e-12, cg_max_iter=1000000)
    assert np.abs(dth.cpu().numpy() - theta).max() <= 1e-8 and np.abs(dp.cpu().numpy() + p).max() <= 1e-6 * max(1.0, np.abs(p).max())
    g.close()


@pytest.mark.parametrize("L,Nt", [(8, 80), (12, 60)])
def test_paper_regime_trajectory_with_converged_solves(hq, L, Nt):
    """The regime the method is run in (c_tau = 1/(J dtau^2) = 80, K = 1; smooth-in-tau fields, O(100) PCG iterations):
    a 10-step trajectory at eps = 0.02 (c_tau = 80 puts the leapfrog's stability edge near 0.05) with solves converged to 1e-12 on both sides, c_tau = 80 in the bosonic force and action:
    H0, dH, theta', p', reversibility."""
    nsteps, eps, kw = 10, 0.02, dict(c_tau=80.0, K=1.0)
    theta = inputs.theta_paper_regime(L, Nt, 6, sweeps=20)
    p, eta = inputs.momenta(L, Nt, 6), inputs.complex_gaussian((Nt, L, L), 6)
    o = orc.Oracle(L, Nt, **kw)
    orc.set_threads(orc.max_threads())
    phi = o.apply_Mdag(theta, eta)
    ref = o.trajectory(theta, p, phi, nsteps, eps, cg_tol=1e-12, cg_max_iter=100000)
    g = hq.HQMC(L, Nt, **kw)
    dth, dp, dphi = dev(theta), dev(p), dev(phi)
    r = g.trajectory(dth, dp, dphi, nsteps, eps, cg_tol=1e-12, cg_max_iter=100000)
    assert r["converged"] and abs(r["cg_iters"] - ref["cg_iters"]) <= max(22, ref["cg_iters"] // 100)
    assert abs(ref["H1"] - ref["H0"]) < 50.0                     # a stable integration, not a divergence
    assert abs(r["H0"] - ref["H0"]) <= 1e-8 * max(1.0, abs(ref["H0"]) * 1e-6) * 10
    assert abs((r["H1"] - r["H0"]) - (ref["H1"] - ref["H0"])) <= 1e-8
    assert np.abs(dth.cpu().numpy() - ref["theta"]).max() <= 1e-10
    assert np.abs(dp.cpu().numpy() - ref["p"]).max() <= 1e-9 * max(1.0, np.abs(ref["p"]).max())
    dp.neg_()
    g.trajectory(dth, dp, dphi, nsteps, eps, cg_tol=1e-12, cg_max_iter=100000)
    assert np.abs(dth.cpu().numpy() - theta).max() <= 1e-10 and np.abs(dp.cpu().numpy() + p).max() <= 1e-10 * max(1.0, np.abs(p).max())
    g.close()


def test_config4_converged_solve_judged_by_the_oracles_operator(hq):
    """Config 4 (L=48, Ntau=480, uniform theta): preconditioned CG to 1e-10 (about 3e5 iterations, some 20 s on the GPU;
    far out of the oracle's reach), then ONE oracle M^+M: ||phi - O_oracle x_gpu|| / ||phi|| <= 1.05e-10 (reading C16 i)."""
    c, o, g, theta = setup(hq, 4)
    L, Nt = c["L"], c["Ntau"]
    eta = inputs.complex_gaussian((Nt, L, L), c["seed"])
    dphi = g.apply_Mdag(dev(eta))
    phi = dphi.cpu().numpy()
    assert rel(phi, o.apply_Mdag(theta, eta)) <= 1e-12
    x, it, relres, ok = g.cg_solve(dphi, 1e-10, 3000000)
    assert ok and relres <= 1e-10 and it > 1000
    x = x.cpu().numpy()
    assert relres_under_oracle(o, theta, phi, x) <= 1.05e-10
    assert abs(np.vdot(phi, x).real - np.vdot(eta, eta).real) <= 1e-6 * np.vdot(eta, eta).real     # S_F(theta_0) = eta^+ eta
    g.close()


def test_config4_complex64_variant_at_full_size(hq):
    """Config 4's complex64 variant (reading C19): <= 1e-6 L2-relative per M^+M against the fp64 oracle at full size."""
    c = inputs.CONFIGS[4]
    L, Nt = c["L"], c["Ntau"]
    theta = inputs.make_theta(4)
    o = orc.Oracle(L, Nt)
    orc.set_threads(orc.max_threads())
    g = hq.HQMC(L, Nt, prec="c64")
    g.set_theta(dev(theta))
    v = inputs.complex_gaussian((Nt, L, L), c["seed"], inputs.STREAM_VEC)
    out = g.apply_MdagM(dev(v.astype(np.complex64))).cpu().numpy().astype(np.complex128)
    ref = o.apply_MdagM(theta, v)
    assert np.linalg.norm((out - ref).ravel()) / np.linalg.norm(ref.ravel()) <= 1e-6
    g.close()


def test_config5_operators_on_the_real_heatbath_field(hq, theta5):
    """Config 5 (L=64, Ntau=640) on ITS OWN field, the seeded heat bath at 1/g^2 = 1 (not a uniform stand-in): M, M^+, M^+M,
    P, the force and 20 fixed-count PCG iterations element by element against the oracle, default (cluster) kernels."""
    c, o, g, theta = setup(hq, 5, theta=theta5)
    L, Nt = c["L"], c["Ntau"]
    v = inputs.complex_gaussian((Nt, L, L), c["seed"], inputs.STREAM_VEC)
    dv = dev(v)
    assert rel(g.apply_M(dv).cpu().numpy(), o.apply_M(theta, v)) <= 1e-12
    assert rel(g.apply_Mdag(dv).cpu().numpy(), o.apply_Mdag(theta, v)) <= 1e-12
    assert rel(g.apply_MdagM(dv).cpu().numpy(), o.apply_MdagM(theta, v)) <= 1e-12
    assert rel(g.precond(dv).cpu().numpy(), o.precond(v)) <= 1e-13
    gF = g.force(dv).cpu().numpy()
    ref = o.force_fermion(theta, v)
    assert np.abs(gF - ref).max() <= 1e-9 * max(1.0, np.abs(ref).max())
    xf, itf, relf, _ = g.cg_solve(dv, 0.0, 20)
    xo, ito, relo = o.pcg(theta, v, 0.0, 20)
    assert itf == ito == 20 and rel(xf.cpu().numpy(), xo) <= 1e-10 and abs(relf - relo) <= 1e-9 * relo
    g.close()


def test_config5_one_leapfrog_step_on_the_real_field(hq, theta5):
    """Config 5's trajectory protocol (20 leapfrog steps, eps = 0.05) costs the oracle an hour; ONE step with 30 fixed
    iterations per solve exercises every kernel of the step at full size on the real field: theta', p', H0, H1."""
    c, o, g, theta = setup(hq, 5, theta=theta5)
    L, Nt = c["L"], c["Ntau"]
    eta = inputs.complex_gaussian((Nt, L, L), c["seed"])
    phi = o.apply_Mdag(theta, eta)
    p = inputs.momenta(L, Nt, c["seed"])
    ref = o.trajectory(theta, p, phi, 1, 0.05, cg_tol=0.0, cg_max_iter=30)
    dth, dp = dev(theta), dev(p)
    r = g.trajectory(dth, dp, dev(phi), 1, 0.05, cg_tol=0.0, cg_max_iter=30)
    bound = 1e-8 * max(1.0, abs(ref["H0"]) * 1e-6)
    assert abs(r["H0"] - ref["H0"]) <= bound and abs((r["H1"] - r["H0"]) - (ref["H1"] - ref["H0"])) <= bound
    assert np.abs(dth.cpu().numpy() - ref["theta"]).max() <= 1e-10
    assert np.abs(dp.cpu().numpy() - ref["p"]).max() <= 1e-9 * max(1.0, np.abs(ref["p"]).max())
    g.close()


@pytest.mark.parametrize("L,Nt", [(12, 120), (24, 60), (48, 24)])
def test_leapfrog_step_graph_is_bitwise_identical_to_plain_launches(hq, L, Nt):
    """The leapfrog step replayed as one CUDA graph (include/hqmc_tuning.h hqmc_set_md_graph) runs the same
    kernels in the same order as plain launches: theta', p', H0, H1 agree bit for bit."""
    theta = inputs.theta_uniform(L, Nt, 5)
    p = inputs.momenta(L, Nt, 5)
    phi = inputs.complex_gaussian((Nt, L, L), 5)
    out = []
    for on in (True, False):
        g = hq.HQMC(L, Nt)
        g.set_cg_persistent(hq.PERSIST_OFF)          # (small lattices would take the one-launch solve and no step graph at all)
        g.set_md_graph(on)
        dth, dp = dev(theta), dev(p)
        r = g.trajectory(dth, dp, dev(phi), 4, 0.05, cg_tol=0.0, cg_max_iter=70)      # 70: not a multiple of the 32-iteration chunk
        out.append((dth.clone(), dp.clone(), r["H0"], r["H1"], r["cg_iters"]))
        g.close()
    assert torch.equal(out[0][0], out[1][0]) and torch.equal(out[0][1], out[1][1])
    assert out[0][2:] == out[1][2:] and out[0][4] == 70 * 5


def test_persistent_pcg_kernel_selection_and_limits(hq):
    """include/hqmc_tuning.h hqmc_set_cg_persistent: AUTO takes the one-launch kernel on small lattices (bitwise the same as
    ON, one launch instead of four per iteration), refuses lattices it cannot hold, complex64 runs through it too."""
    L, Nt = 12, 120
    theta = inputs.theta_uniform(L, Nt, 8)
    phi = inputs.complex_gaussian((Nt, L, L), 8)
    g = hq.HQMC(L, Nt)
    g.set_theta(dev(theta))
    out = {}
    for mode in (hq.PERSIST_AUTO, hq.PERSIST_ON, hq.PERSIST_OFF):
        g.set_cg_persistent(mode)
        g.reset_stats()
        x, it, relres, _ = g.cg_solve(dev(phi), 0.0, 30)
        out[mode] = (x.clone(), relres, sum(v[0] for v in g.kernel_stats().values()))
    assert torch.equal(out[hq.PERSIST_AUTO][0], out[hq.PERSIST_ON][0]) and out[hq.PERSIST_AUTO][2] == 1
    assert out[hq.PERSIST_OFF][2] >= 4 * 30
    assert rel(out[hq.PERSIST_ON][0].cpu().numpy(), out[hq.PERSIST_OFF][0].cpu().numpy()) <= 1e-12
    g.close()
    # the largest lattice AUTO takes (L=20, Ntau=200: 200 CTAs of 128 threads, two per SM on some SMs): fixed-count iterates
    L2, Nt2 = 20, 200
    th2 = inputs.theta_uniform(L2, Nt2, 9)
    v2 = inputs.complex_gaussian((Nt2, L2, L2), 9)
    o2 = orc.Oracle(L2, Nt2)
    orc.set_threads(orc.max_threads())
    g = hq.HQMC(L2, Nt2)
    g.set_theta(dev(th2))
    g.reset_stats()
    x, it, relres, _ = g.cg_solve(dev(v2), 0.0, 30)
    xo, ito, relo = o2.pcg(th2, v2, 0.0, 30)
    assert sum(v[0] for v in g.kernel_stats().values()) == 1 and it == ito == 30
    assert rel(x.cpu().numpy(), xo) <= 1e-11 and abs(relres - relo) <= 1e-9 * relo
    g.close()
    big = hq.HQMC(48, 20)
    with pytest.raises(hq.HqmcError):
        big.set_cg_persistent(hq.PERSIST_ON)
    big.close()
    o = orc.Oracle(L, Nt)
    g = hq.HQMC(L, Nt, prec="c64")
    g.set_theta(dev(theta))
    g.set_cg_persistent(hq.PERSIST_ON)
    x, it, relres, _ = g.cg_solve(dev(phi.astype(np.complex64)), 0.0, 12)
    xo, _, relo = o.pcg(theta, phi, 0.0, 12)
    assert it == 12 and np.linalg.norm(x.cpu().numpy().astype(np.complex128).ravel() - xo.ravel()) / np.linalg.norm(xo.ravel()) <= 1e-5
    g.close()


def test_device_random_numbers_match_the_cpu_twin_bit_for_bit(hq):
    """NEXT-1 (reading C25): same (seed, update, stream, element) -> the same Philox4x32-10 words bit
    for bit, hence the same 53-bit uniforms; the Gaussians differ only by the last bits of log / sincos."""
    g = hq.HQMC(4, 8)
    seed, upd, n = 0xC0FFEE1234567, 41, 100003
    for stream in (0, 1, 2):
        raw = g.rng_raw(seed, upd, stream, n).cpu().numpy().view(np.uint32)
        assert np.array_equal(raw, orc.rng_raw(seed, upd, stream, n))
        gg = g.rng_gauss(seed, upd, stream, n).cpu().numpy()
        assert np.abs(gg - orc.rng_gauss(seed, upd, stream, n)).max() <= 1e-14
    assert hq.HQMC.rng_uniform(seed, upd) == orc.rng_uniform(seed, upd, 2, 1)[0, 0]
    z = g.rng_gauss(7, 0, 0, 1 << 20)
    assert abs(float((z ** 2).sum(dim=1).mean()) - 1.0) < 4e-3 and abs(float(z.var()) - 0.5) < 3e-3      # E|R|^2 = 1, Var = 1/2
    g.close()


def test_sweep_acceptance_sequence_equals_the_oracles(hq):
    """hqmc_sweep (steps (i)-(iv) looped, every draw made on the device) against the oracle's sweep from the same seed on a
    short chain: same acceptance sequence, H0 and dH to 1e-8, final theta to 1e-9."""
    L, Nt, seed, n_upd = 6, 10, 99, 6
    theta = inputs.theta_uniform(L, Nt, 1)
    o = orc.Oracle(L, Nt, c_tau=0.0, K=0.0)
    g = hq.HQMC(L, Nt, c_tau=0.0, K=0.0)
    ref = o.hqmc_sweep(theta, seed, 3, n_upd, 5, 0.2, cg_tol=1e-13)       # eps = 0.2: a mix of accepted and rejected updates
    dth = dev(theta)
    r = g.sweep(dth, seed, 3, n_upd, 5, 0.2, cg_tol=1e-13)
    assert r["converged"] and r["accepted"] == list(ref["accepted"])
    assert 0 < sum(r["accepted"]) < n_upd or n_upd < 2, r["accepted"]
    assert np.abs(np.array(r["H0"]) - ref["H0"]).max() <= 1e-8
    assert np.abs((np.array(r["H1"]) - np.array(r["H0"])) - (ref["H1"] - ref["H0"])).max() <= 1e-8
    assert np.abs(dth.cpu().numpy() - ref["theta"]).max() <= 1e-9
    g.close()
