"""GPU parity of the tau-slab path (include/hqmc.h "tau-slab sharding"): the lattice cut into
S slabs, every slab an ordinary libhqmc.so context on its extended lattice, halos exchanged and sums combined by
paper_2508_16298_b200/slab.py -- here all slabs on ONE GPU, slab after slab (nothing waits on anything), which runs the same
kernels, ranges, signs and sums as one slab per GPU.  Against the oracle's GLOBAL operators and PCG (Eq.8,
:250-261 Eq.20, :316-326, :455-477): <= 1e-12 per operator, 1e-13 for P, 1e-9 per force component and CG solution, iteration
counts within max(2, 1 %), the converged residual judged by the oracle's operator (reading C16)."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2508_16298_b200 import inputs
from paper_2508_16298_b200.slab import CudaSlabOps, SlabLayout, SlabSolver

pytestmark = pytest.mark.gpu


def rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def parts(a, lay):
    return [torch.from_numpy(np.ascontiguousarray(a[lay.bounds[g]:lay.bounds[g + 1]])).cuda() for g in lay.owned]


def gather(vs, sol):
    return np.concatenate([sol.own(v, i).cpu().numpy() for i, v in enumerate(vs)], axis=0)


def make(L, Nt, S, W, theta):
    lay = SlabLayout(L, Nt, S, W=W)
    ops = CudaSlabOps(lay)
    sol = SlabSolver(lay, ops)
    sol.set_theta(parts(theta, lay))
    return lay, ops, sol


@pytest.mark.parametrize("L,Nt,S,W", [(8, 40, 1, 6), (8, 40, 2, 6), (8, 41, 3, 6), (6, 24, 4, 2), (48, 64, 2, 6), (64, 42, 2, 6)])
def test_slab_operators_equal_the_oracles_global_ones(cuda_device, L, Nt, S, W):
    """M, M^+, M^+M, P and the fermion force of the sharded lattice, incl. uneven slabs, the streaming kernels' sizes (L = 48)
    and the cluster kernel's (L = 64)."""
    theta = inputs.theta_uniform(L, Nt, 21)
    v = inputs.complex_gaussian((Nt, L, L), 21)
    o = orc.Oracle(L, Nt, W=W)
    orc.set_threads(orc.max_threads())
    lay, ops, sol = make(L, Nt, S, W, theta)
    for i, g in enumerate(lay.owned):
        assert np.array_equal(sol.theta_ext[i].cpu().numpy(), theta[lay.ext_slices(g)])
    vs = sol.extend(parts(v, lay), ops.new_vec)
    outs = [ops.new_vec(i) for i in range(S)]
    assert rel(gather(sol.apply_M(vs, outs), sol), o.apply_M(theta, v)) <= 1e-12
    assert rel(gather(sol.apply_Mdag(vs, outs), sol), o.apply_Mdag(theta, v)) <= 1e-12
    assert rel(gather(sol.apply_MdagM(vs, outs), sol), o.apply_MdagM(theta, v)) <= 1e-12
    assert rel(gather(sol.precond(vs, outs), sol), o.precond(v)) <= 1e-13
    fo = [ops.new_field(i) for i in range(S)]
    ref = o.force_fermion(theta, v)
    assert np.abs(gather(sol.force(vs, fo), sol) - ref).max() <= 1e-9 * max(1.0, np.abs(ref).max())
    ops.close()


@pytest.mark.parametrize("S", [1, 2, 3])
def test_slab_pcg_equals_the_oracles_and_the_one_context_solve(cuda_device, S):
    from paper_2508_16298_b200 import hqmc
    L, Nt, W = 8, 40, 6
    theta = inputs.theta_uniform(L, Nt, 22)
    eta = inputs.complex_gaussian((Nt, L, L), 22)
    o = orc.Oracle(L, Nt, W=W)
    phi = o.apply_Mdag(theta, eta)
    lay, ops, sol = make(L, Nt, S, W, theta)
    rhs = sol.extend(parts(phi, lay), ops.new_vec)
    xs = [ops.new_vec(i) for i in range(S)]
    it, relres, conv = sol.solve(rhs, xs, 1e-10, 100000)
    x_ref, it_ref, rel_ref = o.pcg(theta, phi, 1e-10, 100000)
    x = gather(xs, sol)
    assert conv and relres <= 1e-10 and abs(it - it_ref) <= max(2, it_ref // 100), (it, it_ref)
    assert rel(x, x_ref) <= 1e-9
    assert np.linalg.norm((phi - o.apply_MdagM(theta, x)).ravel()) / np.linalg.norm(phi.ravel()) <= 1.05e-10
    g = hqmc.HQMC(L, Nt, W=W)                           # the unsharded solve of the same library
    g.set_theta(torch.from_numpy(theta).cuda())
    x1, it1, rel1, ok1 = g.cg_solve(torch.from_numpy(phi).cuda(), 1e-10, 100000)
    assert ok1 and abs(it - it1) <= 2 and rel(x, x1.cpu().numpy()) <= 1e-9
    it, relres, conv = sol.solve(rhs, xs, 0.0, 25)      # fixed count: iterates element by element
    x25, it25, rel25 = o.pcg(theta, phi, 0.0, 25)
    assert it == it25 == 25 and rel(gather(xs, sol), x25) <= 1e-11 and abs(relres - rel25) <= 1e-9 * rel25
    x_plain = [v.clone() for v in xs]
    for n_it in (25, 24, 25):                           # pairs of iterations replayed as one CUDA graph: bit for bit the same
        itg, relg, _ = sol.solve(rhs, xs, 0.0, n_it, graph=True)
        assert itg == n_it
    assert relg == relres and all(torch.equal(a, b) for a, b in zip(xs, x_plain))
    it2, _, _ = sol.solve(rhs, xs, 1e-10, 100000, check_every=16)       # sparse host checks overshoot by < 16 iterations
    assert it_ref - 2 <= it2 < it_ref + 2 + 16
    assert np.linalg.norm((phi - o.apply_MdagM(theta, gather(xs, sol))).ravel()) / np.linalg.norm(phi.ravel()) <= 1.05e-10
    g.close(); ops.close()


@pytest.mark.parametrize("S,compact", [(1, True), (2, True), (3, False)])
def test_slab_trajectory_dH_and_reversibility(cuda_device, S, compact):
    """Leapfrog trajectory on the sharded lattice against the oracle's (Eq.16): H0, dH <= 1e-8, theta' <= 1e-10,
    p' <= 1e-9, and the reversed trajectory returns to the start to <= 1e-10 (tight solves, reading C17)."""
    L, Nt, W, nsteps, eps = 6, 26, 6, 4, 0.05
    theta, p = inputs.theta_uniform(L, Nt, 23), inputs.momenta(L, Nt, 23)
    eta = inputs.complex_gaussian((Nt, L, L), 23)
    kw = dict(compact=compact, c_tau=0.8, K=1.2)
    o = orc.Oracle(L, Nt, W=W, **kw)
    phi = o.apply_Mdag(theta, eta)
    ref = o.trajectory(theta, p, phi, nsteps, eps, cg_tol=1e-13)
    lay = SlabLayout(L, Nt, S, W=W)
    ops = CudaSlabOps(lay, **kw)
    sol = SlabSolver(lay, ops)
    th_own, p_own = parts(theta, lay), parts(p, lay)
    phis = sol.extend(parts(phi, lay), ops.new_vec)
    r = sol.trajectory(th_own, p_own, phis, nsteps, eps, cg_tol=1e-13)
    assert r["converged"]
    assert abs(r["H0"] - ref["H0"]) <= 1e-8 and abs((r["H1"] - r["H0"]) - (ref["H1"] - ref["H0"])) <= 1e-8
    th = np.concatenate([t.cpu().numpy() for t in th_own]); pp = np.concatenate([t.cpu().numpy() for t in p_own])
    assert np.abs(th - ref["theta"]).max() <= 1e-10 and np.abs(pp - ref["p"]).max() <= 1e-9 * max(1.0, np.abs(ref["p"]).max())
    for t in p_own:
        t.neg_()
    sol.trajectory(th_own, p_own, phis, nsteps, eps, cg_tol=1e-13)
    th = np.concatenate([t.cpu().numpy() for t in th_own]); pp = np.concatenate([t.cpu().numpy() for t in p_own])
    assert np.abs(th - theta).max() <= 1e-10 and np.abs(pp + p).max() <= 1e-10 * max(1.0, np.abs(p).max())
    ops.close()


def test_config2_solve_in_four_slabs(cuda_device):
    """BASELINE config 2 (L=12, Ntau=120, heat-bath theta) solved to 1e-10 in four slabs of 30 slices."""
    c = inputs.CONFIGS[2]
    L, Nt = c["L"], c["Ntau"]
    theta = inputs.make_theta(2)
    eta = inputs.complex_gaussian((Nt, L, L), c["seed"])
    o = orc.Oracle(L, Nt)
    orc.set_threads(orc.max_threads())
    phi = o.apply_Mdag(theta, eta)
    lay, ops, sol = make(L, Nt, 4, 6, theta)
    xs = [ops.new_vec(i) for i in range(4)]
    it, relres, conv = sol.solve(sol.extend(parts(phi, lay), ops.new_vec), xs, 1e-10, 200000)
    x_ref, it_ref, _ = o.pcg(theta, phi, 1e-10, 200000)
    x = gather(xs, sol)
    assert conv and relres <= 1e-10 and abs(it - it_ref) <= max(2, it_ref // 100), (it, it_ref)
    assert np.linalg.norm((phi - o.apply_MdagM(theta, x)).ravel()) / np.linalg.norm(phi.ravel()) <= 1.05e-10
    assert rel(x, x_ref) <= 1e-9
    ops.close()
