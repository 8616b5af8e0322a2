"""Host logic of the tau-slab path (paper_2508_16298_b200/slab.py) on CPU: the product's
exchange / sign / range / sum logic driven with the oracle as the arithmetic (tests/slab_cpu_ops.py), in one process (several
slabs per process) and over gloo with world_size 2, against the oracle's GLOBAL operators and PCG (Eq.8,
:250-261 Eq.20, :316-326)."""
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2508_16298_b200 import inputs
from paper_2508_16298_b200.slab import SlabLayout, SlabSolver
from tests.slab_cpu_ops import OracleSlabOps

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def parts(a, lay):
    """The owned parts of a global array for the slabs of this process."""
    return [torch.from_numpy(np.ascontiguousarray(a[lay.bounds[g]:lay.bounds[g + 1]])) for g in lay.owned]


def gather(vs, lay, sol):
    return np.concatenate([sol.own(v, i).numpy() for i, v in enumerate(vs)], axis=0)


def test_layout_covers_the_lattice_once():
    lay = SlabLayout(8, 26, 3, W=6)
    assert [lay.nt(g) for g in range(3)] == [8, 9, 9] and lay.bounds[-1] == 26
    assert lay.ext_slices(0)[:6] == [20, 21, 22, 23, 24, 25] and lay.ext_slices(2)[-6:] == [0, 1, 2, 3, 4, 5]
    with pytest.raises(AssertionError):
        SlabLayout(8, 10, 2, W=6)          # a slab shorter than the halo


def test_layout_properties_on_random_shapes():
    """Any admissible (Ntau, slabs, W, world): the slabs tile [0, Ntau) once, sizes differ by at most one, every process owns the
    same number of consecutive slabs, and a slab's extended lattice is its slices with H slices of its neighbours either side."""
    rng = np.random.default_rng(5)
    seen = 0
    for _ in range(300):
        W = int(rng.integers(0, 9)); world = int(rng.integers(1, 5)); per = int(rng.integers(1, 4)); S = world * per
        Nt = int(rng.integers(S * max(1, W), S * max(1, W) + 60))
        lay = [SlabLayout(4, Nt, S, W=W, world=world, rank=r) for r in range(world)]
        sizes = [lay[0].nt(g) for g in range(S)]
        assert sum(sizes) == Nt and max(sizes) - min(sizes) <= 1 and min(sizes) >= lay[0].H
        assert sorted(g for l in lay for g in l.owned) == list(range(S)) and all(len(l.owned) == per for l in lay)
        covered = []
        for g in range(S):
            ext = lay[0].ext_slices(g)
            H, n = lay[0].H, lay[0].nt(g)
            assert len(ext) == n + 2 * H and ext[H:H + n] == list(range(lay[0].bounds[g], lay[0].bounds[g + 1]))
            assert ext[:H] == [(lay[0].bounds[g] - H + j) % Nt for j in range(H)] and ext[H + n:] == [(lay[0].bounds[g + 1] + j) % Nt for j in range(H)]
            assert lay[0].owner(g) == g // per
            covered += ext[H:H + n]
        assert covered == list(range(Nt))
        seen += 1
    assert seen == 300


@pytest.mark.parametrize("S,W", [(1, 6), (2, 6), (3, 2), (4, 0)])
def test_slab_operators_and_pcg_equal_the_global_ones(S, W):
    L, Nt = 4, 26
    theta = inputs.theta_uniform(L, Nt, 7)
    v = inputs.complex_gaussian((Nt, L, L), 7)
    o = orc.Oracle(L, Nt, W=W)
    lay = SlabLayout(L, Nt, S, W=W)
    ops = OracleSlabOps(lay)
    sol = SlabSolver(lay, ops)
    sol.set_theta(parts(theta, lay))
    for g in lay.owned:                    # the extended theta of every slab is the global one at the extended slices
        assert np.array_equal(sol.theta_ext[g].numpy(), theta[lay.ext_slices(g)])
    vs = sol.extend(parts(v, lay), ops.new_vec)
    outs = [ops.new_vec(i) for i in range(S)]
    assert rel(gather(sol.apply_M(vs, outs), lay, sol), o.apply_M(theta, v)) <= 1e-14
    assert rel(gather(sol.apply_Mdag(vs, outs), lay, sol), o.apply_Mdag(theta, v)) <= 1e-14
    assert rel(gather(sol.apply_MdagM(vs, outs), lay, sol), o.apply_MdagM(theta, v)) <= 1e-14
    if W:
        assert rel(gather(sol.precond(vs, outs), lay, sol), o.precond(v)) <= 1e-14
    fo = [ops.new_field(i) for i in range(S)]
    ref = o.force_fermion(theta, v)
    assert np.abs(gather(sol.force(vs, fo), lay, sol) - ref).max() <= 1e-13 * np.abs(ref).max()
    phi = o.apply_Mdag(theta, v)
    xs = [ops.new_vec(i) for i in range(S)]
    it, relres, conv = sol.solve(sol.extend(parts(phi, lay), ops.new_vec), xs, 1e-10, 5000)
    x_ref, it_ref, rel_ref = o.pcg(theta, phi, 1e-10, 5000)
    assert conv and abs(it - it_ref) <= 2 and relres <= 1e-10
    assert rel(gather(xs, lay, sol), x_ref) <= 1e-9
    it, relres, conv = sol.solve(sol.extend(parts(phi, lay), ops.new_vec), xs, 0.0, 9)      # fixed count
    x9, it9, rel9 = o.pcg(theta, phi, 0.0, 9)
    assert it == it9 == 9 and rel(gather(xs, lay, sol), x9) <= 1e-12 and abs(relres - rel9) <= 1e-10 * rel9


@pytest.mark.parametrize("S,compact", [(1, True), (3, True), (2, False)])
def test_slab_trajectory_equals_the_oracles(S, compact):
    """Leapfrog trajectory on the sharded lattice (drift, extended theta with the neighbours' slices, sharded solve, fermion and
    boson force, energies summed over owned slices) against the oracle's trajectory (PAPER.md:207-214 Eq.16, :181 Eq.12)."""
    L, Nt, W = 4, 24, 4
    theta, p = inputs.theta_uniform(L, Nt, 5), inputs.momenta(L, Nt, 5)
    eta = inputs.complex_gaussian((Nt, L, L), 5)
    o = orc.Oracle(L, Nt, W=W, compact=compact, c_tau=0.7, K=1.3)
    phi = o.apply_Mdag(theta, eta)
    ref = o.trajectory(theta, p, phi, 3, 0.05, cg_tol=1e-13)
    lay = SlabLayout(L, Nt, S, W=W)
    ops = OracleSlabOps(lay, compact=compact, c_tau=0.7, K=1.3)
    sol = SlabSolver(lay, ops)
    th_own = [t.clone() for t in parts(theta, lay)]
    p_own = [t.clone() for t in parts(p, lay)]
    r = sol.trajectory(th_own, p_own, sol.extend(parts(phi, lay), ops.new_vec), 3, 0.05, cg_tol=1e-13)
    assert r["converged"] and abs(r["cg_iters"] - ref["cg_iters"]) <= 8
    assert abs(r["H0"] - ref["H0"]) <= 1e-9 and abs((r["H1"] - r["H0"]) - (ref["H1"] - ref["H0"])) <= 1e-9
    assert np.abs(np.concatenate([t.numpy() for t in th_own]) - ref["theta"]).max() <= 1e-11
    assert np.abs(np.concatenate([t.numpy() for t in p_own]) - ref["p"]).max() <= 1e-10


WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
from oracle import oracle as orc
from paper_2508_16298_b200 import inputs
from paper_2508_16298_b200.slab import SlabLayout, SlabSolver
from tests.slab_cpu_ops import OracleSlabOps
rank, world, S = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"]), int(sys.argv[3])
dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{sys.argv[2]}", rank=rank, world_size=world)
orc.set_threads(1)
L, Nt, W = 4, 30, 6
theta = inputs.theta_uniform(L, Nt, 11)
eta = inputs.complex_gaussian((Nt, L, L), 11)
o = orc.Oracle(L, Nt, W=W)
phi = o.apply_Mdag(theta, eta)
lay = SlabLayout(L, Nt, S, W=W, world=world, rank=rank)
ops = OracleSlabOps(lay)
sol = SlabSolver(lay, ops)
part = lambda a: [torch.from_numpy(np.ascontiguousarray(a[lay.bounds[g]:lay.bounds[g + 1]])) for g in lay.owned]
sol.set_theta(part(theta))                              # every rank passes ONLY its own slices; halos arrive over gloo
vs = sol.extend(part(eta), ops.new_vec)
outs = [ops.new_vec(i) for i in range(len(lay.owned))]
sol.apply_MdagM(vs, outs)
ref = o.apply_MdagM(theta, eta)
e_op = max(float(np.abs(sol.own(outs[i], i).numpy() - ref[lay.bounds[g]:lay.bounds[g + 1]]).max()) for i, g in enumerate(lay.owned))
xs = [ops.new_vec(i) for i in range(len(lay.owned))]
it, relres, conv = sol.solve(sol.extend(part(phi), ops.new_vec), xs, 1e-10, 5000)
x_ref, it_ref, _ = o.pcg(theta, phi, 1e-10, 5000)
e_x = max(float(np.abs(sol.own(xs[i], i).numpy() - x_ref[lay.bounds[g]:lay.bounds[g + 1]]).max()) for i, g in enumerate(lay.owned))
p = inputs.momenta(L, Nt, 11)
tr = o.trajectory(theta, p, phi, 2, 0.05, cg_tol=1e-13)
th_own, p_own = [v.clone() for v in part(theta)], [v.clone() for v in part(p)]
r = sol.trajectory(th_own, p_own, sol.extend(part(phi), ops.new_vec), 2, 0.05, cg_tol=1e-13)
e_th = max(float(np.abs(th_own[i].numpy() - tr["theta"][lay.bounds[g]:lay.bounds[g + 1]]).max()) for i, g in enumerate(lay.owned))
e_H = max(abs(r["H0"] - tr["H0"]), abs((r["H1"] - r["H0"]) - (tr["H1"] - tr["H0"])))
dist.barrier()
print(f"RESULT {rank} {e_op / np.abs(ref).max():.3e} {e_x / np.abs(x_ref).max():.3e} {it} {it_ref} {int(conv)} {e_th:.3e} {e_H:.3e}")
dist.destroy_process_group()
'''


@pytest.mark.parametrize("world,S", [(2, 2), (2, 4), (3, 3)])
def test_slab_pcg_gloo(tmp_path, world, S):
    """N>1 path: two processes with one or two slabs each (both neighbours of a rank are the same peer) and three processes
    (distinct peers below and above), halos and sums over gloo; every rank's slices of M^+M v and of the PCG
    solution equal the oracle's global result, and so does a two-step leapfrog trajectory (theta', H0, dH)."""
    script = tmp_path / "slab_worker.py"
    script.write_text(WORKER)
    port = 30100 + (os.getpid() % 300) + 10 * world + S
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT, str(port), str(S)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    seen = 0
    for out, _ in outs:
        for line in out.splitlines():
            if line.startswith("RESULT"):
                _, rank, e_op, e_x, it, it_ref, conv, e_th, e_H = line.split()
                assert float(e_op) <= 1e-14 and float(e_x) <= 1e-9 and abs(int(it) - int(it_ref)) <= 2 and conv == "1"
                assert float(e_th) <= 1e-11 and float(e_H) <= 1e-9            # the trajectory: theta' and H0, dH on every rank
                seen += 1
    assert seen == world
