"""(1) Oracle against the stored theta = 0 closed-form values (tests/golden/free_fermion_closed_form.txt, written by
tests/golden/make_free_fermion_golden.py from the mathematics alone); (2) the multi-GPU host logic (replicas only,
DESIGN.md "Multi-GPU") over gloo with world_size 2; (3) bench.py's reference arm and JSON contract on a tiny config.
CPU only."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from oracle import oracle as orc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLD = os.path.join(ROOT, "tests", "golden", "free_fermion_closed_form.txt")


def _golden():
    rows = []
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        rows.append((int(f[0]), int(f[1])) + tuple(float(x) for x in f[2:]))
    return rows


@pytest.mark.parametrize("row", _golden(), ids=lambda r: f"L{r[0]}_Nt{r[1]}")
def test_oracle_matches_free_fermion_golden(row):
    L, Nt, logdet, lmin, lmax, trace = row
    o = orc.Oracle(L, Nt)
    Vs = L * L
    # trace(M^+M) = N + Ntau * tr(B^2) at theta = 0 (every slice equal): needs only the oracle's single-slice B
    th = np.zeros((2, L, L))
    E = np.eye(Vs, dtype=np.complex128)
    B = np.stack([o.apply_B(th, e) for e in E], axis=1)
    assert abs((o.N + Nt * np.trace(B @ B).real) - trace) < 1e-11 * trace
    if o.N <= 1000:   # dense spectrum and determinant through the oracle's full M
        theta = np.zeros((Nt, 2, L, L))
        M = np.stack([o.apply_M(theta, e) for e in np.eye(o.N, dtype=np.complex128)], axis=1)
        ev = np.linalg.eigvalsh(M.conj().T @ M)
        assert abs(ev.min() - lmin) < 1e-12 and abs(ev.max() - lmax) < 1e-12
        sign, ld = np.linalg.slogdet(M)
        assert abs(ld - logdet) < 1e-10 and abs(sign - 1.0) < 1e-10      # det M real and positive
    else:             # extreme eigenvalues by Rayleigh quotients of M^+M bracket the closed-form spectrum
        theta = np.zeros((Nt, 2, L, L))
        rng = np.random.default_rng(7)
        for _ in range(3):
            v = rng.standard_normal(o.N) + 1j * rng.standard_normal(o.N)
            q = np.vdot(v, o.apply_MdagM(theta, v)).real / np.vdot(v, v).real
            assert lmin * (1 - 1e-12) <= q <= lmax * (1 + 1e-12)


WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
from paper_2508_16298_b200 import replicas
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{sys.argv[2]}", rank=rank, world_size=world)
seed = replicas.replica_seed(3, rank)
t, u = replicas.aggregate(1.0 + rank, 100 * (rank + 1), world)   # rank 1 is slower and did more work
dist.barrier()
print(f"RESULT {rank} {seed} {t} {u}")
dist.destroy_process_group()
'''


def test_replicas_gloo_world2(tmp_path):
    """N>1 path: every rank runs its own lattice (distinct seed), time = max over ranks, work = sum over ranks."""
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = 29500 + (os.getpid() % 500)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT, str(port)], env=env, stdout=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=120)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    res = {}
    for o in outs:
        for line in o.splitlines():
            if line.startswith("RESULT"):
                _, rank, seed, t, u = line.split()
                res[int(rank)] = (int(seed), float(t), int(u))
    assert res[0][0] == 3 and res[1][0] != res[0][0]
    assert res[0][1:] == res[1][1:] == (2.0, 300)


def test_replica_seed_and_single_rank_aggregate():
    from paper_2508_16298_b200 import replicas
    assert replicas.replica_seed(4, 0) == 4
    assert len({replicas.replica_seed(4, r) for r in range(8)}) == 8
    assert replicas.aggregate(1.5, 7, 1) == (1.5, 7)


def test_bench_reference_arm_json_contract():
    """bench.py --impl reference runs the oracle on the host cores and prints the contract's JSON line."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "2",
                          "--warmup", "1", "--ref-cg-iters", "3"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in line, k
    assert line["impl"] == "reference" and line["value"] > 0 and line["unit"] == "Gsite/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    # `config` names the WORKLOAD (the GPU arm's: 500 fixed iterations per solve), `sample` what was run of it
    assert line["config"]["cg_iters_per_solve"] == 500 and " 3 of its 500 " in line["cpu_baseline"]["sample"]
