"""tau-slab sharding of the hot path over several GPUs (include/hqmc.h "tau-slab sharding").

`M` and `M^+` couple time slice t only to t -+ 1 (Eq.8), the preconditioner to t +- W, the
force is local to a slice given X of the next one: the lattice shards into contiguous runs of slices.

  * The Ntau slices are dealt out to `n_slabs` slabs as evenly as possible; a process owns `n_slabs / world` consecutive slabs
    (one per GPU in production; several per process lets ONE GPU run the whole scheme, slab after slab, for tests and timing).
  * A slab stores every vector on its EXTENDED lattice: its nt_loc owned slices with H = max(1, W) halo slices on either
    side.  Before `M^+M` the halo of d is refreshed one slice deep, before `P` the halo of r W slices deep: from the
    neighbouring slab by a device copy when this process owns it, else by a send / receive pair (torch.distributed: NCCL
    over NVLink on GPUs, gloo in the CPU tests).  A halo that crossed the antiperiodic boundary tau = Ntau-1 -> 0 is
    multiplied by -1 (reading C1); the operators of the extended lattice then return on the owned slices exactly what the
    global operators return (their own wrap only reaches the outermost halo slices, which are never used).
  * Inner products run over the owned slices only (one contiguous range), are summed over the process's slabs in slab
    order, then all-reduced; alpha and beta stay on the device as quotients of those sums, so the host reads one number per
    convergence test and nothing else.

This module is the host logic (who sends what to whom, which sign, which range, which sum): every arithmetic step is a call
into an `ops` object.  `CudaSlabOps` is the product's (libhqmc.so kernels; no CPU fallback); the CPU tests drive the same
logic over gloo with an `ops` of their own.  PCG as in hqmc_cg_solve: x_0 = 0, d_0 = P r_0, stop on ||r|| / ||rhs|| <= tol
after the r update, tol <= 0 = exactly max_iter iterations (PAPER.md:250-261 Eq.20, :348; readings C8, C9).
"""
from __future__ import annotations

import contextlib

import torch

# columns of the scalar table: ||rhs||^2, <d,Od>, then (||r||^2, <r,z>) of even and of odd iterations
BB, DOD, RR0, RZ0, RR1, RZ1, NSCAL = 0, 1, 2, 3, 4, 5, 6


class SlabLayout:
    """Which slices a slab owns and what its extended lattice looks like."""

    def __init__(self, L: int, Ntau: int, n_slabs: int, W: int = 6, world: int = 1, rank: int = 0):
        assert n_slabs >= 1 and world >= 1 and n_slabs % world == 0, "every process owns the same number of slabs"
        self.L, self.Ntau, self.S, self.W, self.H = L, Ntau, n_slabs, W, max(1, W)
        self.world, self.rank, self.per = world, rank, n_slabs // world
        self.bounds = [(g * Ntau) // n_slabs for g in range(n_slabs + 1)]
        assert min(self.nt(g) for g in range(n_slabs)) >= self.H, "a halo must come from the immediate neighbour alone"
        self.owned = list(range(rank * self.per, (rank + 1) * self.per))

    def nt(self, g: int) -> int:
        return self.bounds[g + 1] - self.bounds[g]

    def nt_ext(self, g: int) -> int:
        return self.nt(g) + 2 * self.H

    def owner(self, g: int) -> int:
        return g // self.per

    def ext_slices(self, g: int):
        """Global slice index of every slice of slab g's extended lattice."""
        return [(self.bounds[g] - self.H + j) % self.Ntau for j in range(self.nt_ext(g))]

    def own(self, v: torch.Tensor, g: int) -> torch.Tensor:
        """The owned slices of an extended tensor (contiguous view)."""
        return v[self.H:self.H + self.nt(g)]


class SlabComm:
    """Halo exchange and sums for the slabs of one process."""

    def __init__(self, lay: SlabLayout, ops, group=None):
        self.lay, self.ops, self.group = lay, ops, group
        if lay.world > 1:
            import torch.distributed as dist
            assert dist.is_initialized() and dist.get_world_size(group) == lay.world and dist.get_rank(group) == lay.rank

    def exchange(self, vs, h: int, antiperiodic: bool = True):
        """Fill h halo slices on either side of every owned slab's extended tensor vs[i] (leading axis = slices)."""
        lay, H, S = self.lay, self.lay.H, self.lay.S
        assert 1 <= h <= H and len(vs) == len(lay.owned)
        sends, recvs = [], []
        for i, g in enumerate(lay.owned):
            n = lay.nt(g)
            lo, hi = vs[i][H - h:H], vs[i][H + n:H + n + h]            # my lower / upper halo
            g_dn, g_up = (g - 1) % S, (g + 1) % S
            if lay.owner(g_dn) == lay.rank:                             # last h owned slices of the slab below
                j = lay.owned.index(g_dn)
                lo.copy_(vs[j][H + lay.nt(g_dn) - h:H + lay.nt(g_dn)])
            else:
                recvs.append((1, lo, lay.owner(g_dn)))
                sends.append((0, vs[i][H:H + h], lay.owner(g_dn)))      # my first owned slices are its upper halo
            if lay.owner(g_up) == lay.rank:                             # first h owned slices of the slab above
                j = lay.owned.index(g_up)
                hi.copy_(vs[j][H:H + h])
            else:
                recvs.append((0, hi, lay.owner(g_up)))
                sends.append((1, vs[i][H + n - h:H + n], lay.owner(g_up)))   # my last owned slices are its lower halo
        if sends or recvs:
            import torch.distributed as dist
            # tag 0: "first slices, going down"; tag 1: "last slices, going up".  Per peer the sends are issued in tag order and
            # the receives in the order the peer sends them (NCCL matches by order, gloo by tag): with two processes both
            # neighbours are the same peer.
            sends.sort(key=lambda s: s[0])
            recvs.sort(key=lambda s: s[0])
            p2p = [dist.P2POp(dist.isend, t, peer, self.group, tag) for tag, t, peer in sends]
            p2p += [dist.P2POp(dist.irecv, t, peer, self.group, tag) for tag, t, peer in recvs]
            for req in dist.batch_isend_irecv(p2p):
                req.wait()
        if antiperiodic:
            for i, g in enumerate(lay.owned):
                n = lay.nt(g)
                if g == 0:
                    self.ops.scale(i, vs[i][H - h:H], -1.0)
                if g == S - 1:
                    self.ops.scale(i, vs[i][H + n:H + n + h], -1.0)

    def reduce(self, rows: torch.Tensor, c0: int, c1: int, out: torch.Tensor):
        """out[c0:c1] = sum over the process's slabs (in order) of rows[:, c0:c1], then summed over the processes."""
        self.ops.sum_rows(rows, c0, c1, out)
        if self.lay.world > 1:
            import torch.distributed as dist
            dist.all_reduce(out[c0:c1], op=dist.ReduceOp.SUM, group=self.group)


class CudaSlabOps:
    """The arithmetic of the slabs one process owns: one libhqmc.so context per slab, created for its extended lattice."""

    def __init__(self, lay: SlabLayout, device="cuda:0", **params):
        from . import hqmc                         # raises if libhqmc.so is missing: there is no CPU fallback
        self.lay, self.device = lay, torch.device(device)
        assert self.device.type == "cuda", "the slab path runs in CUDA kernels only"
        # a stream of the path's own (every context enqueues on it), so that a pair of PCG iterations can be captured in a graph
        self.stream = torch.cuda.Stream(self.device)
        with torch.cuda.stream(self.stream):
            self.ctx = [hqmc.HQMC(lay.L, lay.nt_ext(g), W=lay.W, device=device, **params) for g in lay.owned]
        self.cdtype = self.ctx[0].cdtype

    def close(self):
        for c in self.ctx:
            c.close()

    def new_vec(self, i):
        return torch.zeros((self.lay.nt_ext(self.lay.owned[i]), self.lay.L, self.lay.L), dtype=self.cdtype, device=self.device)

    def new_field(self, i):
        return torch.zeros((self.lay.nt_ext(self.lay.owned[i]), 2, self.lay.L, self.lay.L), dtype=torch.float64, device=self.device)

    def scalars(self, *shape):
        return torch.zeros(shape, dtype=torch.float64, device=self.device)

    def set_theta(self, i, theta_ext):
        self.ctx[i].set_theta(theta_ext)

    def apply_M(self, i, v, out):
        self.ctx[i].apply_M(v, out)

    def apply_Mdag(self, i, v, out):
        self.ctx[i].apply_Mdag(v, out)

    def apply_MdagM(self, i, v, out):
        self.ctx[i].apply_MdagM(v, out)

    def precond(self, i, r, z):
        self.ctx[i].precond(r, z)

    def force(self, i, x, out):
        self.ctx[i].force(x, out)

    def force_boson(self, i, out):
        self.ctx[i].force_boson(out)

    def field_axpy(self, i, y, x, a):
        self.ctx[i].slab_field_axpy(y, x, a)

    def action_boson(self, i, first, count, out):
        self.ctx[i].slab_action_boson(first, count, out)

    def sum_squares(self, i, f, out):
        """out[0] = sum of f^2 over a float64 view (its pairs of doubles read as complex numbers: Re <f, f>)."""
        assert self.cdtype == torch.complex128, "the slab trajectory runs in complex128"
        v = torch.view_as_complex(f.reshape(-1, 2))
        self.ctx[i].slab_dot(v, v, out)

    def dot(self, i, a, b, out):
        self.ctx[i].slab_dot(a, b, out)

    def axpy(self, i, x, r, d, Od, num, den, rr_out):
        self.ctx[i].slab_axpy(x, r, d, Od, num, den, rr_out)

    def dupdate(self, i, d, z, num, den):
        self.ctx[i].slab_dupdate(d, z, num, den)

    def scale(self, i, v, s):
        self.ctx[i].slab_scale(v, s)

    def sum_rows(self, rows, c0, c1, out):
        self.ctx[0].slab_sum_rows(rows, c0, c1, out)


class SlabSolver:
    """Operators and the PCG of Eq.20 on a lattice sharded into tau-slabs."""

    def __init__(self, lay: SlabLayout, ops, group=None):
        self.lay, self.ops, self.comm = lay, ops, SlabComm(lay, ops, group)
        k = len(lay.owned)
        self.k = k
        with self._stream():
            self.r = [ops.new_vec(i) for i in range(k)]
            self.z = [ops.new_vec(i) for i in range(k)]       # Od, then z = P r (Od is dead once r is updated)
            self.d = [ops.new_vec(i) for i in range(k)]
            self.rows = ops.scalars(k, NSCAL)                 # per-slab partial sums
            self.s = ops.scalars(NSCAL)                       # their sums over all slabs of all processes
        self._graph, self._graph_key = None, None

    @contextlib.contextmanager
    def _stream(self):
        """Run the body on the ops' own stream (if it has one), ordered after the caller's stream and before what follows."""
        st = getattr(self.ops, "stream", None)
        if st is None:
            yield
            return
        cur = torch.cuda.current_stream(st.device)
        if cur == st:
            yield
            return
        st.wait_stream(cur)
        with torch.cuda.stream(st):
            yield
        cur.wait_stream(st)

    # ---- setting up ---------------------------------------------------------------------------------
    def own(self, v, i):
        return self.lay.own(v, self.lay.owned[i])

    def extend(self, owned_parts, new):
        """Extended tensors (halo zero) from the owned parts [nt_loc, ...] of every owned slab."""
        out = []
        with self._stream():
            for i, part in enumerate(owned_parts):
                e = new(i)
                self.own(e, i).copy_(part)
                out.append(e)
        return out

    def set_theta(self, theta_owned):
        """theta_owned[i]: this process's slices of theta for its i-th slab, [nt_loc][2][L][L].  The halo slices come from the
        neighbours (theta is periodic in tau: no sign, reading C14)."""
        th = self.extend(theta_owned, self.ops.new_field)
        with self._stream():
            self.comm.exchange(th, self.lay.H, antiperiodic=False)
            for i in range(self.k):
                self.ops.set_theta(i, th[i])
        self.theta_ext = th

    # ---- operators on the sharded lattice (v: extended tensors, owned part filled; results: owned part valid) ---------
    def _apply(self, fn, vs, outs, h):
        with self._stream():
            self.comm.exchange(vs, h)
            for i in range(self.k):
                fn(i, vs[i], outs[i])
        return outs

    def apply_M(self, vs, outs):
        return self._apply(self.ops.apply_M, vs, outs, 1)

    def apply_Mdag(self, vs, outs):
        return self._apply(self.ops.apply_Mdag, vs, outs, 1)

    def apply_MdagM(self, vs, outs):
        return self._apply(self.ops.apply_MdagM, vs, outs, 1)

    def precond(self, vs, outs):
        if self.lay.W == 0:
            with self._stream():
                for i in range(self.k):
                    outs[i].copy_(vs[i])
            return outs
        return self._apply(self.ops.precond, vs, outs, self.lay.W)

    def force(self, xs, outs):
        """dS_F/dtheta on the owned slices from the owned slices of X = (M^+M)^{-1} phi (outs: extended fp64 fields)."""
        return self._apply(self.ops.force, xs, outs, 1)

    # ---- PCG ------------------------------------------------------------------------------------------
    def _dots(self, a, b, col):
        for i in range(self.k):
            self.ops.dot(i, self.own(a[i], i), self.own(b[i], i), self.rows[i, col:col + 1])

    @staticmethod
    def _cols(p):
        """(old <r,z>, new ||r||^2, new <r,z>) columns of an even / odd iteration."""
        return (RZ0, RR1, RZ1) if p == 0 else (RZ1, RR0, RZ0)

    def _iteration(self, x, p):
        """Everything of iteration `it` (parity p) up to the stopping test: Od, alpha, x, r, z = P r, the three sums."""
        ops, comm, s, rows, r, z, d = self.ops, self.comm, self.s, self.rows, self.r, self.z, self.d
        rz_old, rr_new, rz_new = self._cols(p)
        self.apply_MdagM(d, z)                                                         # z = Od
        self._dots(d, z, DOD)
        comm.reduce(rows, DOD, DOD + 1, s)
        for i in range(self.k):
            ops.axpy(i, self.own(x[i], i), self.own(r[i], i), self.own(d[i], i), self.own(z[i], i),
                     s[rz_old:rz_old + 1], s[DOD:DOD + 1], rows[i, rr_new:rr_new + 1])
        self.precond(r, z)                                                             # z = P r over the dead Od
        self._dots(r, z, rz_new)
        comm.reduce(rows, rr_new, rz_new + 1, s)

    def _dupdate(self, p):
        rz_old, _, rz_new = self._cols(p)
        for i in range(self.k):
            self.ops.dupdate(i, self.own(self.d[i], i), self.own(self.z[i], i), self.s[rz_new:rz_new + 1], self.s[rz_old:rz_old + 1])

    def _pair(self, x):
        self._iteration(x, 0); self._dupdate(0)
        self._iteration(x, 1); self._dupdate(1)

    def _pair_graph(self, x):
        """A CUDA graph of two iterations (an even and an odd one, each with its d update) on these x tensors."""
        key = tuple(v.data_ptr() for v in x)
        if self._graph is None or self._graph_key != key:
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=self.ops.stream, capture_error_mode="relaxed"):
                self._pair(x)
            self._graph, self._graph_key = g, key
        return self._graph

    def solve(self, rhs, x, tol=1e-10, max_iter=1000000, check_every=1, graph=False):
        """M^+M x = rhs.  rhs, x: extended tensors per owned slab (owned part of rhs filled; owned part of x receives the
        solution).  -> (iterations, ||r|| / ||rhs||, converged).  The host reads the residual every `check_every` iterations
        (1 = the stopping rule of hqmc_cg_solve exactly; larger values overshoot by fewer than check_every iterations).
        graph=True (fixed-count solves, tol <= 0, on CUDA): pairs of iterations are replayed as one CUDA graph,
        exchange and all-reduce included."""
        with self._stream():
            return self._solve(rhs, x, tol, max_iter, check_every, graph)

    def _solve(self, rhs, x, tol, max_iter, check_every, graph):
        comm, s, rows, k = self.comm, self.s, self.rows, self.k
        r, z, d = self.r, self.z, self.d
        for i in range(k):
            self.own(x[i], i).zero_()
            self.own(r[i], i).copy_(self.own(rhs[i], i))
        self._dots(r, r, BB)
        comm.reduce(rows, BB, BB + 1, s)
        self.precond(r, z)
        self._dots(r, z, RZ0)
        comm.reduce(rows, RZ0, RZ0 + 1, s)
        for i in range(k):
            self.own(d[i], i).copy_(self.own(z[i], i))
        it, rel, conv = 0, float("nan"), tol <= 0
        if graph and tol <= 0 and getattr(self.ops, "stream", None) is not None and max_iter >= 4:
            self._pair(x)                                   # the first pair eagerly: it warms up whatever the capture may not do
            it = 2
            g = self._pair_graph(x)
            while it + 2 <= max_iter:
                g.replay()
                it += 2
        bb = None
        while it < max_iter:
            p = it & 1
            self._iteration(x, p)
            it += 1
            if tol > 0 and (it % check_every == 0 or it == max_iter):
                if bb is None:
                    bb = float(s[BB])
                rr = float(s[self._cols(p)[1]])
                if not rr == rr:                            # NaN: det M ~ 0 or overflow
                    break
                if rr <= tol * tol * bb:
                    conv = True
                    break
            if it == max_iter:
                break
            self._dupdate(p)
        if it > 0:
            last = RR1 if (it & 1) == 1 else RR0
            rel = (float(s[last]) / float(s[BB])) ** 0.5 if float(s[BB]) > 0 else 0.0
        return it, rel, conv


    # ---- molecular dynamics on the sharded lattice (PAPER.md:207-214 Eq.16, :181 Eq.12; reading C7) -----------------------
    def energies(self, p_own, phi, x):
        """H = S_B + sum p^2 + Re <phi, x>, every term summed over the owned slices of every slab, then over the processes."""
        lay, ops = self.lay, self.ops
        if not hasattr(self, "_erows"):
            self._erows, self._es = ops.scalars(self.k, 3), ops.scalars(3)
        with self._stream():
            for i, g in enumerate(lay.owned):
                ops.action_boson(i, lay.H, lay.nt(g), self._erows[i, 0:1])
                ops.sum_squares(i, p_own[i], self._erows[i, 1:2])
                ops.dot(i, self.own(phi[i], i), self.own(x[i], i), self._erows[i, 2:3])
            self.comm.reduce(self._erows, 0, 3, self._es)
            e = self._es.cpu()
        return float(e[0]), float(e[1]), float(e[2])

    def _kick(self, p_own, x, h):
        """p -= h (dS_F/dtheta + dS_B/dtheta) on the owned slices."""
        ops = self.ops
        with self._stream():
            self.force(x, self._fF)
            for i in range(self.k):
                ops.force_boson(i, self._fB[i])
                ops.field_axpy(i, p_own[i], self.own(self._fF[i], i), -h)
                ops.field_axpy(i, p_own[i], self.own(self._fB[i], i), -h)

    def trajectory(self, theta_own, p_own, phi, nsteps, eps, cg_tol=1e-10, cg_max_iter=1000000):
        """One leapfrog trajectory, in place on theta_own[i], p_own[i] (this process's slices, [nt_loc][2][L][L] float64,
        contiguous); phi: extended pseudofermion tensors.  -> dict(H0, H1, cg_iters, converged), as hqmc_leapfrog_trajectory."""
        ops = self.ops
        if not hasattr(self, "_fF"):
            with self._stream():
                self._fF = [ops.new_field(i) for i in range(self.k)]
                self._fB = [ops.new_field(i) for i in range(self.k)]
                self._X = [ops.new_vec(i) for i in range(self.k)]
        X, total, ok = self._X, 0, True

        def solve():
            nonlocal total, ok
            it, _, conv = self.solve(phi, X, cg_tol, cg_max_iter)
            total += it
            ok = ok and conv

        self.set_theta(theta_own)
        solve()
        H0 = sum(self.energies(p_own, phi, X))
        self._kick(p_own, X, 0.5 * eps)
        for n in range(nsteps):
            with self._stream():
                for i in range(self.k):
                    ops.field_axpy(i, theta_own[i], p_own[i], 2.0 * eps)          # theta += 2 p eps
            self.set_theta(theta_own)
            solve()
            self._kick(p_own, X, 0.5 * eps if n == nsteps - 1 else eps)
        H1 = sum(self.energies(p_own, phi, X))
        return dict(H0=H0, H1=H1, cg_iters=total, converged=ok)
