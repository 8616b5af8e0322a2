"""CPU stand-in for the arithmetic of the tau-slab path (paper_2508_16298_b200/slab.py), TEST INFRASTRUCTURE ONLY: the
operators of a slab's extended lattice come from the oracle, the vector steps are numpy.  It lets the CPU tests drive the
product's host logic (who sends what to whom, which sign, which range, which sum) over gloo without a GPU."""
import numpy as np
import torch

from oracle import oracle as orc


class OracleSlabOps:
    def __init__(self, lay, **params):
        self.lay = lay
        self.o = [orc.Oracle(lay.L, lay.nt_ext(g), W=lay.W, **params) for g in lay.owned]
        self.theta = [None] * len(lay.owned)

    def new_vec(self, i):
        return torch.zeros((self.lay.nt_ext(self.lay.owned[i]), self.lay.L, self.lay.L), dtype=torch.complex128)

    def new_field(self, i):
        return torch.zeros((self.lay.nt_ext(self.lay.owned[i]), 2, self.lay.L, self.lay.L), dtype=torch.float64)

    def scalars(self, *shape):
        return torch.zeros(shape, dtype=torch.float64)

    def set_theta(self, i, theta_ext):
        self.theta[i] = theta_ext.numpy().copy()

    def _op(self, i, fn, v, out):
        out.copy_(torch.from_numpy(fn(self.theta[i], v.numpy())))

    def apply_M(self, i, v, out):
        self._op(i, self.o[i].apply_M, v, out)

    def apply_Mdag(self, i, v, out):
        self._op(i, self.o[i].apply_Mdag, v, out)

    def apply_MdagM(self, i, v, out):
        self._op(i, self.o[i].apply_MdagM, v, out)

    def precond(self, i, r, z):
        z.copy_(torch.from_numpy(self.o[i].precond(r.numpy())))

    def force(self, i, x, out):
        out.copy_(torch.from_numpy(self.o[i].force_fermion(self.theta[i], x.numpy())))

    def force_boson(self, i, out):
        out.copy_(torch.from_numpy(self.o[i].force_boson(self.theta[i])))

    def field_axpy(self, i, y, x, a):
        y += a * x

    def action_boson(self, i, first, count, out):
        """The share of S_B of the slices [first, first + count): plaquettes of those slices and the temporal terms t -> t + 1."""
        th = self.theta[i]
        P = self.o[i].P
        tx, ty = th[first:first + count, 0], th[first:first + count, 1]
        curl = tx + np.roll(ty, -1, axis=2) - np.roll(tx, -1, axis=1) - ty          # theta_x(s) + theta_y(s+x) - theta_x(s+y) - theta_y(s)
        d = th[first + 1:first + count + 1] - th[first:first + count]
        temporal = (1.0 - np.cos(d)).sum() if P.compact else (d * d).sum()
        out[0] = float(P.c_tau * temporal + P.K * np.cos(curl).sum())

    def sum_squares(self, i, f, out):
        out[0] = float((f.numpy() ** 2).sum())

    def dot(self, i, a, b, out):
        out[0] = float(np.vdot(a.numpy().ravel(), b.numpy().ravel()).real)

    def axpy(self, i, x, r, d, Od, num, den, rr_out):
        alpha = float(num[0]) / float(den[0])
        x += alpha * d
        r -= alpha * Od
        rr_out[0] = float(np.vdot(r.numpy().ravel(), r.numpy().ravel()).real)

    def dupdate(self, i, d, z, num, den):
        beta = float(num[0]) / float(den[0])
        d.copy_(z + beta * d)

    def scale(self, i, v, s):
        v *= s

    def sum_rows(self, rows, c0, c1, out):
        out[c0:c1] = rows[:, c0:c1].sum(dim=0)
