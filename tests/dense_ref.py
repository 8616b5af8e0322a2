"""Dense, textbook constructions used ONLY to pin the oracle (tests/test_oracle_*.py).

Independent of oracle/ and of the CUDA path: every family factor is a generic scipy matrix
exponential of the dense hopping matrix of that family (not the cosh/sinh closed form), and M is
assembled block by block from PAPER.md:155 (Eq.8).
"""
import numpy as np
import scipy.linalg as sla


def family_bonds(L, fam):
    """[(i, j, mu, x, y)] for bond family fam in 1..4 (reading C4)."""
    out = []
    mu = 0 if fam <= 2 else 1
    par = 0 if fam in (1, 3) else 1
    for y in range(L):
        for x in range(L):
            c = x if mu == 0 else y
            if c % 2 != par:
                continue
            i = x + L * y
            j = ((x + 1) % L + L * y) if mu == 0 else (x + L * ((y + 1) % L))
            out.append((i, j, mu, x, y))
    return out


def family_matrix(L, th_slice, fam):
    """Dense sum of T_ij over the family: [i,j] = e^{i theta}, [j,i] = e^{-i theta}."""
    Vs = L * L
    V = np.zeros((Vs, Vs), dtype=np.complex128)
    for (i, j, mu, x, y) in family_bonds(L, fam):
        V[i, j] += np.exp(1j * th_slice[mu, y, x])
        V[j, i] += np.exp(-1j * th_slice[mu, y, x])
    return V


def dense_B(L, th_slice, dtau=0.1, t=1.0):
    """Eq.22: B = e^{V4/2} e^{V3/2} e^{V2/2} e^{V1/2} e^{V1/2} e^{V2/2} e^{V3/2} e^{V4/2}."""
    E = {f: sla.expm(0.5 * dtau * t * family_matrix(L, th_slice, f)) for f in (1, 2, 3, 4)}
    return E[4] @ E[3] @ E[2] @ E[1] @ E[1] @ E[2] @ E[3] @ E[4]


def dense_M(L, Ntau, theta, dtau=0.1, t=1.0):
    """Eq.8: 1 on the diagonal, -B_t in block (t+1, t), +B_{Nt-1} in block (0, Nt-1)."""
    Vs = L * L
    M = np.eye(Ntau * Vs, dtype=np.complex128)
    Bs = [dense_B(L, theta[tt], dtau, t) for tt in range(Ntau)]
    for tt in range(Ntau - 1):
        M[(tt + 1) * Vs:(tt + 2) * Vs, tt * Vs:(tt + 1) * Vs] = -Bs[tt]
    M[0:Vs, (Ntau - 1) * Vs:Ntau * Vs] = Bs[Ntau - 1]
    return M, Bs


def dense_SB(theta, c_tau, K, compact=True):
    """PAPER.md:52-54 written with numpy rolls (axes tau, mu, y, x)."""
    d = np.roll(theta, -1, axis=0) - theta
    st = (1.0 - np.cos(d)).sum() if compact else (d * d).sum()
    ax, ay = theta[:, 0], theta[:, 1]
    curl = ax + np.roll(ay, -1, axis=2) - np.roll(ax, -1, axis=1) - ay
    return c_tau * st + K * np.cos(curl).sum()
