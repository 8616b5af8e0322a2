"""Seeded synthetic input generators (shared by the tests of the oracle and of the CUDA path).

This module holds NONE of the method's arithmetic (no sweep, no M, no CG, no force): it only draws
random arrays with the shapes and distributions DESIGN.md §"Input recipe" states, so that the CPU
oracle and the GPU library consume bit-identical inputs.  It imports numpy only.

Layouts: theta[tau][mu][y][x] (mu=0: x-bond s->s+x, mu=1: y-bond s->s+y), vectors
[tau][y][x] complex128.  Random streams: numpy.random.default_rng([seed, stream]) with
stream 0=theta, 1=eta, 2=p, 3=gauge alpha, 4=heat bath, 5=bench vectors.
"""
from __future__ import annotations

import numpy as np

STREAM_THETA, STREAM_ETA, STREAM_P, STREAM_ALPHA, STREAM_HEATBATH, STREAM_VEC = range(6)

# (L, Ntau, seed, theta kind) of the five BASELINE.json configs
CONFIGS = {
    1: dict(L=4, Ntau=8, seed=0, theta="uniform"),
    2: dict(L=12, Ntau=120, seed=1, theta="heatbath"),
    3: dict(L=24, Ntau=240, seed=2, theta="uniform"),
    4: dict(L=48, Ntau=480, seed=3, theta="uniform"),
    5: dict(L=64, Ntau=640, seed=4, theta="heatbath"),
}


def rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.default_rng([seed, stream])


def theta_uniform(L: int, Ntau: int, seed: int) -> np.ndarray:
    """theta ~ U[-pi, pi), shape [Ntau][2][L][L] (BASELINE.json configs 1, 3, 4)."""
    return rng(seed, STREAM_THETA).uniform(-np.pi, np.pi, (Ntau, 2, L, L))


def pi_flux_background(L: int, Ntau: int) -> np.ndarray:
    """A_pi: x-bond at (x, y) carries pi*(y mod 2), y-bonds 0 (flux pi through every plaquette)."""
    a = np.zeros((Ntau, 2, L, L))
    a[:, 0, 1::2, :] = np.pi
    return a


def complex_gaussian(shape, seed: int, stream: int = STREAM_ETA) -> np.ndarray:
    """(N(0,1) + i N(0,1))/sqrt(2): weight exp(-R^dagger R) (reading C6)."""
    g = rng(seed, stream)
    re = g.standard_normal(shape)
    im = g.standard_normal(shape)
    return ((re + 1j * im) / np.sqrt(2.0)).astype(np.complex128)


def momenta(L: int, Ntau: int, seed: int) -> np.ndarray:
    """p ~ N(0, 1/2): weight exp(-sum p^2) (reading C6)."""
    return rng(seed, STREAM_P).standard_normal((Ntau, 2, L, L)) / np.sqrt(2.0)


def gauge_alpha(L: int, seed: int) -> np.ndarray:
    """Site phases alpha[y][x] of a (time-independent) gauge transformation, U[-pi, pi)."""
    return rng(seed, STREAM_ALPHA).uniform(-np.pi, np.pi, (L, L))


def gauge_transform_theta(theta: np.ndarray, alpha: np.ndarray) -> np.ndarray:
    """theta_ij -> theta_ij + alpha_i - alpha_j on every slice (bond i -> j = i + mu)."""
    out = theta.copy()
    out[:, 0] += alpha - np.roll(alpha, -1, axis=1)  # j = (x+1, y)
    out[:, 1] += alpha - np.roll(alpha, -1, axis=0)  # j = (x, y+1)
    return out


def bench_vectors(n: int, L: int, Ntau: int, seed: int) -> np.ndarray:
    return complex_gaussian((n, Ntau, L, L), seed, STREAM_VEC)


# ------------------------------------------------------------------------------------------------
# Heat bath for the pure-gauge Wilson weight exp(+beta * sum_plaq cos(a_plaq)) on the (2+1)d
# lattice with temporal links fixed to 0 (BASELINE.json configs 2 and 5).
# ------------------------------------------------------------------------------------------------
def _staple_sum(a: np.ndarray, mu: int, w_space: float = 1.0, w_time: float = 1.0) -> np.ndarray:
    """sum_k w_k exp(+i c_k) over the 4 plaquettes containing each mu-link, where the plaquette angle
    is (a_link + c_k); w_k = w_space for the two spatial plaquettes, w_time for the two temporal ones.
    a has shape [Ntau][2][L][L] (axes tau, mu, y, x)."""
    ax, ay = a[:, 0], a[:, 1]
    if mu == 0:
        # plaquette at s:      +ax(s) + ay(s+x) - ax(s+y) - ay(s)
        c_up = np.roll(ay, -1, axis=2) - np.roll(ax, -1, axis=1) - ay
        # plaquette at s-y:    ax(s-y) + ay(s-y+x) - ax(s) - ay(s-y)  => angle = -(ax(s) + c), use cos even
        c_dn = -(np.roll(ax, 1, axis=1) + np.roll(np.roll(ay, 1, axis=1), -1, axis=2) - np.roll(ay, 1, axis=1))
        link = ax
    else:
        # plaquette at s:      ax(s) + ay(s+x) - ax(s+y) - ay(s)  => angle = -(ay(s) + c)
        c_up = -(ax + np.roll(ay, -1, axis=2) - np.roll(ax, -1, axis=1))
        # plaquette at s-x:    ax(s-x) + ay(s) - ax(s-x+y) - ay(s-x)
        c_dn = np.roll(ax, 1, axis=2) - np.roll(np.roll(ax, 1, axis=2), -1, axis=1) - np.roll(ay, 1, axis=2)
        link = ay
    # temporal plaquettes: angle = a(tau+1) - a(tau) and a(tau) - a(tau-1)
    c_tp = -np.roll(link, -1, axis=0)
    c_tm = -np.roll(link, 1, axis=0)
    return w_space * (np.exp(1j * c_up) + np.exp(1j * c_dn)) + w_time * (np.exp(1j * c_tp) + np.exp(1j * c_tm))


def heatbath_theta(L: int, Ntau: int, seed: int, beta: float = 1.0, sweeps: int = 10,
                   add_pi_flux: bool = True, beta_time: float | None = None, cold_start: bool = False) -> np.ndarray:
    """Hot start U[-pi,pi) then `sweeps` von-Mises heat-bath sweeps at coupling beta = 1/g^2.

    Each link's conditional density is prop. to exp(beta * Re[e^{i a} * S]) with S = sum_k e^{i c_k},
    i.e. von Mises(mu = -arg S, kappa = beta |S|).  Colour order per sweep: mu=x with parity
    (y+tau) = 0, 1, then mu=y with parity (x+tau) = 0, 1 (links of one colour share no plaquette;
    needs L and Ntau even).  Returns theta = a + A_pi (reading C12) unless add_pi_flux is False.
    """
    assert L % 2 == 0 and Ntau % 2 == 0
    g = rng(seed, STREAM_HEATBATH)
    bt = beta if beta_time is None else beta_time       # separate temporal coupling (paper regime: c_tau = 1/(J dtau^2) = 80, K = 1)
    a = np.zeros((Ntau, 2, L, L)) if cold_start else g.uniform(-np.pi, np.pi, (Ntau, 2, L, L))
    tau = np.arange(Ntau)[:, None, None]
    yy = np.arange(L)[None, :, None]
    xx = np.arange(L)[None, None, :]
    for _ in range(sweeps):
        for mu in (0, 1):
            par = (yy + tau + 0 * xx) % 2 if mu == 0 else (xx + tau + 0 * yy) % 2
            for colour in (0, 1):
                S = _staple_sum(a, mu, beta, bt)
                mask = par == colour
                kappa = np.abs(S[mask])
                centre = -np.angle(S[mask])
                a[:, mu][mask] = g.vonmises(centre, kappa)
    if add_pi_flux:
        a = a + pi_flux_background(L, Ntau)
    return a


def mean_plaquettes(a: np.ndarray):
    """(<cos a_xy>, <cos a_tau-plaquette>) of a link field (diagnostic for the heat bath)."""
    ax, ay = a[:, 0], a[:, 1]
    curl = ax + np.roll(ay, -1, axis=2) - np.roll(ax, -1, axis=1) - ay
    dt = np.roll(a, -1, axis=0) - a
    return float(np.cos(curl).mean()), float(np.cos(dt).mean())


def make_theta(cfg: int) -> np.ndarray:
    c = CONFIGS[cfg]
    if c["theta"] == "uniform":
        return theta_uniform(c["L"], c["Ntau"], c["seed"])
    return heatbath_theta(c["L"], c["Ntau"], c["seed"])


def theta_paper_regime(L: int, Ntau: int, seed: int, J: float = 1.25, K: float = 1.0, dtau: float = 0.1, sweeps: int = 50) -> np.ndarray:
    """A field typical of the paper's own simulations (J = 1.25, K = 1, dtau = 0.1, so the temporal
    coupling is c_tau = 1/(J dtau^2) = 80): heat bath of the pure-gauge part of the compact action from a
    cold start, theta = a + A_pi.  Smooth in tau, which is the regime the banded preconditioner was built for."""
    return heatbath_theta(L, Ntau, seed, beta=K, sweeps=sweeps, beta_time=1.0 / (J * dtau * dtau), cold_start=True)
