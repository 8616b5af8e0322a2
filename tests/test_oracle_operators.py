"""Pins of the CPU oracle's operators (sweep, B, M, M^+, M^+M, P) against things other than itself:
generic dense matrix exponentials, determinant identities, the theta=0 Fourier closed form,
adjointness / Hermiticity, gauge covariance.  CPU only."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2508_16298_b200 import inputs
from tests import dense_ref as dr

DTAU = 0.1


def _rand_vec(n, seed):
    return inputs.complex_gaussian((n,), seed, inputs.STREAM_VEC)


@pytest.mark.parametrize("L", [4, 6])
@pytest.mark.parametrize("fam", [1, 2, 3, 4])
def test_sweep_equals_generic_expm(L, fam):
    """Eq.23-26: the cosh/sinh 2x2 form equals expm(a * V_fam)."""
    th = inputs.theta_uniform(L, 2, 11)[0]
    o = orc.Oracle(L, 2)
    v = _rand_vec(L * L, 5)
    for a in (0.05, 0.1, -0.05):
        import scipy.linalg as sla
        ref = sla.expm(a * dr.family_matrix(L, th, fam)) @ v
        got = o.sweep(th, fam, a, v)
        assert np.abs(got - ref).max() < 1e-14
    # within a family all terms commute: every site appears in exactly one bond
    sites = [s for b in dr.family_bonds(L, fam) for s in b[:2]]
    assert sorted(sites) == list(range(L * L))


@pytest.mark.parametrize("L", [4, 6])
def test_B_dense_and_invariants(L):
    th = inputs.theta_uniform(L, 2, 12)[1]
    o = orc.Oracle(L, 2)
    Bd = dr.dense_B(L, th, DTAU)
    Bo = np.stack([o.apply_B(th, e) for e in np.eye(L * L, dtype=np.complex128)], axis=1)
    assert np.abs(Bo - Bd).max() < 1e-14
    assert np.abs(Bo - Bo.conj().T).max() < 1e-15          # Hermitian
    assert np.linalg.eigvalsh(Bo).min() > 0                # positive
    assert abs(np.linalg.det(Bo) - 1.0) < 1e-12            # each 2x2 block has cosh^2 - sinh^2 = 1
    # a transposed operand / wrong bond orientation (C3) would break this at generic theta:
    assert np.abs(Bo - Bo.T).max() > 1e-3


@pytest.mark.parametrize("L,Nt,seed", [(4, 8, 0), (6, 10, 3)])
def test_M_Mdag_dense(L, Nt, seed):
    theta = inputs.theta_uniform(L, Nt, seed)
    o = orc.Oracle(L, Nt)
    Md, Bs = dr.dense_M(L, Nt, theta, DTAU)
    v = _rand_vec(o.N, seed + 1)
    u = _rand_vec(o.N, seed + 2)
    scale = np.abs(Md @ v).max()
    assert np.abs(o.apply_M(theta, v) - Md @ v).max() < 1e-13 * scale
    assert np.abs(o.apply_Mdag(theta, v) - Md.conj().T @ v).max() < 1e-13 * scale
    assert np.abs(o.apply_MdagM(theta, v) - Md.conj().T @ (Md @ v)).max() < 1e-13 * scale
    # adjointness <u, M v> = <M^+ u, v>
    lhs = np.vdot(u, o.apply_M(theta, v))
    rhs = np.vdot(o.apply_Mdag(theta, u), v)
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    # det M = det(1 + prod_t B_t), real (Eq.7, 157)
    prod = np.eye(L * L, dtype=np.complex128)
    for B in Bs:
        prod = B @ prod
    d1 = np.linalg.det(Md)
    d2 = np.linalg.det(np.eye(L * L) + prod)
    assert abs(d1 - d2) < 1e-9 * abs(d1)
    assert abs(d1.imag) < 1e-9 * abs(d1)


def test_config1_worked_values():
    """SURVEY.md section 8(c) quotes survey-probe values for config 1 'to be reproduced, not trusted':
    det M = 99808.83034061, sigma_max = 2.2022003409, sigma_min = 0.2611748716, cond(M^+M) = 71.0969338.
    Here they are reproduced from the dense construction AND from the oracle applied to unit vectors."""
    L, Nt = 4, 8
    theta = inputs.make_theta(1)
    o = orc.Oracle(L, Nt)
    Mo = np.stack([o.apply_M(theta, e) for e in np.eye(o.N, dtype=np.complex128)], axis=1)
    Md, _ = dr.dense_M(L, Nt, theta, DTAU)
    assert np.abs(Mo - Md).max() < 1e-14
    sv = np.linalg.svd(Mo, compute_uv=False)
    assert abs(np.linalg.det(Mo).real - 99808.83034061) < 1e-5
    assert abs(sv.max() - 2.2022003409) < 1e-9
    assert abs(sv.min() - 0.2611748716) < 1e-9
    assert abs((sv.max() / sv.min()) ** 2 - 71.0969338) < 1e-6


@pytest.mark.parametrize("L,Nt", [(4, 8), (8, 8)])
def test_theta0_fourier_closed_form(L, Nt):
    """At theta=0 x- and y-sweeps commute, B = Bx (x) By; on the 2-site unit cell
    E2(a/2) E1(a) E2(a/2) has eigenvalues e^{+-lambda(k)}, cosh(lambda) = cosh^2(dtau) + sinh^2(dtau) cos(2k),
    k = 2 pi m / L, m = 0..L/2-1; spec(M^+M) = {1 + b^2 - 2 b cos(w_n)}, w_n = (2n+1) pi / Nt;
    log det M = sum_b log(1 + b^Nt)."""
    theta = np.zeros((Nt, 2, L, L))
    o = orc.Oracle(L, Nt)
    ks = 2 * np.pi * np.arange(L // 2) / L
    lam = np.arccosh(np.maximum(1.0, np.cosh(DTAU) ** 2 + np.sinh(DTAU) ** 2 * np.cos(2 * ks)))
    b = np.array([np.exp(sx * lx + sy * ly) for lx in lam for ly in lam for sx in (1, -1) for sy in (1, -1)])
    assert b.size == L * L
    w = (2 * np.arange(Nt) + 1) * np.pi / Nt
    spec = np.sort((1 + b[:, None] ** 2 - 2 * b[:, None] * np.cos(w[None, :])).ravel())
    Oo = np.stack([o.apply_MdagM(theta, e) for e in np.eye(o.N, dtype=np.complex128)], axis=1)
    ev = np.linalg.eigvalsh(Oo)
    assert np.abs(ev - spec).max() < 1e-12
    Mo = np.stack([o.apply_M(theta, e) for e in np.eye(o.N, dtype=np.complex128)], axis=1)
    sign, logdet = np.linalg.slogdet(Mo)
    assert abs(logdet - np.log1p(b ** Nt).sum()) < 1e-10
    if (L, Nt) == (4, 8):   # survey's worked values
        assert abs(logdet - 15.309995676791) < 1e-9
        assert abs(ev.min() - 0.152240934977) < 1e-10 and abs(ev.max() - 5.982073536984) < 1e-10
    if (L, Nt) == (8, 8):
        assert abs(logdet - 61.428051211853) < 1e-9 and abs(ev.min() - 0.146820470727) < 1e-10


def test_gauge_covariance_of_M():
    """theta_ij -> theta_ij + alpha_i - alpha_j  <=>  M(theta') G = G M(theta), G = diag(e^{i alpha_i}) (C3)."""
    L, Nt = 6, 10
    theta = inputs.theta_uniform(L, Nt, 21)
    alpha = inputs.gauge_alpha(L, 21)
    thp = inputs.gauge_transform_theta(theta, alpha)
    o = orc.Oracle(L, Nt)
    G = np.tile(np.exp(1j * alpha).ravel(), Nt)
    v = _rand_vec(o.N, 22)
    assert np.abs(o.apply_M(thp, G * v) - G * o.apply_M(theta, v)).max() < 1e-13
    assert np.abs(o.apply_MdagM(thp, G * v) - G * o.apply_MdagM(theta, v)).max() < 1e-13


def test_MdagM_hermitian_psd():
    L, Nt = 6, 10
    theta = inputs.theta_uniform(L, Nt, 31)
    o = orc.Oracle(L, Nt)
    u, v = _rand_vec(o.N, 32), _rand_vec(o.N, 33)
    a = np.vdot(u, o.apply_MdagM(theta, v))
    b = np.conj(np.vdot(v, o.apply_MdagM(theta, u)))
    assert abs(a - b) < 1e-12 * abs(a)
    q = np.vdot(v, o.apply_MdagM(theta, v))
    assert q.real > 0 and abs(q.imag) < 1e-12 * q.real


# ---------------------------------------------------------------------------------- preconditioner
def test_precond_taps_independent_route():
    """c_k = [B_pi^k]_00 from a dense generic-expm B at pi-flux; p_m = sum_k c_k c_{k+m} (C10).
    Also the size-independent bulk values SURVEY.md quotes (L >= 16)."""
    L, W = 16, 6
    th = inputs.pi_flux_background(L, 1)[0]
    Bd = dr.dense_B(L, th, DTAU)
    c_ref = np.array([np.linalg.matrix_power(Bd, k)[0, 0].real for k in range(W + 1)])
    p_ref = np.array([sum(c_ref[k] * c_ref[k + m] for k in range(W + 1 - m)) for m in range(W + 1)])
    c, p = orc.precond_taps(L, DTAU, 1.0, W)
    assert np.abs(c - c_ref).max() < 1e-13 and np.abs(p - p_ref).max() < 1e-12
    # all sites equal by symmetry
    assert np.abs(np.diag(np.linalg.matrix_power(Bd, 3)) - c_ref[3]).max() < 1e-13
    quoted_c = [1, 1.020167424, 1.081688550, 1.187677663, 1.343521191, 1.557184209, 1.839665534]
    quoted_p = [12.235611056, 9.960846388, 8.067652634, 6.427612208, 4.922054940, 3.433951059, 1.839665534]
    assert np.abs(c - quoted_c).max() < 2e-9 and np.abs(p - quoted_p).max() < 2e-8


@pytest.mark.parametrize("L,Nt,W", [(4, 8, 6), (4, 16, 6), (6, 10, 3)])
def test_precond_is_TdagT(L, Nt, W):
    """P = T^+ T with T = sum_k c_k S^k, S the antiperiodic tau-shift: Hermitian, positive definite,
    site-diagonal (commutes with gauge transformations)."""
    o = orc.Oracle(L, Nt, W=W)
    c, p = orc.precond_taps(L, DTAU, 1.0, W)
    S = np.zeros((Nt, Nt))
    for t in range(1, Nt):
        S[t, t - 1] = 1.0
    S[0, Nt - 1] = -1.0
    T = sum(c[k] * np.linalg.matrix_power(S, k) for k in range(W + 1))
    Pd = np.kron(T.T @ T, np.eye(L * L))
    v = _rand_vec(o.N, 41)
    assert np.abs(o.precond(v) - Pd @ v).max() < 1e-12 * np.abs(Pd @ v).max()
    ev = np.linalg.eigvalsh(T.T @ T)
    assert ev.min() > 0
    G = np.tile(np.exp(1j * inputs.gauge_alpha(L, 42)).ravel(), Nt)
    assert np.abs(o.precond(G * v) - G * o.precond(v)).max() < 1e-13 * np.abs(Pd @ v).max()
