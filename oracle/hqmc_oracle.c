/*
 * hqmc_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct fp64 restatement of the pseudofermion hot path of
 * arxiv/paper_2508_16298 (hybrid quantum Monte Carlo for a U(1) gauge field coupled to fermions),
 * written from the paper's text (/root/reference/PAPER.md, cited as PAPER.md:<line>) and the
 * readings C1-C22 of SURVEY.md section 8(c) (restated in DESIGN.md).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares NO code with the CUDA path (paper_2508_16298_b200/csrc) and neither
 * imports the other.  There is no blocking, fusion or reordering beyond what the paper states:
 * every operator is applied factor by factor in the paper's order.  OpenMP is used only to run
 * independent time slices in parallel; all reductions are summed per slice and then over slices in
 * a fixed order, so results do not depend on the thread count.
 *
 * Parity pins (tests/test_oracle_*.py): dense M from a generic matrix exponential + LU; theta=0
 * Fourier closed form; det M = det(1 + prod B) real; adjointness / Hermiticity; gauge covariance;
 * central finite differences of S_F and S_B; leapfrog reversibility and dH ~ eps^2.
 * Unpinned against the paper's own numbers: the preconditioner entries (reading C10 -- the paper's
 * recipe is not reproducible from its text); it is pinned only by its defining properties.
 *
 * Layouts: site s = x + L*y; vector element (tau, s) at tau*Vs + s, complex128;
 * theta[tau][mu][y][x], mu=0: bond s -> s+x, mu=1: bond s -> s+y, periodic in space.
 */
#define _GNU_SOURCE
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

typedef struct {
    int L, Ntau;
    double dtau, t;     /* Trotter step (0.1) and hopping (1) */
    double c_tau, K;    /* boson couplings 1/(J dtau^2) and K  */
    int compact;        /* 1: L_B^c, 0: L_B^nc (Eq.2)         */
    int W;              /* preconditioner half bandwidth (reading C10), 0 = identity      */
    double taps[33];    /* p_0..p_W                                                       */
} orc_params;

static int g_threads = 1;
void orc_set_threads(int n) { g_threads = n > 0 ? n : 1; }
int orc_get_threads(void) { return g_threads; }
int orc_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * Family sweep  e^{a V_fam} v   (Eq.23-26).
 * Families (reading C4): 1 = x-bonds with x even, 2 = x-bonds with x odd,
 *                        3 = y-bonds with y even, 4 = y-bonds with y odd.   L must be even.
 * For each bond i -> j with phase theta:  T_ij = [[0, e^{i theta}], [e^{-i theta}, 0]]  (C3) and
 *   v_i' = cosh(a) v_i + sinh(a) e^{+i theta} v_j,   v_j' = cosh(a) v_j + sinh(a) e^{-i theta} v_i.
 * th points at one slice: th[mu][y][x].
 * ------------------------------------------------------------------------------------------- */
void orc_sweep(int L, const double *th, int fam, double a, cplx *v) {
    const double ch = cosh(a), sh = sinh(a);
    const int mu = (fam <= 2) ? 0 : 1;
    const int par = (fam == 1 || fam == 3) ? 0 : 1;
    for (int y = 0; y < L; ++y)
        for (int x = 0; x < L; ++x) {
            int c = (mu == 0) ? x : y;
            if ((c & 1) != par) continue;
            int i = x + L * y;
            int j = (mu == 0) ? ((x + 1) % L + L * y) : (x + L * ((y + 1) % L));
            cplx ph = cexp(I * th[(mu * L + y) * L + x]);
            cplx vi = v[i], vj = v[j];
            v[i] = ch * vi + sh * ph * vj;
            v[j] = ch * vj + sh * conj(ph) * vi;
        }
}

/* The 8 factors of Eq.22 in the order they hit a vector (rightmost first):
 *   B = e^{V4/2} e^{V3/2} e^{V2/2} e^{V1/2} e^{V1/2} e^{V2/2} e^{V3/2} e^{V4/2},  [V]_ij = dtau t e^{i theta_ij}. */
static const int FACT[8] = {4, 3, 2, 1, 1, 2, 3, 4};

void orc_apply_B(int L, const double *th, double dtau_t, const cplx *in, cplx *out) {
    int Vs = L * L;
    if (out != in) memcpy(out, in, sizeof(cplx) * Vs);
    for (int k = 0; k < 8; ++k) orc_sweep(L, th, FACT[k], 0.5 * dtau_t, out);
}

/* ---------------------------------------------------------------------------------------------
 * M and M^dagger  (Eq.8; reading C1; 0-based slices):
 *   (M v)_t     = v_t - B_{t-1} v_{t-1}   (t >= 1),    (M v)_0        = v_0 + B_{Nt-1} v_{Nt-1}
 *   (M^+ w)_t   = w_t - B_t w_{t+1}       (t < Nt-1),  (M^+ w)_{Nt-1} = w_{Nt-1} + B_{Nt-1} w_0
 * (B is Hermitian: each factor is, and the product is palindromic.)
 * ------------------------------------------------------------------------------------------- */
void orc_apply_M(const orc_params *P, const double *theta, const cplx *in, cplx *out) {
    const int L = P->L, Nt = P->Ntau, Vs = L * L;
    const double a = P->dtau * P->t;
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int t = 0; t < Nt; ++t) {
        int tp = (t + Nt - 1) % Nt;               /* source slice t-1 */
        double sgn = (t == 0) ? +1.0 : -1.0;
        cplx *tmp = (cplx *)malloc(sizeof(cplx) * Vs);
        orc_apply_B(L, theta + (size_t)tp * 2 * Vs, a, in + (size_t)tp * Vs, tmp);
        for (int s = 0; s < Vs; ++s) out[(size_t)t * Vs + s] = in[(size_t)t * Vs + s] + sgn * tmp[s];
        free(tmp);
    }
}

void orc_apply_Mdag(const orc_params *P, const double *theta, const cplx *in, cplx *out) {
    const int L = P->L, Nt = P->Ntau, Vs = L * L;
    const double a = P->dtau * P->t;
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int t = 0; t < Nt; ++t) {
        int tn = (t + 1) % Nt;
        double sgn = (t == Nt - 1) ? +1.0 : -1.0;
        cplx *tmp = (cplx *)malloc(sizeof(cplx) * Vs);
        orc_apply_B(L, theta + (size_t)t * 2 * Vs, a, in + (size_t)tn * Vs, tmp);
        for (int s = 0; s < Vs; ++s) out[(size_t)t * Vs + s] = in[(size_t)t * Vs + s] + sgn * tmp[s];
        free(tmp);
    }
}

/* O = M^+ M; tmp is caller scratch of N elements. */
void orc_apply_MdagM(const orc_params *P, const double *theta, const cplx *in, cplx *out, cplx *tmp) {
    orc_apply_M(P, theta, in, tmp);
    orc_apply_Mdag(P, theta, tmp, out);
}

/* ---------------------------------------------------------------------------------------------
 * Preconditioner (reading C10 -- the paper's recipe cannot be
 * reproduced from its text; parity with the paper's entries is UNPINNED).
 * What the text fixes: theta-independent, built once at pi-flux; banded in tau
 * only, site-diagonal; of the form L^{-1} L^{-+}.
 * Concrete definition (C10): M is lower block-bidiagonal, 1 - M = S B (S = antiperiodic tau-shift),
 * Neumann series M^{-1} ~ sum_k (S B)^k; keep its site-diagonal part at pi-flux, truncated at W:
 *   T = sum_{k=0..W} c_k S^k,  c_k = [B_pi^k]_{00},   P = T^+ T = sum_{m=-W..W} p_|m| S^m,
 *   p_m = sum_k c_k c_{k+m}.
 * pi-flux: theta_x(x,y) = pi * (y mod 2), theta_y = 0.
 * ------------------------------------------------------------------------------------------- */
void orc_precond_taps(int L, double dtau_t, int W, double *c_out /*W+1*/, double *p_out /*W+1*/) {
    int Vs = L * L;
    double *th = (double *)calloc((size_t)2 * Vs, sizeof(double));
    for (int y = 1; y < L; y += 2)
        for (int x = 0; x < L; ++x) th[(0 * L + y) * L + x] = M_PI;
    cplx *v = (cplx *)calloc((size_t)Vs, sizeof(cplx));
    v[0] = 1.0;
    for (int k = 0; k <= W; ++k) {
        c_out[k] = creal(v[0]);
        orc_apply_B(L, th, dtau_t, v, v);
    }
    for (int m = 0; m <= W; ++m) {
        double s = 0.0;
        for (int k = 0; k + m <= W; ++k) s += c_out[k] * c_out[k + m];
        p_out[m] = s;
    }
    free(v);
    free(th);
}

/* z_{t,i} = sum_{m=-W..W} p_|m| s(t,m) r_{t+m,i},  s = -1 when t+m leaves [0,Nt) (antiperiodic). */
void orc_precond(const orc_params *P, const cplx *in, cplx *out) {
    const int Nt = P->Ntau, Vs = P->L * P->L, W = P->W;
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int t = 0; t < Nt; ++t)
        for (int s = 0; s < Vs; ++s) {
            cplx acc = 0.0;
            for (int m = -W; m <= W; ++m) {
                int tt = t + m;
                double sg = 1.0;
                while (tt < 0) { tt += Nt; sg = -sg; }
                while (tt >= Nt) { tt -= Nt; sg = -sg; }
                acc += (P->taps[m < 0 ? -m : m] * sg) * in[(size_t)tt * Vs + s];
            }
            out[(size_t)t * Vs + s] = acc;
        }
}

/* <a, b> = sum conj(a) b : per-slice partial sums, then summed over slices in order. */
cplx orc_dot(int Nt, int Vs, const cplx *a, const cplx *b) {
    cplx *part = (cplx *)malloc(sizeof(cplx) * Nt);
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int t = 0; t < Nt; ++t) {
        cplx s = 0.0;
        for (int i = 0; i < Vs; ++i) s += conj(a[(size_t)t * Vs + i]) * b[(size_t)t * Vs + i];
        part[t] = s;
    }
    cplx tot = 0.0;
    for (int t = 0; t < Nt; ++t) tot += part[t];
    free(part);
    return tot;
}

/* ---------------------------------------------------------------------------------------------
 * Preconditioned CG on  O X = v,  O = M^+ M   (Eq.20).
 * Readings: C8 (d_0 = P r_0, X_0 = 0), C9 (stop when ||r_{n+1}|| / ||v|| <= tol, tested after the
 * r update; tol <= 0 runs exactly max_iter iterations -- the paper's fixed-count mode).
 * Paper's names: zeta = alpha, rho = beta.
 * Returns iterations done; relres_out = recurrence residual ||r|| / ||v|| at exit.
 * ------------------------------------------------------------------------------------------- */
long orc_pcg(const orc_params *P, const double *theta, const cplx *rhs, cplx *x, double tol, long max_iter,
             double *relres_out) {
    const int Nt = P->Ntau, Vs = P->L * P->L;
    const size_t N = (size_t)Nt * Vs;
    cplx *r = (cplx *)malloc(sizeof(cplx) * N), *z = (cplx *)malloc(sizeof(cplx) * N);
    cplx *d = (cplx *)malloc(sizeof(cplx) * N), *Od = (cplx *)malloc(sizeof(cplx) * N);
    cplx *tmp = (cplx *)malloc(sizeof(cplx) * N);
    memset(x, 0, sizeof(cplx) * N);                      /* X_0 = 0           */
    memcpy(r, rhs, sizeof(cplx) * N);                    /* r_0 = v - O X_0   */
    if (P->W > 0) orc_precond(P, r, z); else memcpy(z, r, sizeof(cplx) * N);
    memcpy(d, z, sizeof(cplx) * N);                      /* d_0 = P r_0 (C8)  */
    double bb = creal(orc_dot(Nt, Vs, rhs, rhs));
    double rz = creal(orc_dot(Nt, Vs, r, z));
    double rr = bb;
    long it = 0;
    if (bb == 0.0) { if (relres_out) *relres_out = 0.0; goto done; }
    while (it < max_iter) {
        orc_apply_MdagM(P, theta, d, Od, tmp);
        double dOd = creal(orc_dot(Nt, Vs, d, Od));
        double alpha = rz / dOd;                         /* zeta_n            */
#pragma omp parallel for num_threads(g_threads) schedule(static)
        for (size_t i = 0; i < N; ++i) { x[i] += alpha * d[i]; r[i] -= alpha * Od[i]; }
        rr = creal(orc_dot(Nt, Vs, r, r));
        ++it;
        if (tol > 0.0 && sqrt(rr / bb) <= tol) break;
        if (P->W > 0) orc_precond(P, r, z); else memcpy(z, r, sizeof(cplx) * N);
        double rz_new = creal(orc_dot(Nt, Vs, r, z));
        double beta = rz_new / rz;                       /* rho_n             */
#pragma omp parallel for num_threads(g_threads) schedule(static)
        for (size_t i = 0; i < N; ++i) d[i] = z[i] + beta * d[i];
        rz = rz_new;
    }
    if (relres_out) *relres_out = sqrt(rr / bb);
done:
    free(r); free(z); free(d); free(Od); free(tmp);
    return it;
}

/* ---------------------------------------------------------------------------------------------
 * Fermionic force  dS_F/dtheta,  S_F = phi^+ (M^+ M)^{-1} phi   (SI; reading C11).
 * With X = (M^+M)^{-1} phi, Y = M X:  dS_F = -X^+ d(M^+M) X = -2 Re[ Y^+ (dM) X ], and dM has
 * -dB_t in block (t+1, t), +dB_{Nt-1} in block (0, Nt-1) (Eq.8), so with sigma_t = +1 (t < Nt-1),
 * -1 (t = Nt-1):
 *      dS_F/dtheta_{b,t} = 2 sigma_t Re[ Y_{t+1}^+ (dB_t/dtheta_b) X_t ].
 * dB/dtheta_b by the product rule over the 8 factors (Eq.S5): for factor k whose
 * family holds bond b = (i -> j),  d e^{aT}/dtheta = sinh(a) [[0, i e^{i th}], [-i e^{-i th}, 0]].
 * R_k = (first k factors) X_t are stored; L_k = (factors after k)^+ Y_{t+1} is walked backwards
 * (each factor is Hermitian).
 * ------------------------------------------------------------------------------------------- */
void orc_force_fermion(const orc_params *P, const double *theta, const cplx *X, double *dSF) {
    const int L = P->L, Nt = P->Ntau, Vs = L * L;
    const double a = 0.5 * P->dtau * P->t, sh = sinh(a);
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int t = 0; t < Nt; ++t) {
        const double *th = theta + (size_t)t * 2 * Vs;
        double *g = dSF + (size_t)t * 2 * Vs;
        const int tn = (t + 1) % Nt;
        const double sigma = (t == Nt - 1) ? -1.0 : +1.0;
        cplx *R = (cplx *)malloc(sizeof(cplx) * Vs * 9);   /* R_0 .. R_8 */
        cplx *Lv = (cplx *)malloc(sizeof(cplx) * Vs);
        memcpy(R, X + (size_t)t * Vs, sizeof(cplx) * Vs);
        for (int k = 0; k < 8; ++k) {
            memcpy(R + (size_t)(k + 1) * Vs, R + (size_t)k * Vs, sizeof(cplx) * Vs);
            orc_sweep(L, th, FACT[k], a, R + (size_t)(k + 1) * Vs);
        }
        /* Y_{t+1} = X_{t+1} - sigma_t B_t X_t */
        for (int s = 0; s < Vs; ++s) Lv[s] = X[(size_t)tn * Vs + s] - sigma * R[(size_t)8 * Vs + s];
        for (int b = 0; b < 2 * Vs; ++b) g[b] = 0.0;
        for (int k = 7; k >= 0; --k) {
            const cplx *Rk = R + (size_t)k * Vs;            /* state before factor k */
            const int fam = FACT[k], mu = (fam <= 2) ? 0 : 1, par = (fam == 1 || fam == 3) ? 0 : 1;
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    int c = (mu == 0) ? x : y;
                    if ((c & 1) != par) continue;
                    int i = x + L * y;
                    int j = (mu == 0) ? ((x + 1) % L + L * y) : (x + L * ((y + 1) % L));
                    int b = (mu * L + y) * L + x;
                    cplx ph = cexp(I * th[b]);
                    cplx val = conj(Lv[i]) * (I * sh * ph) * Rk[j] + conj(Lv[j]) * (-I * sh * conj(ph)) * Rk[i];
                    g[b] += 2.0 * sigma * creal(val);
                }
            orc_sweep(L, th, fam, a, Lv);                    /* L_{k} = E_k^+ L_{k+1} */
        }
        free(R);
        free(Lv);
    }
}

/* ---------------------------------------------------------------------------------------------
 * Bosonic action and force (readings C12, C14, C15).
 *   compact:      S_B = c_tau sum_{b,t} [1 - cos(th_{b,t+1} - th_{b,t})] + K sum_{plaq,t} cos(curl th_t)
 *   non-compact:  S_B = c_tau sum_{b,t} (th_{b,t+1} - th_{b,t})^2        + K sum_{plaq,t} cos(curl th_t)
 *   curl th (s) = th_x(s) + th_y(s+x) - th_x(s+y) - th_y(s);  theta periodic in tau.
 * ------------------------------------------------------------------------------------------- */
static double curl_at(int L, const double *th, int x, int y) {
    int xp = (x + 1) % L, yp = (y + 1) % L;
    return th[(0 * L + y) * L + x] + th[(1 * L + y) * L + xp] - th[(0 * L + yp) * L + x] - th[(1 * L + y) * L + x];
}

double orc_action_boson(const orc_params *P, const double *theta) {
    const int L = P->L, Nt = P->Ntau, Vs = L * L;
    double *part = (double *)malloc(sizeof(double) * Nt);
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int t = 0; t < Nt; ++t) {
        const double *th = theta + (size_t)t * 2 * Vs, *thn = theta + (size_t)((t + 1) % Nt) * 2 * Vs;
        double s = 0.0;
        for (int b = 0; b < 2 * Vs; ++b) {
            double d = thn[b] - th[b];
            s += P->c_tau * (P->compact ? (1.0 - cos(d)) : d * d);
        }
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) s += P->K * cos(curl_at(L, th, x, y));
        part[t] = s;
    }
    double tot = 0.0;
    for (int t = 0; t < Nt; ++t) tot += part[t];
    free(part);
    return tot;
}

void orc_force_boson(const orc_params *P, const double *theta, double *dSB) {
    const int L = P->L, Nt = P->Ntau, Vs = L * L;
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int t = 0; t < Nt; ++t) {
        const double *th = theta + (size_t)t * 2 * Vs;
        const double *thn = theta + (size_t)((t + 1) % Nt) * 2 * Vs;
        const double *thp = theta + (size_t)((t + Nt - 1) % Nt) * 2 * Vs;
        double *g = dSB + (size_t)t * 2 * Vs;
        for (int b = 0; b < 2 * Vs; ++b) {
            double dm = th[b] - thp[b], dp = thn[b] - th[b];
            g[b] = P->compact ? P->c_tau * (sin(dm) - sin(dp)) : 2.0 * P->c_tau * (dm - dp);
        }
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                /* d/dcurl of K cos(curl(s)) = -K sin(curl(s)); curl(s) holds +th_x(s), +th_y(s+x), -th_x(s+y), -th_y(s) */
                double f = -P->K * sin(curl_at(L, th, x, y));
                int xp = (x + 1) % L, yp = (y + 1) % L;
                g[(0 * L + y) * L + x] += f;
                g[(1 * L + y) * L + xp] += f;
                g[(0 * L + yp) * L + x] -= f;
                g[(1 * L + y) * L + x] -= f;
            }
    }
}

double orc_sum_p2(const orc_params *P, const double *p) {
    const int Nt = P->Ntau, nb = 2 * P->L * P->L;
    double tot = 0.0;
    for (int t = 0; t < Nt; ++t) {
        double s = 0.0;
        for (int b = 0; b < nb; ++b) s += p[(size_t)t * nb + b] * p[(size_t)t * nb + b];
        tot += s;
    }
    return tot;
}

/* ---------------------------------------------------------------------------------------------
 * Leapfrog trajectory (Eq.16) with H = S_B + sum p^2 + phi^+ (M^+M)^{-1} phi
 * (Eq.12; reading C7: theta_dot = 2p):
 *     p += F dt/2;  theta += 2 p dt;  p += F dt/2,   F = -dS_B/dtheta - dS_F/dtheta.
 * nsteps steps = nsteps+1 CG solves.  theta, p updated in place.  H0/H1 at start/end.
 * parts_out (may be NULL): [S_B0, sum p0^2, S_F0, S_B1, sum p1^2, S_F1].
 * ------------------------------------------------------------------------------------------- */
long orc_trajectory(const orc_params *P, double *theta, double *p, const cplx *phi, int nsteps, double eps,
                    double cg_tol, long cg_max_iter, double *H0, double *H1, double *parts_out) {
    const int Nt = P->Ntau, Vs = P->L * P->L;
    const size_t N = (size_t)Nt * Vs, NB = 2 * N;
    cplx *X = (cplx *)malloc(sizeof(cplx) * N);
    double *gF = (double *)malloc(sizeof(double) * NB), *gB = (double *)malloc(sizeof(double) * NB);
    long iters = 0;
    iters += orc_pcg(P, theta, phi, X, cg_tol, cg_max_iter, NULL);
    double SB = orc_action_boson(P, theta), pp = orc_sum_p2(P, p), SF = creal(orc_dot(Nt, Vs, phi, X));
    *H0 = SB + pp + SF;
    if (parts_out) { parts_out[0] = SB; parts_out[1] = pp; parts_out[2] = SF; }
    orc_force_fermion(P, theta, X, gF);
    orc_force_boson(P, theta, gB);
    for (int n = 0; n < nsteps; ++n) {
        for (size_t b = 0; b < NB; ++b) p[b] += -(gB[b] + gF[b]) * (0.5 * eps);
        for (size_t b = 0; b < NB; ++b) theta[b] += 2.0 * p[b] * eps;
        iters += orc_pcg(P, theta, phi, X, cg_tol, cg_max_iter, NULL);
        orc_force_fermion(P, theta, X, gF);
        orc_force_boson(P, theta, gB);
        for (size_t b = 0; b < NB; ++b) p[b] += -(gB[b] + gF[b]) * (0.5 * eps);
    }
    SB = orc_action_boson(P, theta); pp = orc_sum_p2(P, p); SF = creal(orc_dot(Nt, Vs, phi, X));
    *H1 = SB + pp + SF;
    if (parts_out) { parts_out[3] = SB; parts_out[4] = pp; parts_out[5] = SF; }
    free(X); free(gF); free(gB);
    return iters;
}

/* ---------------------------------------------------------------------------------------------
 * One HQMC update, steps (i)-(iv) of PAPER.md:185-201 (NEXT-1 of SURVEY.md 8f).  The random numbers are INPUTS
 * (eta complex Gaussian, p Gaussian, u uniform in [0,1)), so that oracle and GPU consume identical draws:
 *   (i)   phi = M^+(theta_0) eta                                   (reading C6)
 *   (ii)  leapfrog trajectory (theta_0, p_0) -> (theta_t, p_t)      (Eq.13-16)
 *   (iii) accept with probability r = min(1, exp(H_0 - H_t))        (Eq.15): accepted iff u < r
 *   (iv)  on rejection theta stays theta_0 (p is discarded either way: it is redrawn next update)
 * theta, p updated in place (p holds p_t afterwards, whatever the decision).  Returns 1 if accepted, else 0.
 * ------------------------------------------------------------------------------------------- */
int orc_hqmc_step(const orc_params *P, double *theta, double *p, const cplx *eta, double u, int nsteps, double eps,
                  double cg_tol, long cg_max_iter, double *H0, double *H1, long *iters_out) {
    const size_t N = (size_t)P->Ntau * P->L * P->L, NB = 2 * N;
    cplx *phi = (cplx *)malloc(sizeof(cplx) * N);
    double *theta0 = (double *)malloc(sizeof(double) * NB);
    memcpy(theta0, theta, sizeof(double) * NB);
    orc_apply_Mdag(P, theta, eta, phi);
    long it = orc_trajectory(P, theta, p, phi, nsteps, eps, cg_tol, cg_max_iter, H0, H1, NULL);
    if (iters_out) *iters_out = it;
    double r = exp(*H0 - *H1);
    if (r > 1.0) r = 1.0;
    int accepted = (u < r) ? 1 : 0;
    if (!accepted) memcpy(theta, theta0, sizeof(double) * NB);
    free(phi); free(theta0);
    return accepted;
}

/* ---------------------------------------------------------------------------------------------
 * Random numbers of the HQMC update (PAPER.md:185 step (i): "sample p and R from Gaussian distributions"
 * step (iii): uniform u; reading C6: weights e^{-R^+R} and e^{-sum p^2}, so Re R, Im R, p ~ N(0, 1/2), E|R|^2 = 1).
 * The paper names no generator.  Both sides implement the SAME counter-based one, so that a sweep is reproducible from
 * (seed, update index) alone: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11: ten rounds of
 *     (c0, c1, c2, c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0)),  then (k0, k1) += (W0, W1)
 * with M0 = 0xD2511F53, M1 = 0xCD9E8D57, W0 = 0x9E3779B9, W1 = 0xBB67AE85), counter = (index lo, index hi, stream, update),
 * key = (seed lo, seed hi); streams: 0 = R (eta), 1 = p, 2 = Metropolis u.  From the four output words x0..x3:
 *     u1 = ((x0 >> 5) 2^26 + (x1 >> 6)) / 2^53,   u2 = ((x2 >> 5) 2^26 + (x3 >> 6)) / 2^53      (both in [0, 1))
 * and by Box-Muller the pair  sqrt(-ln(1 - u1)) (cos 2 pi u2, sin 2 pi u2): two independent N(0, 1/2).
 * Element i of stream 0 is the complex number R_i; element i of stream 1 is the pair (p_{2i}, p_{2i+1}).
 * Pins (tests/test_oracle_rng.py): the published known-answer vectors of Philox4x32-10; moments and a Kolmogorov-Smirnov
 * bound of the uniforms and Gaussians; E|R|^2 = 1, Var p = 1/2.
 * ------------------------------------------------------------------------------------------- */
#include <stdint.h>
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
static void rng_words(uint64_t seed, uint32_t update, uint32_t stream, uint64_t i, uint32_t x[4]) {
    const uint32_t ctr[4] = {(uint32_t)i, (uint32_t)(i >> 32), stream, update}, key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    orc_philox4x32_10(ctr, key, x);
}
/* raw words of elements 0..n-1: out[4 n] */
void orc_rng_raw(uint64_t seed, uint32_t update, uint32_t stream, long n, uint32_t *out) {
    for (long i = 0; i < n; ++i) rng_words(seed, update, stream, (uint64_t)i, out + 4 * i);
}
static double u53(uint32_t a, uint32_t b) { return ((double)(a >> 5) * 67108864.0 + (double)(b >> 6)) * (1.0 / 9007199254740992.0); }
/* the two uniforms of elements 0..n-1: out[2 n] */
void orc_rng_uniform(uint64_t seed, uint32_t update, uint32_t stream, long n, double *out) {
    for (long i = 0; i < n; ++i) {
        uint32_t x[4];
        rng_words(seed, update, stream, (uint64_t)i, x);
        out[2 * i] = u53(x[0], x[1]); out[2 * i + 1] = u53(x[2], x[3]);
    }
}
/* the Gaussian pair (variance 1/2 each) of elements 0..n-1: out[2 n] */
void orc_rng_gauss(uint64_t seed, uint32_t update, uint32_t stream, long n, double *out) {
    for (long i = 0; i < n; ++i) {
        uint32_t x[4];
        rng_words(seed, update, stream, (uint64_t)i, x);
        const double u1 = u53(x[0], x[1]), u2 = u53(x[2], x[3]);
        const double r = sqrt(-log(1.0 - u1)), a = 6.283185307179586476925286766559 * u2;
        out[2 * i] = r * cos(a); out[2 * i + 1] = r * sin(a);
    }
}
/* `n_updates` HQMC updates (steps (i)-(iv)) from update index `first`: update k draws R from stream 0,
 * p from stream 1 and u = first uniform of element 0 of stream 2, all at counter word `update` = k.  Per-update outputs. */
void orc_hqmc_sweep(const orc_params *P, double *theta, uint64_t seed, uint32_t first, int n_updates, int nsteps, double eps,
                    double cg_tol, long cg_max_iter, double *H0, double *H1, int *accepted, long *iters) {
    const size_t N = (size_t)P->Ntau * P->L * P->L;
    cplx *eta = (cplx *)malloc(sizeof(cplx) * N);
    double *p = (double *)malloc(sizeof(double) * 2 * N), u2[2];
    for (int k = 0; k < n_updates; ++k) {
        const uint32_t upd = first + (uint32_t)k;
        orc_rng_gauss(seed, upd, 0, (long)N, (double *)eta);
        orc_rng_gauss(seed, upd, 1, (long)N, p);
        orc_rng_uniform(seed, upd, 2, 1, u2);
        accepted[k] = orc_hqmc_step(P, theta, p, eta, u2[0], nsteps, eps, cg_tol, cg_max_iter, H0 + k, H1 + k, iters + k);
    }
    free(eta); free(p);
}
