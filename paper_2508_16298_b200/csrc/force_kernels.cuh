// force_kernels.cuh -- fermionic force (PAPER.md:455-477 SI, reading C11), bosonic action / force
// (readings C12, C14, C15) and the fused momentum kick (Eq.16).
#pragma once
#include "kernels.cuh"

namespace hqmc {

// curl theta (s) = th_x(s) + th_y(s+x) - th_x(s+y) - th_y(s)  on slice th[mu][y][x]
__device__ __forceinline__ double curl_at(const double *__restrict__ th, int L, int Vs, int x, int y) {
    int xp = (x + 1 == L) ? 0 : x + 1, yp = (y + 1 == L) ? 0 : y + 1;
    return th[y * L + x] + th[Vs + y * L + xp] - th[yp * L + x] - th[Vs + y * L + x];
}

// dS_B/dtheta for bond (t, r) with r = mu*Vs + y*L + x the offset inside the slice.
__device__ __forceinline__ double dSB_bond(const double *__restrict__ theta, const Geo &g, int t, int r, double c_tau,
                                           double K, int compact) {
    const int L = g.L, Vs = g.Vs, Nt = g.Nt;
    const int mu = r / Vs, s = r - mu * Vs, y = s / L, x = s - y * L;
    const double *th = theta + (size_t)t * 2 * Vs;
    const double *thn = theta + (size_t)((t + 1 == Nt) ? 0 : t + 1) * 2 * Vs;
    const double *thp = theta + (size_t)((t == 0) ? Nt - 1 : t - 1) * 2 * Vs;
    double dm = th[r] - thp[r], dp = thn[r] - th[r];
    double gb = compact ? c_tau * (sin(dm) - sin(dp)) : 2.0 * c_tau * (dm - dp);
    // the two plaquettes sharing the bond: d/dtheta K cos(curl) = -K sin(curl) * (d curl / d theta)
    if (mu == 0) {
        int ym = (y == 0) ? L - 1 : y - 1;
        gb += -K * sin(curl_at(th, L, Vs, x, y)) + K * sin(curl_at(th, L, Vs, x, ym));
    } else {
        int xm = (x == 0) ? L - 1 : x - 1;
        gb += K * sin(curl_at(th, L, Vs, x, y)) - K * sin(curl_at(th, L, Vs, xm, y));
    }
    return gb;
}

__global__ void k_force_boson(Geo g, const double *__restrict__ theta, double *__restrict__ out, double c_tau, double K,
                              int compact) {
    size_t n = (size_t)2 * g.Vs * g.Nt;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        int t = (int)(i / (size_t)(2 * g.Vs));
        int r = (int)(i - (size_t)t * 2 * g.Vs);
        out[i] = dSB_bond(theta, g, t, r, c_tau, K, compact);
    }
}

// S_B partial sums: one term per bond (temporal) plus one per site (plaquette).
__global__ void k_action_boson(Geo g, const double *__restrict__ theta, double c_tau, double K, int compact,
                               double *__restrict__ part) {
    __shared__ double red[32];
    size_t n = (size_t)2 * g.Vs * g.Nt;
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        int t = (int)(i / (size_t)(2 * g.Vs));
        int r = (int)(i - (size_t)t * 2 * g.Vs);
        int tn = (t + 1 == g.Nt) ? 0 : t + 1;
        double d = theta[(size_t)tn * 2 * g.Vs + r] - theta[i];
        acc += c_tau * (compact ? (1.0 - cos(d)) : d * d);
        if (r < g.Vs) {
            int y = r / g.L, x = r - y * g.L;
            acc += K * cos(curl_at(theta + (size_t)t * 2 * g.Vs, g.L, g.Vs, x, y));
        }
    }
    double s = block_sum(acc, red);
    if (threadIdx.x == 0) part[blockIdx.x] = s;
}

// inverse of one normalised factor: (1 + T(P))^{-1} = (1 - T(P)) / (1 - |P|^2); |P|^2 = tanh^2(a) is a constant of the
// factor's family, so s = 1 / (1 - tanh^2 a) = cosh^2 a comes in as a number (no division per bond)
template <typename T2, typename TS> __device__ __forceinline__ void unrot(T2 &vi, T2 &vj, const T2 P, const TS s) {
    T2 m; m.x = -P.x; m.y = -P.y;
    rot(vi, vj, m);
    vi.x *= s; vi.y *= s; vj.x *= s; vj.y *= s;
}
// Re[ conj(L_i) (i P) R_j + conj(L_j) (-i conj(P)) R_i ]
template <typename T2> __device__ __forceinline__ double bond_term(const T2 Li, const T2 Lj, const T2 Ri, const T2 Rj, const T2 P) {
    double Ax = (double)P.x * Rj.x - (double)P.y * Rj.y, Ay = (double)P.x * Rj.y + (double)P.y * Rj.x;   // P R_j
    double Bx = (double)P.x * Ri.x + (double)P.y * Ri.y, By = (double)P.x * Ri.y - (double)P.y * Ri.x;   // conj(P) R_i
    return -((double)Li.x * Ay - (double)Li.y * Ax) + ((double)Lj.x * By - (double)Lj.y * Bx);
}
// one reverse step for the y-pairs / x-pairs of a block: R <- E^{-1} R, accumulate, Lv <- E Lv
template <typename T2, typename TS> __device__ __forceinline__ void rev_y(T2 (&R)[4], T2 (&Lv)[4], const T2 (&P)[2], double (&acc)[2], const TS s) {
    unrot(R[0], R[2], P[0], s); unrot(R[1], R[3], P[1], s);
    acc[0] += bond_term(Lv[0], Lv[2], R[0], R[2], P[0]);
    acc[1] += bond_term(Lv[1], Lv[3], R[1], R[3], P[1]);
    rot(Lv[0], Lv[2], P[0]); rot(Lv[1], Lv[3], P[1]);
}
template <typename T2, typename TS> __device__ __forceinline__ void rev_x(T2 (&R)[4], T2 (&Lv)[4], const T2 (&P)[2], double (&acc)[2], const TS s) {
    unrot(R[0], R[1], P[0], s); unrot(R[2], R[3], P[1], s);
    acc[0] += bond_term(Lv[0], Lv[1], R[0], R[1], P[0]);
    acc[1] += bond_term(Lv[2], Lv[3], R[2], R[3], P[1]);
    rot(Lv[0], Lv[1], P[0]); rot(Lv[2], Lv[3], P[1]);
}

// sin(curl theta_t) for every site of slice t from the link-phase table (all threads of the CTA; publish with a barrier):
// Im(U_x(s) U_y(s+x) conj(U_x(s+y)) conj(U_y(s))) / (|U_x|^2 |U_y|^2), |U| = tanh(a) of the bond's family.
template <typename T2>
__device__ __forceinline__ void force_splaq(const Geo &g, const T2 *__restrict__ pht, double *__restrict__ Splaq, double i_half, double i_full) {
    for (int s = threadIdx.x; s < g.Vs; s += blockDim.x) {
        const int y = s / g.L, x = s - y * g.L, xp = (x + 1 == g.L) ? 0 : x + 1, yp = (y + 1 == g.L) ? 0 : y + 1;
        const T2 ux = pht[s], uy1 = pht[g.Vs + y * g.L + xp], ux1 = pht[yp * g.L + x], uy = pht[g.Vs + s];
        const double ax = (double)ux.x * uy1.x - (double)ux.y * uy1.y, ay = (double)ux.x * uy1.y + (double)ux.y * uy1.x;     // U_x(s) U_y(s+x)
        const double bx = (double)ux1.x * uy.x - (double)ux1.y * uy.y, by = (double)ux1.x * uy.y + (double)ux1.y * uy.x;     // U_x(s+y) U_y(s)
        Splaq[s] = (ay * bx - ax * by) * ((x & 1) ? i_half : i_full) * i_half;
    }
}

// The write of one block's eight bonds (two per family: 4, 3, 2, 1): dS_F/dtheta = f val, or with FUSE_P the kick
// p += -(dS_B + dS_F) half_eps (nkick times).  Pt: the block's link phases in the same order; (bx, by): the block.
template <typename T, bool FUSE_P>
__device__ __forceinline__ void force_write(const Geo &g, int t, int bx, int by, const typename Cx<T>::type (&Pt)[8], const double (&val)[8],
                                            double f, const typename Cx<T>::type *__restrict__ ph, double *__restrict__ out,
                                            const double *__restrict__ theta, const double *__restrict__ Splaq, double half_eps, double c_tau,
                                            double K, int compact, int nkick, double i_half, double i_full) {
    typedef typename Cx<T>::type T2;
    constexpr bool PHASE_BOSON = FUSE_P && sizeof(T) == 8;
    const int L = g.L, Vs = g.Vs;
    const int tn = (t + 1 == g.Nt) ? 0 : t + 1, tp = (t == 0) ? g.Nt - 1 : t - 1;
    const int xa = 2 * bx + 1, xb = (xa + 1 == L) ? 0 : xa + 1, ya = 2 * by + 1;
    // site of each bond (block_engine.cuh make_block): y-bonds (xa,ya) (xb,ya) (xa,2by) (xb,2by), x-bonds (xa,2by) (xa,2by+1) (2bx,2by) (2bx,2by+1)
    const int bxs[8] = {xa, xb, xa, xb, xa, xa, 2 * bx, 2 * bx}, bys[8] = {ya, ya, 2 * by, 2 * by, 2 * by, 2 * by + 1, 2 * by, 2 * by + 1};
    int off[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) off[j] = (j < 4 ? Vs : 0) + bys[j] * L + bxs[j];
    double *o = out + (size_t)t * 2 * Vs;
    // two groups of four bonds (y-bonds, then x-bonds): the group's global reads first, in one batch (the stores to o[] would
    // otherwise fence the later loads of o[]); four at a time keeps the batch within the register budget
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        double pv[4]; T2 Pp[4], Pn[4]; double thm[4], th0[4], thq[4];
        if (FUSE_P) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int j = 4 * h + i;
                pv[i] = o[off[j]];
                if (PHASE_BOSON) {
                    if (compact) { Pp[i] = ph[(size_t)tp * 2 * Vs + off[j]]; Pn[i] = ph[(size_t)tn * 2 * Vs + off[j]]; }
                    else { thm[i] = theta[(size_t)tp * 2 * Vs + off[j]]; th0[i] = theta[(size_t)t * 2 * Vs + off[j]]; thq[i] = theta[(size_t)tn * 2 * Vs + off[j]]; }
                }
            }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int j = 4 * h + i;
            const double gF = f * val[j];
            if (FUSE_P) {
                double gB;
                if (PHASE_BOSON) {
                    const int x = bxs[j], y = bys[j], sN = y * L + x;
                    if (compact) {                    // c_tau [sin(theta_t - theta_{t-1}) - sin(theta_{t+1} - theta_t)]
                        const double i2 = (j >= 6) ? i_full : i_half;              // family 1 carries tanh(a), the others tanh(a/2)
                        const double sm = ((double)Pt[j].y * Pp[i].x - (double)Pt[j].x * Pp[i].y) * i2, sp = ((double)Pn[i].y * Pt[j].x - (double)Pn[i].x * Pt[j].y) * i2;
                        gB = c_tau * (sm - sp);
                    } else {
                        gB = 2.0 * c_tau * ((th0[i] - thm[i]) - (thq[i] - th0[i]));
                    }
                    if (h == 1) gB += -K * Splaq[sN] + K * Splaq[((y == 0) ? L - 1 : y - 1) * L + x];       // x-bonds
                    else        gB += K * Splaq[sN] - K * Splaq[y * L + ((x == 0) ? L - 1 : x - 1)];       // y-bonds
                } else {
                    gB = dSB_bond(theta, g, t, off[j], c_tau, K, compact);
                }
                double pvj = pv[i];
                for (int n = 0; n < nkick; ++n) pvj = fma(-(gB + gF), half_eps, pvj);   // nkick half kicks with the same F (Eq.16)
                o[off[j]] = pvj;
            } else {
                o[off[j]] = gF;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S9 (+S10): one CTA per slice t.
//   dS_F/dtheta_{b,t} = 2 sigma_t Re[ Y_{t+1}^+ (dB_t/dtheta_b) X_t ],  Y_{t+1} = X_{t+1} - sigma_t B_t X_t.
// Forward: R = prod_k (1 + T_k) X_t.  Then the factors are walked in reverse: R is un-swept
// (R_{k-1} = E_k^{-1} R_k), the bond terms of family k are accumulated from (L_k, R_{k-1}), and
// L_{k-1} = E_k L_k.  FUSE_P: p += -(dS_B + dS_F) * half_eps instead of writing dS_F.
// The bosonic force of the fused kick is built from the link-phase table the kernel reads anyway (complex128 only): with
// U = e^{i theta}, sin(theta_a - theta_b) = Im(U_a conj U_b) and sin(curl theta) = Im(U_x(s) U_y(s+x) conj(U_x(s+y)) conj(U_y(s))),
// so the four sines per bond of dS_B/dtheta cost a few multiplications instead of four fp64 sin() calls;
// sin(curl) is formed once per site of the slice into shared memory (every plaquette serves four bonds).
// Dynamic shared memory: exchange buffers (4 nb elements) + 32 doubles + Vs doubles.
// ------------------------------------------------------------------------------------------------
template <typename T, int BPT, int MAXT, bool FUSE_P>
__global__ void __launch_bounds__(MAXT) k_force(Geo g, const typename Cx<T>::type *__restrict__ ph, const typename Cx<T>::type *__restrict__ X, T C,
                        double *__restrict__ out, const double *__restrict__ theta, double half_eps, double c_tau,
                        double K, int compact, int nkick, double th_full, double th_half) {
    typedef typename Cx<T>::type T2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Exch<T2> ex; ex.buf = reinterpret_cast<T2 *>(smem_raw); ex.nb = g.nb; ex.parity = 0;
    BlockIdx b[BPT];
#pragma unroll
    for (int k = 0; k < BPT; ++k) make_block(g, threadIdx.x + k * blockDim.x, b[k]);
    {   // blockIdx.y: chain of a batch (hqmc_api_mdb.inl), each with its own gauge field, phase table, solution and momenta
        const size_t nv = (size_t)blockIdx.y * g.Vs * g.Nt;
        ph += 2 * nv; X += nv; out += 2 * nv; theta += 2 * nv;
    }
    const int t = blockIdx.x, tn = (t + 1 == g.Nt) ? 0 : t + 1;
    const double sigma = (t == g.Nt - 1) ? -1.0 : 1.0;
    constexpr bool PHASE_BOSON = FUSE_P && sizeof(T) == 8;          // boson force from the phase table (fp64 phases only)
    double *Splaq = reinterpret_cast<double *>(smem_raw + sizeof(T2) * 4 * g.nb + 32 * sizeof(double));
    const double i_half = 1.0 / (th_half * th_half), i_full = 1.0 / (th_full * th_full);
    if (PHASE_BOSON) force_splaq(g, ph + (size_t)t * 2 * g.Vs, Splaq, i_half, i_full);
    const T s_half = (T)(1.0 / (1.0 - th_half * th_half)), s_full = (T)(1.0 / (1.0 - th_full * th_full));
    const T sC = (T)(-sigma) * C;
    T2 R[BPT][4], Lv[BPT][4];
    Phases<T2> P[BPT];
    double a4[BPT][2], a3[BPT][2], a2[BPT][2], a1[BPT][2];
#pragma unroll
    for (int k = 0; k < BPT; ++k) {
        a4[k][0] = a4[k][1] = a3[k][0] = a3[k][1] = a2[k][0] = a2[k][1] = a1[k][0] = a1[k][1] = 0.0;
        if (b[k].act) { load_phases(ph + (size_t)t * 2 * g.Vs, b[k], P[k]); load_block(X + (size_t)t * g.Vs, b[k], R[k]); }
    }
    apply_B_norm<BPT>(ex, b, P, R);
#pragma unroll
    for (int k = 0; k < BPT; ++k)
        if (b[k].act) {
            load_block(X + (size_t)tn * g.Vs, b[k], Lv[k]);
#pragma unroll
            for (int i = 0; i < 4; ++i) { Lv[k][i].x = fma(sC, R[k][i].x, Lv[k][i].x); Lv[k][i].y = fma(sC, R[k][i].y, Lv[k][i].y); }
        }
    // reverse walk: E4 | E3 E2 | E1 | E2 E3 | E4  (layouts OO, OE, EE, OE, OO)
#pragma unroll
    for (int k = 0; k < BPT; ++k) if (b[k].act) rev_y(R[k], Lv[k], P[k].p4, a4[k], s_half);
    realign<BPT>(0, ex, b, R); realign<BPT>(0, ex, b, Lv);
#pragma unroll
    for (int k = 0; k < BPT; ++k) if (b[k].act) { rev_y(R[k], Lv[k], P[k].p3, a3[k], s_half); rev_x(R[k], Lv[k], P[k].p2, a2[k], s_half); }
    realign<BPT>(1, ex, b, R); realign<BPT>(1, ex, b, Lv);
#pragma unroll
    for (int k = 0; k < BPT; ++k) if (b[k].act) rev_x(R[k], Lv[k], P[k].p1, a1[k], s_full);
    realign<BPT>(2, ex, b, R); realign<BPT>(2, ex, b, Lv);
#pragma unroll
    for (int k = 0; k < BPT; ++k) if (b[k].act) { rev_x(R[k], Lv[k], P[k].p2, a2[k], s_half); rev_y(R[k], Lv[k], P[k].p3, a3[k], s_half); }
    realign<BPT>(3, ex, b, R); realign<BPT>(3, ex, b, Lv);                    // (their barriers also publish Splaq)
#pragma unroll
    for (int k = 0; k < BPT; ++k) if (b[k].act) rev_y(R[k], Lv[k], P[k].p4, a4[k], s_half);
    // write: every bond of the slice is owned by exactly one (thread, family) pair
    const double f = 2.0 * sigma * (double)C;
#pragma unroll
    for (int k = 0; k < BPT; ++k)
        if (b[k].act) {
            const T2 Pt[8] = {P[k].p4[0], P[k].p4[1], P[k].p3[0], P[k].p3[1], P[k].p2[0], P[k].p2[1], P[k].p1[0], P[k].p1[1]};
            const double val[8] = {a4[k][0], a4[k][1], a3[k][0], a3[k][1], a2[k][0], a2[k][1], a1[k][0], a1[k][1]};
            const int by = b[k].q / g.h, bx = b[k].q - by * g.h;
            force_write<T, FUSE_P>(g, t, bx, by, Pt, val, f, ph, out, theta, Splaq, half_eps, c_tau, K, compact, nkick, i_half, i_full);
        }
}

}  // namespace hqmc
