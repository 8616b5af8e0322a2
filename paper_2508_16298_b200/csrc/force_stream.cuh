// force_stream.cuh -- streaming form of the fermionic force + fused kick (sm_100a), PAPER.md:455-477 (SI), reading C11:
//   dS_F/dtheta_{b,t} = 2 sigma_t Re[ Y_{t+1}^+ (dB_t/dtheta_b) X_t ],  Y_{t+1} = X_{t+1} - sigma_t B_t X_t.
//
// Same arithmetic as k_force (force_kernels.cuh: forward product R = prod E_k X_t, then the factors walked in reverse with
// R un-swept and Y swept, every bond's term accumulated once per factor that contains it; same epilogue force_write), but on
// the streaming engine of the M^+M kernels (mdagm_stream.cuh) instead of one cold CTA per slice:
//  * one CTA per SM owns a run of consecutive slices and walks it from t1-1 down to t0, so X_{t+1} of one step is X_t of the
//    step before: every slice of X is fetched once per CTA (+1 halo slice), by 1-D TMA bulk copies into a ring of TWO
//    shared-memory buffers, one step ahead, completed on mbarriers;
//  * the links come as 8-byte packed phases (TMA, one slice ahead) and are decoded in the kernel, as in k_mdagm_back;
//  * the eight bond sums of a thread go through the (then idle) exchange buffers into the slice's own [mu][y][x] order, so the
//    epilogue -- dS_F/dtheta, or the kick with the bosonic force from the link-phase table -- reads p and the phases and
//    writes p in full lines.  What the epilogue reads for the first time (the phases of slice t-1, p of slice t) is pulled into
//    L2 by two bulk prefetches the leader issues at the start of the step: 70 -> 66 us in situ.  (Per-thread prefetch.global.L2
//    instructions a step ahead had lost, 78 us: they compete with the sweeps for the LSU.)
// Slices are addressed by n = t1 - t (n = 0: the halo slice t1); slice n lives in X buffer n mod 2.
#pragma once
#include "force_kernels.cuh"
#include "mdagm_back.cuh"

namespace hqmc {

template <typename T> struct ForceSmem {
    size_t tab, xbuf, pbuf, exch, splaq, bars, total;       // xbuf: 2 slice buffers
    __host__ __device__ ForceSmem(int Vs, int nbp) {
        typedef typename Cx<T>::type T2;
        size_t o = 0;
        tab = o;   o += (sizeof(T) == 8) ? (size_t)2 * HQMC_PHASE_TAB * sizeof(double2) : 0;
        xbuf = o;  o += (size_t)2 * Vs * sizeof(T2);
        pbuf = o;  o += (size_t)2 * Vs * 8;
        exch = o;  o += (size_t)4 * nbp * sizeof(T2);
        splaq = o; o += (size_t)Vs * sizeof(double);
        bars = o;  o += 8 * sizeof(uint64_t);
        total = o;
    }
};

// one reverse step on the lean (one block per thread) register layout: v0..v3 = (xa,ya) (xb,ya) (xa,yb) (xb,yb)
template <typename T2, typename TS>
__device__ __forceinline__ void lean_rev_y(T2 &r0, T2 &r1, T2 &r2, T2 &r3, T2 &l0, T2 &l1, T2 &l2, T2 &l3, const T2 Pa, const T2 Pb,
                                           double &acc_a, double &acc_b, const TS s) {
    unrot(r0, r2, Pa, s); unrot(r1, r3, Pb, s);
    acc_a += bond_term(l0, l2, r0, r2, Pa); acc_b += bond_term(l1, l3, r1, r3, Pb);
    rot(l0, l2, Pa); rot(l1, l3, Pb);
}
template <typename T2, typename TS>
__device__ __forceinline__ void lean_rev_x(T2 &r0, T2 &r1, T2 &r2, T2 &r3, T2 &l0, T2 &l1, T2 &l2, T2 &l3, const T2 Pa, const T2 Pb,
                                           double &acc_a, double &acc_b, const TS s) {
    unrot(r0, r1, Pa, s); unrot(r2, r3, Pb, s);
    acc_a += bond_term(l0, l1, r0, r1, Pa); acc_b += bond_term(l2, l3, r2, r3, Pb);
    rot(l0, l1, Pa); rot(l2, l3, Pb);
}

// Epilogue of one slice, coalesced: the threads have put f * (their eight bond sums) into `stage` in the slice's own order
// [mu][y][x]; now thread i takes bonds i, i + blockDim, ...: dS_F/dtheta, or with FUSE_P the kick p += -(dS_B + dS_F) half_eps
// (nkick times) with the bosonic force from the link-phase table (see force_kernels.cuh), every global access a full line.
template <typename T, bool FUSE_P>
__device__ __forceinline__ void force_slice_epilogue(const Geo &g, int t, const double *__restrict__ stage, const double *__restrict__ Splaq,
                                                     const typename Cx<T>::type *__restrict__ ph, double *__restrict__ out,
                                                     const double *__restrict__ theta, double half_eps, double c_tau, double K, int compact,
                                                     int nkick, double i_half, double i_full) {
    typedef typename Cx<T>::type T2;
    constexpr bool PHASE_BOSON = FUSE_P && sizeof(T) == 8;
    const int L = g.L, Vs = g.Vs, n2 = 2 * Vs;
    const int tn = (t + 1 == g.Nt) ? 0 : t + 1, tp = (t == 0) ? g.Nt - 1 : t - 1;
    double *o = out + (size_t)t * n2;
    const T2 *pt = ph + (size_t)t * n2, *pp = ph + (size_t)tp * n2, *pn = ph + (size_t)tn * n2;
#pragma unroll 4
    for (int r = threadIdx.x; r < n2; r += blockDim.x) {
        const double gF = stage[r];
        if (!FUSE_P) { o[r] = gF; continue; }
        double gB;
        if (PHASE_BOSON) {
            const int mu = r >= Vs, sN = r - mu * Vs, y = sN / L, x = sN - y * L;
            if (compact) {
                const T2 Pt = pt[r], Pp = pp[r], Pn = pn[r];
                const double i2 = (mu == 0 && !(x & 1)) ? i_full : i_half;
                gB = c_tau * (((double)Pt.y * Pp.x - (double)Pt.x * Pp.y) - ((double)Pn.y * Pt.x - (double)Pn.x * Pt.y)) * i2;
            } else {
                const double th0 = theta[(size_t)t * n2 + r];
                gB = 2.0 * c_tau * ((th0 - theta[(size_t)tp * n2 + r]) - (theta[(size_t)tn * n2 + r] - th0));
            }
            if (mu == 0) gB += -K * Splaq[sN] + K * Splaq[((y == 0) ? L - 1 : y - 1) * L + x];
            else         gB += K * Splaq[sN] - K * Splaq[y * L + ((x == 0) ? L - 1 : x - 1)];
        } else {
            gB = dSB_bond(theta, g, t, r, c_tau, K, compact);
        }
        double pv = o[r];
        for (int n = 0; n < nkick; ++n) pv = fma(-(gB + gF), half_eps, pv);
        o[r] = pv;
    }
}

// grid = G CTAs; CTA i owns slices [i*Nt/G, (i+1)*Nt/G); blockDim.x = nb rounded up to 32 (one 2x2 block per thread).
// packed / tab_g as in k_mdagm_back; ph: the complex link-phase table (bosonic force of the fused kick); out: dS_F/dtheta, or
// with FUSE_P the momenta p (in/out).
template <typename T, bool FUSE_P>
__global__ void __launch_bounds__(576, 1) k_force_stream(Geo g, const typename PhasePack<T>::word *__restrict__ packed,
                        const double2 *__restrict__ tab_g, const typename Cx<T>::type *__restrict__ ph,
                        const typename Cx<T>::type *__restrict__ X, T C, double *__restrict__ out, const double *__restrict__ theta,
                        double half_eps, double c_tau, double K, int compact, int nkick, double th_full, double th_half) {
    typedef typename Cx<T>::type T2;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nbp = blockDim.x;
    const ForceSmem<T> lay(g.Vs, nbp);
    const double2 *tab = reinterpret_cast<const double2 *>(smem_raw + lay.tab);
    unsigned char *pbuf = smem_raw + lay.pbuf;
    T2 *ex = reinterpret_cast<T2 *>(smem_raw + lay.exch);
    double *Splaq = reinterpret_cast<double *>(smem_raw + lay.splaq);
    uint64_t *bar_x = reinterpret_cast<uint64_t *>(smem_raw + lay.bars), *bar_p = bar_x + 2, *bar_t = bar_x + 3;
    LeanIdx b;
    make_lean(g, threadIdx.x, b);
    constexpr bool PHASE_BOSON = FUSE_P && sizeof(T) == 8;

    const int G = gridDim.x;
    const int t0 = (int)(((long long)blockIdx.x * g.Nt) / G), t1 = (int)(((long long)(blockIdx.x + 1) * g.Nt) / G);
    if (t0 >= t1) return;
    const int nsl = t1 - t0;
    const uint32_t vbytes = (uint32_t)g.Vs * sizeof(T2), pbytes = (uint32_t)g.Vs * 16;
    const unsigned char *in_b = reinterpret_cast<const unsigned char *>(X);
    const unsigned char *pk_b = reinterpret_cast<const unsigned char *>(packed);
    const bool leader = threadIdx.x == 0;
    auto slice_of = [&](int n) { int t = t1 - n; if (t >= g.Nt) t -= g.Nt; return t; };
    auto xb = [&](int n) { return smem_raw + lay.xbuf + (size_t)(n & 1) * vbytes; };
    auto load_x = [&](int n) { bulk_load(xb(n), in_b + (size_t)slice_of(n) * vbytes, vbytes, bar_x + (n & 1)); };
    auto load_p = [&](int n) { bulk_load(pbuf, pk_b + (size_t)slice_of(n) * pbytes, pbytes, bar_p); };
    uint32_t parx = 0, par_p = 0;
    auto wait_x = [&](int n) { const int k = n & 1; mbar_wait(bar_x + k, (parx >> k) & 1u); parx ^= (1u << k); };

    if (leader) {
        mbar_init(bar_x, 1); mbar_init(bar_x + 1, 1); mbar_init(bar_p, 1); mbar_init(bar_t, 1);
        mbar_fence_init();
        if (sizeof(T) == 8) bulk_load(smem_raw + lay.tab, tab_g, 2 * HQMC_PHASE_TAB * sizeof(double2), bar_t);
        load_p(1); load_x(1); load_x(0);
    }
    __syncthreads();
    if (sizeof(T) == 8) mbar_wait(bar_t, 0);
    const int qd = b.act ? b.q : 0;
    const int by = qd / g.h, bx = qd - by * g.h;
    const double i_half = 1.0 / (th_half * th_half), i_full = 1.0 / (th_full * th_full);
    const T s_half = (T)(1.0 / (1.0 - th_half * th_half)), s_full = (T)(1.0 / (1.0 - th_full * th_full));
    wait_x(0);                                                // the halo slice X_{t1}

    for (int j = 0; j < nsl; ++j) {
        const int n = j + 1, t = slice_of(n);
        const double sigma = (t == g.Nt - 1) ? -1.0 : 1.0;
        const T sC = (T)(-sigma) * C;
        LeanPh<T2> P;
        mbar_wait(bar_p, par_p); par_p ^= 1;
        lean_load_phases<T>(pbuf, tab, g.nb, qd, P);          // links of slice t
        wait_x(n);
        T2 r0, r1, r2, r3;
        load_block_swz(reinterpret_cast<const T2 *>(xb(n)), b, r0, r1, r2, r3);
        // forward: R = prod_k (1 + T_k) X_t.  Behind its first barrier every thread has decoded the links: fetch the next ones.
        lean_apply_B2(ex, nbp, b, P, r0, r1, r2, r3, [&]() {
            if (leader) {
                if (n + 1 <= nsl) load_p(n + 1);
                if (FUSE_P) {      // what this step's epilogue will read for the first time: into L2 while the sweeps run
                    const int tpp = (t == 0) ? g.Nt - 1 : t - 1;
                    if (PHASE_BOSON && compact) bulk_prefetch_l2(ph + (size_t)tpp * 2 * g.Vs, (uint32_t)(2 * g.Vs * sizeof(T2)));
                    bulk_prefetch_l2(out + (size_t)t * 2 * g.Vs, (uint32_t)(2 * g.Vs * sizeof(double)));
                }
            }
        }, []() {});
        // (the barriers of the forward product separate the previous step's reads of Splaq from these writes)
        if (PHASE_BOSON) force_splaq(g, ph + (size_t)t * 2 * g.Vs, Splaq, i_half, i_full);
        T2 l0, l1, l2, l3;                                    // Y_{t+1} = X_{t+1} - sigma C R
        load_block_swz(reinterpret_cast<const T2 *>(xb(n - 1)), b, l0, l1, l2, l3);
        l0.x = fma(sC, r0.x, l0.x); l0.y = fma(sC, r0.y, l0.y); l1.x = fma(sC, r1.x, l1.x); l1.y = fma(sC, r1.y, l1.y);
        l2.x = fma(sC, r2.x, l2.x); l2.y = fma(sC, r2.y, l2.y); l3.x = fma(sC, r3.x, l3.x); l3.y = fma(sC, r3.y, l3.y);
        double a4a = 0, a4b = 0, a3a = 0, a3b = 0, a2a = 0, a2b = 0, a1a = 0, a1b = 0;
        // reverse walk: E4 | E3 E2 | E1 | E2 E3 | E4  (layouts OO, OE, EE, OE, OO); R and Y re-aligned one after the other
        lean_rev_y(r0, r1, r2, r3, l0, l1, l2, l3, P.a4, P.b4, a4a, a4b, s_half);
        // behind this barrier every thread has read X_{t+1}: its buffer takes X_{t-1} (slice n + 1)
        lean_realign<0, 0>(ex, nbp, b, r0, r1, r2, r3, [&]() { if (leader && n + 1 <= nsl) load_x(n + 1); });
        lean_realign<0, 1>(ex, nbp, b, l0, l1, l2, l3, []() {});
        lean_rev_y(r0, r1, r2, r3, l0, l1, l2, l3, P.a3, P.b3, a3a, a3b, s_half);
        lean_rev_x(r0, r1, r2, r3, l0, l1, l2, l3, P.a2, P.b2, a2a, a2b, s_half);
        lean_realign<1, 0>(ex, nbp, b, r0, r1, r2, r3, []() {});
        lean_realign<1, 1>(ex, nbp, b, l0, l1, l2, l3, []() {});
        lean_rev_x(r0, r1, r2, r3, l0, l1, l2, l3, P.a1, P.b1, a1a, a1b, s_full);
        lean_realign<2, 0>(ex, nbp, b, r0, r1, r2, r3, []() {});
        lean_realign<2, 1>(ex, nbp, b, l0, l1, l2, l3, []() {});
        lean_rev_x(r0, r1, r2, r3, l0, l1, l2, l3, P.a2, P.b2, a2a, a2b, s_half);
        lean_rev_y(r0, r1, r2, r3, l0, l1, l2, l3, P.a3, P.b3, a3a, a3b, s_half);
        lean_realign<3, 0>(ex, nbp, b, r0, r1, r2, r3, []() {});
        lean_realign<3, 1>(ex, nbp, b, l0, l1, l2, l3, []() {});
        lean_rev_y(r0, r1, r2, r3, l0, l1, l2, l3, P.a4, P.b4, a4a, a4b, s_half);
        // the exchange buffers are idle now: they take the slice's bond sums in the slice's own order (4 nbp elements >= 2 Vs
        // doubles), so that the epilogue reads and writes global memory in full lines
        double *stage = reinterpret_cast<double *>(ex);
        __syncthreads();                                      // everyone is past the last re-alignment's reads
        if (b.act) {
            const int L = g.L, xa = 2 * bx + 1, xb_ = (xa + 1 == L) ? 0 : xa + 1, ya = 2 * by + 1;
            const double f = 2.0 * sigma * (double)C;
            stage[g.Vs + ya * L + xa] = f * a4a;        stage[g.Vs + ya * L + xb_] = f * a4b;              // family 4: y-bonds at (xa,ya) (xb,ya)
            stage[g.Vs + 2 * by * L + xa] = f * a3a;    stage[g.Vs + 2 * by * L + xb_] = f * a3b;          // family 3: y-bonds at (xa,2by) (xb,2by)
            stage[2 * by * L + xa] = f * a2a;           stage[(2 * by + 1) * L + xa] = f * a2b;            // family 2: x-bonds at (xa,2by) (xa,2by+1)
            stage[2 * by * L + 2 * bx] = f * a1a;       stage[(2 * by + 1) * L + 2 * bx] = f * a1b;        // family 1: x-bonds at (2bx,2by) (2bx,2by+1)
        }
        __syncthreads();
        force_slice_epilogue<T, FUSE_P>(g, t, stage, Splaq, ph, out, theta, half_eps, c_tau, K, compact, nkick, i_half, i_full);
        __syncthreads();                                      // before the next step's exchanges overwrite the stage
    }
}

}  // namespace hqmc
