// mdagm_back.cuh -- streaming O v = M^+ M v, time run swept BACKWARDS (sm_100a).
//
//   w_t = v_t - sigma_{t-1} B_{t-1} v_{t-1};   out_t = w_t - sigma_t B_t w_{t+1}      (Eq.8, 284-314)
//
// Same mapping as k_mdagm_stream (one CTA per SM, whole slices, one thread per 2x2 block in registers, packed links,
// TMA bulk copies), but the CTA walks its slices from t1-1 down to t0.  Going down, step t needs
//     q = B_t w_{t+1}           (links of slice t,   w_{t+1} carried in registers from the previous step)
//     a = B_{t-1} v_{t-1}       (links of slice t-1, independent of q)
//     w_t = v_t - sigma a;  out_t = w_t - sigma q;  carry w_t
// so only ONE set of decoded links and two block vectors are live at a time (64 registers instead of the 80 of the
// forward order: nothing spills under the 96-register ceiling), and out_t is staged in the very shared-memory buffer
// v_t was read from (each thread rewrites its own four sites), which frees room for a THIRD v buffer: v is fetched
// 1.5 steps ahead.
#pragma once
#include "mdagm_stream.cuh"

namespace hqmc {

template <typename T> struct BackSmem {
    size_t tab, vbuf, pbuf, exch, red, bars, total;      // vbuf: 3 slice buffers
    __host__ __device__ BackSmem(int Vs, int nbp) {
        typedef typename Cx<T>::type T2;
        size_t o = 0;
        tab = o;  o += (sizeof(T) == 8) ? (size_t)2 * HQMC_PHASE_TAB * sizeof(double2) : 0;
        vbuf = o; o += (size_t)3 * Vs * sizeof(T2);
        pbuf = o; o += (size_t)2 * Vs * 8;
        exch = o; o += (size_t)4 * nbp * sizeof(T2);
        red = o;  o += 32 * sizeof(double);
        bars = o; o += 8 * sizeof(uint64_t);
        total = o;
    }
};

// apply_B with two leader hooks: after the first and after the second barrier of the sweep sequence
template <typename T2, typename Hook1, typename Hook2>
__device__ __forceinline__ void lean_apply_B2(T2 *__restrict__ ex, int nbp, const LeanIdx &b, const LeanPh<T2> &P,
                                              T2 &v0, T2 &v1, T2 &v2, T2 &v3, Hook1 &&h1, Hook2 &&h2) {
    rot(v0, v2, P.a4); rot(v1, v3, P.b4);
    lean_realign<0, 0>(ex, nbp, b, v0, v1, v2, v3, h1);
    rot(v0, v2, P.a3); rot(v1, v3, P.b3);
    rot(v0, v1, P.a2); rot(v2, v3, P.b2);
    lean_realign<1, 1>(ex, nbp, b, v0, v1, v2, v3, h2);
    rot(v0, v1, P.a1); rot(v2, v3, P.b1);
    lean_realign<2, 0>(ex, nbp, b, v0, v1, v2, v3, []() {});
    rot(v0, v1, P.a2); rot(v2, v3, P.b2);
    rot(v0, v2, P.a3); rot(v1, v3, P.b3);
    lean_realign<3, 1>(ex, nbp, b, v0, v1, v2, v3, []() {});
    rot(v0, v2, P.a4); rot(v1, v3, P.b4);
}

// grid = G CTAs; CTA i owns slices [i*Nt/G, (i+1)*Nt/G); blockDim.x = nb rounded up to 32.  Arguments as k_mdagm_stream.
// Slices are addressed by n = t1 - t (n = 0: the halo slice t1 above the run, n = nsl + 1: the halo slice t0 - 1 below);
// slice n lives in v buffer n mod 3.
template <typename T, bool DOT>
__global__ void __launch_bounds__(576, 1) k_mdagm_back(Geo g, const typename PhasePack<T>::word *__restrict__ packed,
                        const double2 *__restrict__ tab_g, const typename Cx<T>::type *__restrict__ in,
                        typename Cx<T>::type *__restrict__ out, T C, double *__restrict__ part, const CgState *__restrict__ st) {
    typedef typename Cx<T>::type T2;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nbp = blockDim.x;
    const BackSmem<T> lay(g.Vs, nbp);
    const double2 *tab = reinterpret_cast<const double2 *>(smem_raw + lay.tab);
    unsigned char *pbuf = smem_raw + lay.pbuf;
    T2 *ex = reinterpret_cast<T2 *>(smem_raw + lay.exch);
    double *red = reinterpret_cast<double *>(smem_raw + lay.red);
    uint64_t *bar_v = reinterpret_cast<uint64_t *>(smem_raw + lay.bars), *bar_p = bar_v + 3, *bar_t = bar_v + 4;
    LeanIdx b;
    make_lean(g, threadIdx.x, b);

    const int G = gridDim.x;
    const int t0 = (int)(((long long)blockIdx.x * g.Nt) / G), t1 = (int)(((long long)(blockIdx.x + 1) * g.Nt) / G);
    if (t0 >= t1) { if (DOT && threadIdx.x == 0) part[blockIdx.x] = 0.0; return; }
    const int nsl = t1 - t0;
    const uint32_t vbytes = (uint32_t)g.Vs * sizeof(T2), pbytes = (uint32_t)g.Vs * 16;
    const unsigned char *in_b = reinterpret_cast<const unsigned char *>(in);
    const unsigned char *pk_b = reinterpret_cast<const unsigned char *>(packed);
    unsigned char *out_b = reinterpret_cast<unsigned char *>(out);
    const bool leader = threadIdx.x == 0;
    auto slice_of = [&](int n) { int t = t1 - n; if (t >= g.Nt) t -= g.Nt; if (t < 0) t += g.Nt; return t; };
    auto vb = [&](int n) { return smem_raw + lay.vbuf + (size_t)(n % 3) * vbytes; };
    auto load_v = [&](int n) { bulk_load(vb(n), in_b + (size_t)slice_of(n) * vbytes, vbytes, bar_v + (n % 3)); };
    auto load_p = [&](int n) { bulk_load(pbuf, pk_b + (size_t)slice_of(n) * pbytes, pbytes, bar_p); };
    const int n_last_v = nsl + 1;                       // last slice index fetched from `in` (the low halo slice t0 - 1)
    uint32_t parv = 0, par_p = 0;                       // bit k of parv: parity of v buffer k
    auto wait_v = [&](int n) { const int k = n % 3; mbar_wait(bar_v + k, (parv >> k) & 1u); parv ^= (1u << k); };

    if (leader) {
        mbar_init(bar_v, 1); mbar_init(bar_v + 1, 1); mbar_init(bar_v + 2, 1); mbar_init(bar_p, 1); mbar_init(bar_t, 1);
        mbar_fence_init();
        if (sizeof(T) == 8) bulk_load(smem_raw + lay.tab, tab_g, 2 * HQMC_PHASE_TAB * sizeof(double2), bar_t);
        load_p(1);                                      // links of slice t1 - 1: do not depend on the previous kernel
    }
    pdl_wait();                                         // `in` and `st` are the previous kernels' output
    if (leader) {
        load_v(1); load_v(0);
        if (2 <= n_last_v) load_v(2);
    }
    const int done = (st != nullptr) ? *(volatile const int *)&st->done : 0;
    __syncthreads();
    if (sizeof(T) == 8) mbar_wait(bar_t, 0);
    if (done) {
        mbar_wait(bar_v, 0); mbar_wait(bar_v + 1, 0); mbar_wait(bar_p, 0);
        if (2 <= n_last_v) mbar_wait(bar_v + 2, 0);
        return;
    }
    const int qd = b.act ? b.q : 0;
    LeanPh<T2> P;
    T2 q0, q1, q2, q3;                                  // w_{t+1}, then B_t w_{t+1}
    double acc = 0.0;
    auto sC_of = [&](int t) -> T { return (t == g.Nt - 1) ? C : -C; };     // -sigma_t C

    // ---- start: w_{t1} = v_{t1} - sigma C B_{t1-1} v_{t1-1}
    mbar_wait(bar_p, par_p); par_p ^= 1;
    lean_load_phases<T>(pbuf, tab, g.nb, qd, P);        // links of slice t1 - 1
    wait_v(1);
    load_block_swz(reinterpret_cast<const T2 *>(vb(1)), b, q0, q1, q2, q3);
    lean_apply_B2(ex, nbp, b, P, q0, q1, q2, q3, []() {}, []() {});
    {
        const T sC = sC_of(slice_of(1));
        wait_v(0);
        T2 v0, v1, v2, v3;
        load_block_swz(reinterpret_cast<const T2 *>(vb(0)), b, v0, v1, v2, v3);
        q0.x = fma(sC, q0.x, v0.x); q0.y = fma(sC, q0.y, v0.y); q1.x = fma(sC, q1.x, v1.x); q1.y = fma(sC, q1.y, v1.y);
        q2.x = fma(sC, q2.x, v2.x); q2.y = fma(sC, q2.y, v2.y); q3.x = fma(sC, q3.x, v3.x); q3.y = fma(sC, q3.y, v3.y);
    }
    for (int j = 0; j < nsl; ++j) {
        const int n = j + 1, t = slice_of(n), tm = slice_of(n + 1);
        const T sCt = sC_of(t), sCm = sC_of(tm);
        if (j == nsl - 1) pdl_launch_dependents();      // let the next kernel's CTAs be dispatched under this CTA's tail
        // 1. q = B_t w_{t+1} / C.  First barrier: everyone is past the previous step -> thread 0 stores out_{t+1} (staged in
        //    buffer n-1) and fetches the links of slice t-1 (pbuf was decoded before the previous step's second sweep).
        //    Second barrier: that store has surely finished reading, so the same buffer can take v_{t-2} (slice n+2).
        lean_apply_B2(ex, nbp, b, P, q0, q1, q2, q3,
            [&]() {
                if (leader) {
                    if (j > 0) { bulk_s2g(out_b + (size_t)slice_of(n - 1) * vbytes, vb(n - 1), vbytes); bulk_commit(); }
                    load_p(n + 1);
                }
            },
            [&]() {
                if (leader && n + 2 <= n_last_v) { bulk_wait_read0(); load_v(n + 2); }
            });
        // 2. links of slice t-1
        mbar_wait(bar_p, par_p); par_p ^= 1;
        lean_load_phases<T>(pbuf, tab, g.nb, qd, P);
        // 3. a = B_{t-1} v_{t-1} / C
        wait_v(n + 1);
        T2 a0, a1, a2, a3;
        load_block_swz(reinterpret_cast<const T2 *>(vb(n + 1)), b, a0, a1, a2, a3);
        lean_apply_B2(ex, nbp, b, P, a0, a1, a2, a3, []() {}, []() {});
        // 4. w_t = v_t - sigma_{t-1} C a;  out_t = w_t - sigma_t C q, staged over v_t;  carry w_t
        T2 *vt = reinterpret_cast<T2 *>(vb(n));
        T2 v0, v1, v2, v3;
        load_block_swz(const_cast<const T2 *>(vt), b, v0, v1, v2, v3);
        v0.x = fma(sCm, a0.x, v0.x); v0.y = fma(sCm, a0.y, v0.y); v1.x = fma(sCm, a1.x, v1.x); v1.y = fma(sCm, a1.y, v1.y);
        v2.x = fma(sCm, a2.x, v2.x); v2.y = fma(sCm, a2.y, v2.y); v3.x = fma(sCm, a3.x, v3.x); v3.y = fma(sCm, a3.y, v3.y);
        if (DOT && b.act)
            acc += ((double)v0.x * v0.x + (double)v0.y * v0.y) + ((double)v1.x * v1.x + (double)v1.y * v1.y) +
                   ((double)v2.x * v2.x + (double)v2.y * v2.y) + ((double)v3.x * v3.x + (double)v3.y * v3.y);
        q0.x = fma(sCt, q0.x, v0.x); q0.y = fma(sCt, q0.y, v0.y); q1.x = fma(sCt, q1.x, v1.x); q1.y = fma(sCt, q1.y, v1.y);
        q2.x = fma(sCt, q2.x, v2.x); q2.y = fma(sCt, q2.y, v2.y); q3.x = fma(sCt, q3.x, v3.x); q3.y = fma(sCt, q3.y, v3.y);
        if (b.act) store_block_swz(vt, b, q0, q1, q2, q3);
        fence_async_smem();
        q0 = v0; q1 = v1; q2 = v2; q3 = v3;
    }
    __syncthreads();
    if (leader) {
        bulk_s2g(out_b + (size_t)slice_of(nsl) * vbytes, vb(nsl), vbytes);
        bulk_commit();
        bulk_wait0();
    }
    if (DOT) {
        double s = block_sum(acc, red);
        if (threadIdx.x == 0) part[blockIdx.x] = s;
    }
}

}  // namespace hqmc
