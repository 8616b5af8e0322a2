// mdagm_stream.cuh -- building blocks of the streaming fused O v = M^+ M v kernels (sm_100a): packed link phases, the lean
// one-block-per-thread sweep engine, conflict-free staging of slices.  The kernels are in mdagm_back.cuh / mdagm_cluster.cuh.
//
//   w_t = v_t - sigma_{t-1} B_{t-1} v_{t-1};   out_t = w_t - sigma_t B_t w_{t+1}      (Eq.8, 284-314)
//
// One CTA owns a run of consecutive time slices [t0, t1) of the WHOLE spatial lattice (one thread per 2x2
// block of sites, block_engine.cuh).  What is new relative to k_mdagm (kernels.cuh):
//  * every global access is a 1-D TMA bulk copy (cp.async.bulk, SASS UBLKCP) issued one slice ahead by one
//    thread and completed on an mbarrier: v_{t+1} and the link phases of slice t+1 land in shared memory while
//    slice t is being swept, and out_t leaves through a staged bulk store -- no thread ever waits on HBM;
//  * link phases are streamed in a PACKED 8-byte form (PhasePack below) instead of 16-byte complex numbers, so
//    one M^+M moves 16 (v) + 16 (two links) + 16 (out) = 48 B/site, the algorithmic minimum of DESIGN.md;
//  * the grid is one CTA per SM with the slices dealt out as evenly as possible (480 slices over 148 SMs =
//    36 runs of 4 + 112 runs of 3) instead of ceil(Nt/Tt) equal tiles.
#pragma once
#include <cstdint>

#include "kernels.cuh"
#include "tma.cuh"

namespace hqmc {

// ------------------------------------------------------------------------------------------------
// PhasePack: 8 bytes per link.
// double:  theta = k*delta + r, delta = 2 pi / 128, |r| <= delta/2.  The word holds sin(r) as an fp64 with its
//          7 low mantissa bits replaced by k (sin r < 2^-5, so the absolute error of the stored sine is
//          <= 2^-5 * 2^-47 = 2.2e-16 before rounding to nearest, 1.1e-16 after -- half an ulp of a unit phase).
//          Decode: cos r = sqrt(1 - q) = 1 - q/2 - q^2/8 - q^3/16 - 5 q^4/128 (q = sin^2 r <= 6.1e-4, next term
//          2e-18), then one complex multiply with the table entry  tanh(a) e^{i k delta}.  The table lives in shared
//          memory with every entry replicated 8 times (128 entries x 8 x 16 B per scale a): lane l reads replica
//          l & 7, so the 8 lanes of a quarter warp always hit 8 different 16-byte bank groups -- the random lookups
//          are bank-conflict free.
// float:   the scaled phase itself as float2 (8 bytes), no decoding.
// ------------------------------------------------------------------------------------------------
#define HQMC_PHASE_K 128
#define HQMC_PHASE_REP 8
#define HQMC_PHASE_TAB (HQMC_PHASE_K * HQMC_PHASE_REP)      // double2 elements per scale

template <typename T> struct PhasePack;
template <> struct PhasePack<double> {
    typedef unsigned long long word;
    static __device__ __forceinline__ word pack(double theta, double /*scale*/) {
        const double inv_delta = 20.371832715762603;         // 128 / (2 pi)
        const double d_hi = 0.04908738521234052;             // fp64(2 pi / 128)
        const double d_lo = 1.9135106236677392e-18;          // 2 pi / 128 - d_hi
        double kf = rint(theta * inv_delta);
        double r = fma(-kf, d_hi, theta);
        r = fma(-kf, d_lo, r);
        long long k = (long long)kf;
        double s = sin(r);
        unsigned long long u = (unsigned long long)__double_as_longlong(s);
        u = (u + 64ull) & ~127ull;                           // round the mantissa to 46 bits
        return u | (unsigned long long)(k & 127ll);
    }
    // tab: this scale's table, already offset by the calling lane's replica (lane & 7)
    static __device__ __forceinline__ double2 decode(word u, const double2 *__restrict__ tab) {
        const unsigned k = (unsigned)u & 127u;
        const double sr = __longlong_as_double((long long)(u & ~127ull));
        const double q = sr * sr;
        const double cr = fma(q, fma(q, fma(q, fma(q, -0.0390625, -0.0625), -0.125), -0.5), 1.0);
        const double2 t = tab[k * HQMC_PHASE_REP];
        double2 P;
        P.x = fma(-t.y, sr, t.x * cr);
        P.y = fma(t.x, sr, t.y * cr);
        return P;
    }
};
template <> struct PhasePack<float> {
    typedef float2 word;
    static __device__ __forceinline__ word pack(double theta, double scale) {
        double s, c;
        sincos(theta, &s, &c);
        return make_float2((float)(scale * c), (float)(scale * s));
    }
    static __device__ __forceinline__ float2 decode(word u, const double2 *) { return u; }
};

// Position of bond (mu, y, x) of a slice in the block-major packed layout [4 pairs][nb blocks][2]:
// pair 0 = family 4 (y-bonds, y odd), 1 = family 3 (y-bonds, y even), 2 = family 2 (x-bonds, x odd),
// 3 = family 1 (x-bonds, x even) -- the order in which block_engine.cuh's BlockIdx lists p4, p3, p2, p1.
__device__ __forceinline__ int packed_slot(const Geo &g, int mu, int y, int x) {
    int j, bx, by, e;
    if (mu == 1) {
        if (x & 1) { bx = (x - 1) >> 1; e = 0; } else { bx = (x >> 1) - 1; if (bx < 0) bx = g.h - 1; e = 1; }
        if (y & 1) { j = 0; by = (y - 1) >> 1; } else { j = 1; by = y >> 1; }
    } else {
        by = y >> 1; e = y & 1;
        if (x & 1) { j = 2; bx = (x - 1) >> 1; } else { j = 3; bx = x >> 1; }
    }
    return ((j * g.nb) + by * g.h + bx) * 2 + e;
}

// S1 (streaming form): packed[t][4][nb][2] from theta[t][2][L][L]; a = dtau*t for family 1, dtau*t/2 otherwise.
template <typename T>
__global__ void k_phase_pack(Geo g, const double *__restrict__ theta, typename PhasePack<T>::word *__restrict__ packed,
                             double th_full, double th_half) {
    const size_t per = (size_t)2 * g.Vs, n = per * g.Nt;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const size_t t = i / per;
        const int r = (int)(i - t * per);
        const int mu = r / g.Vs, s = r - mu * g.Vs, y = s / g.L, x = s - y * g.L;
        const double sc = (mu == 0 && (x & 1) == 0) ? th_full : th_half;
        packed[t * per + packed_slot(g, mu, y, x)] = PhasePack<T>::pack(theta[i], sc);
    }
}

// ------------------------------------------------------------------------------------------------
// Lean single-block-per-thread engine for the streaming kernel: everything a thread needs is a handful of
// shared-memory element offsets computed once; the four re-alignments of block_engine.cuh are written out
// with compile-time buffer parity so that no register is ever moved (the compiler renames).
// Threads beyond nb (ragged last warp) run the same code on a private dummy exchange slot and never store.
// ------------------------------------------------------------------------------------------------
struct LeanIdx {
    int o0, o1, o2, o3;          // OO-layout site offsets inside a slice: (xa,ya) (xb,ya) (xa,yb) (xb,yb)
    int d_yd, d_xd, d_xu, d_yu;  // exchange destinations
    int q;
    bool act;
};
__device__ __forceinline__ void make_lean(const Geo &g, int q, LeanIdx &b) {
    b.q = q; b.act = q < g.nb;
    const int qq = b.act ? q : 0;
    const int by = qq / g.h, bx = qq - by * g.h, L = g.L;
    const int xa = 2 * bx + 1, xb = (xa + 1 == L) ? 0 : xa + 1;
    const int ya = 2 * by + 1, yb = (ya + 1 == L) ? 0 : ya + 1;
    b.o0 = ya * L + xa; b.o1 = ya * L + xb; b.o2 = yb * L + xa; b.o3 = yb * L + xb;
    const int byp = (by + 1 == g.h) ? 0 : by + 1, bym = (by == 0) ? g.h - 1 : by - 1;
    const int bxp = (bx + 1 == g.h) ? 0 : bx + 1, bxm = (bx == 0) ? g.h - 1 : bx - 1;
    b.d_yd = b.act ? bx + g.h * byp : q; b.d_xd = b.act ? bxp + g.h * by : q;
    b.d_xu = b.act ? bxm + g.h * by : q; b.d_yu = b.act ? bx + g.h * bym : q;
}

// ex: [2 parities][2 slots][nbp] elements.  KIND 0: OO->OE (y down), 1: OE->EE (x down), 2: EE->OE (x up), 3: OE->OO (y up).
// v0..v3 are passed and returned in the layout order (xa,ya) (xb,ya) (xa,yb) (xb,yb) of the CURRENT alignment.
template <int KIND, int PAR, typename T2, typename Hook>
__device__ __forceinline__ void lean_realign(T2 *__restrict__ ex, int nbp, const LeanIdx &b, T2 &v0, T2 &v1, T2 &v2, T2 &v3, Hook &&hook) {
    T2 *s0 = ex + (size_t)(PAR * 2) * nbp, *s1 = s0 + nbp;
    if (KIND == 0)      { s0[b.d_yd] = v2; s1[b.d_yd] = v3; }
    else if (KIND == 1) { s0[b.d_xd] = v1; s1[b.d_xd] = v3; }
    else if (KIND == 2) { s0[b.d_xu] = v0; s1[b.d_xu] = v2; }
    else                { s0[b.d_yu] = v0; s1[b.d_yu] = v1; }
    __syncthreads();
    hook();
    const T2 r0 = s0[b.q], r1 = s1[b.q];
    if (KIND == 0)      { v2 = v0; v3 = v1; v0 = r0; v1 = r1; }
    else if (KIND == 1) { v1 = v0; v3 = v2; v0 = r0; v2 = r1; }
    else if (KIND == 2) { v0 = v1; v2 = v3; v1 = r0; v3 = r1; }
    else                { v0 = v2; v1 = v3; v2 = r0; v3 = r1; }
}

template <typename T2> struct LeanPh { T2 a4, b4, a3, b3, a2, b2, a1, b1; };   // p4[0], p4[1], p3[0], ...

// v <- prod_k (1 + t_k T_k) v  (B without its scalar C), OO layout in and out; hook runs on every thread right
// after the first barrier.
template <typename T2, typename Hook>
__device__ __forceinline__ void lean_apply_B(T2 *__restrict__ ex, int nbp, const LeanIdx &b, const LeanPh<T2> &P,
                                             T2 &v0, T2 &v1, T2 &v2, T2 &v3, Hook &&hook) {
    rot(v0, v2, P.a4); rot(v1, v3, P.b4);
    lean_realign<0, 0>(ex, nbp, b, v0, v1, v2, v3, hook);
    rot(v0, v2, P.a3); rot(v1, v3, P.b3);
    rot(v0, v1, P.a2); rot(v2, v3, P.b2);
    lean_realign<1, 1>(ex, nbp, b, v0, v1, v2, v3, []() {});
    rot(v0, v1, P.a1); rot(v2, v3, P.b1);
    lean_realign<2, 0>(ex, nbp, b, v0, v1, v2, v3, []() {});
    rot(v0, v1, P.a2); rot(v2, v3, P.b2);
    rot(v0, v2, P.a3); rot(v1, v3, P.b3);
    lean_realign<3, 1>(ex, nbp, b, v0, v1, v2, v3, []() {});
    rot(v0, v2, P.a4); rot(v1, v3, P.b4);
}

template <typename T> struct PackLoad;
template <> struct PackLoad<double> {
    static __device__ __forceinline__ void pair(const unsigned char *p, const double2 *tab, double2 &A, double2 &B) {
        const ulonglong2 w = *reinterpret_cast<const ulonglong2 *>(p);
        A = PhasePack<double>::decode(w.x, tab); B = PhasePack<double>::decode(w.y, tab);
    }
};
template <> struct PackLoad<float> {
    static __device__ __forceinline__ void pair(const unsigned char *p, const double2 *, float2 &A, float2 &B) {
        const float4 w = *reinterpret_cast<const float4 *>(p);
        A = make_float2(w.x, w.y); B = make_float2(w.z, w.w);
    }
};
template <typename T>
__device__ __forceinline__ void lean_load_phases(const unsigned char *pbuf, const double2 *tab, int nb, int q, LeanPh<typename Cx<T>::type> &P) {
    const unsigned char *p = pbuf + (size_t)q * 16;
    const size_t st = (size_t)nb * 16;
    tab += threadIdx.x & (HQMC_PHASE_REP - 1);             // this lane's replica of the table
    PackLoad<T>::pair(p, tab, P.a4, P.b4);
    PackLoad<T>::pair(p + st, tab, P.a3, P.b3);
    PackLoad<T>::pair(p + 2 * st, tab, P.a2, P.b2);
    PackLoad<T>::pair(p + 3 * st, tab + HQMC_PHASE_TAB, P.a1, P.b1);
}

// Conflict-free block load / store of the staged slices: a thread's sites (xa, y) and (xb, y) are 16 B apart with a
// 32 B stride between lanes, so a plain 128-bit access per site is a 2-way bank conflict.  Lanes 4..7 of every
// quarter warp take the two sites in the opposite order: the 8 lanes then touch 8 different 16-byte bank groups.
template <typename T2, typename Idx>
__device__ __forceinline__ void load_block_swz(const T2 *__restrict__ buf, const Idx &b, T2 &v0, T2 &v1, T2 &v2, T2 &v3) {
    const bool sw = threadIdx.x & 4;
    const T2 a = buf[sw ? b.o1 : b.o0], c = buf[sw ? b.o0 : b.o1];
    const T2 d = buf[sw ? b.o3 : b.o2], e = buf[sw ? b.o2 : b.o3];
    v0 = sw ? c : a; v1 = sw ? a : c; v2 = sw ? e : d; v3 = sw ? d : e;
}
template <typename T2, typename Idx>
__device__ __forceinline__ void store_block_swz(T2 *__restrict__ buf, const Idx &b, const T2 &v0, const T2 &v1, const T2 &v2, const T2 &v3) {
    const bool sw = threadIdx.x & 4;
    buf[sw ? b.o1 : b.o0] = sw ? v1 : v0; buf[sw ? b.o0 : b.o1] = sw ? v0 : v1;
    buf[sw ? b.o3 : b.o2] = sw ? v3 : v2; buf[sw ? b.o2 : b.o3] = sw ? v2 : v3;
}

__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    mbar_expect_tx(bar, bytes);
    bulk_g2s(dst, src, bytes, bar);
}

}  // namespace hqmc
