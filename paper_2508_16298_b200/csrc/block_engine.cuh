// block_engine.cuh -- register-blocked checkerboard sweep engine (device code, sm_100a).
//
// B_tau = e^{V4/2} e^{V3/2} e^{V2/2} e^{V1} e^{V2/2} e^{V3/2} e^{V4/2}   (Eq.22, reading C5)
// Each family factor is a direct sum of 2x2 blocks cosh(a) + sinh(a) T_ij (Eq.23-26).
// We factor out cosh:  e^{aT} = cosh(a) (1 + tanh(a) T), so that one factor costs 4 FMAs per site:
//     v_i' = v_i + P v_j,   v_j' = v_j + conj(P) v_i,   P = tanh(a) e^{i theta_ij}   (phase table entry)
// and the scalar C = cosh(a/2)^6 cosh(a) is folded into the caller's axpy.
//
// Data mapping (differs from the paper's "vector in shared memory"): every thread owns a
// 2x2 block of sites of one time slice IN REGISTERS.  With blocks aligned at (odd x, odd y) family 4 is
// thread-local; at (odd x, even y) families 3 and 2 are local; at (even x, even y) family 1 is local.
// The 7 factors therefore need only 4 re-alignments, each moving 2 of the 4 sites of a thread to a
// neighbouring thread through shared memory (conflict-free: slots are indexed by destination thread):
//     OO:[E4] -> OE:[E3 E2] -> EE:[E1] -> OE:[E2 E3] -> OO:[E4]
// i.e. 64 B/site of shared-memory traffic per B instead of 224 B/site for a vector kept in smem.
#pragma once
#include <cuda_runtime.h>

namespace hqmc {

template <typename T> struct Cx;
template <> struct Cx<double> { typedef double2 type; };
template <> struct Cx<float> { typedef float2 type; };

struct Geo {
    int L, h, nb, Vs, Nt;   // h = L/2, nb = h*h blocks per slice, Vs = L*L
};

// v_i' = v_i + P v_j ; v_j' = v_j + conj(P) v_i      (8 FMAs)
template <typename T2>
__device__ __forceinline__ void rot(T2 &vi, T2 &vj, const T2 P) {
    T2 a = vi, b = vj;
    vi.x = fma(-P.y, b.y, fma(P.x, b.x, a.x));
    vi.y = fma(P.y, b.x, fma(P.x, b.y, a.y));
    vj.x = fma(P.y, a.y, fma(P.x, a.x, b.x));
    vj.y = fma(-P.y, a.x, fma(P.x, a.y, b.y));
}

// Per-thread description of one 2x2 block (constant over slices).
struct BlockIdx {
    int o[4];        // OO-layout site offsets inside a slice: (xa,ya) (xb,ya) (xa,yb) (xb,yb)
    int p4[2], p3[2], p2[2], p1[2];   // phase-table offsets inside a slice (mu stride = Vs)
    int d_yd, d_xd, d_xu, d_yu;       // exchange destinations (block ids)
    int q;
    bool act;
};

__device__ __forceinline__ void make_block(const Geo &g, int q, BlockIdx &b) {
    b.q = q;
    b.act = q < g.nb;
    int qq = b.act ? q : 0;
    int by = qq / g.h, bx = qq - by * g.h;
    int L = g.L;
    int xa = 2 * bx + 1, xb = (xa + 1 == L) ? 0 : xa + 1;
    int ya = 2 * by + 1, yb = (ya + 1 == L) ? 0 : ya + 1;
    b.o[0] = ya * L + xa; b.o[1] = ya * L + xb; b.o[2] = yb * L + xa; b.o[3] = yb * L + xb;
    b.p4[0] = g.Vs + b.o[0];            b.p4[1] = g.Vs + b.o[1];              // y-bonds at (xa,ya),(xb,ya), ya odd
    b.p3[0] = g.Vs + (2 * by) * L + xa; b.p3[1] = g.Vs + (2 * by) * L + xb;   // y-bonds at (xa,2by),(xb,2by)
    b.p2[0] = (2 * by) * L + xa;        b.p2[1] = (2 * by + 1) * L + xa;      // x-bonds at (xa,2by),(xa,2by+1), xa odd
    b.p1[0] = (2 * by) * L + 2 * bx;    b.p1[1] = (2 * by + 1) * L + 2 * bx;  // x-bonds at (2bx,2by),(2bx,2by+1)
    int byp = (by + 1 == g.h) ? 0 : by + 1, bym = (by == 0) ? g.h - 1 : by - 1;
    int bxp = (bx + 1 == g.h) ? 0 : bx + 1, bxm = (bx == 0) ? g.h - 1 : bx - 1;
    b.d_yd = bx + g.h * byp;
    b.d_xd = bxp + g.h * by;
    b.d_xu = bxm + g.h * by;
    b.d_yu = bx + g.h * bym;
}

// The 8 link phases one block needs for one B (each bond of the slice is loaded by exactly one thread).
template <typename T2> struct Phases { T2 p4[2], p3[2], p2[2], p1[2]; };

template <typename T2>
__device__ __forceinline__ void load_phases(const T2 *__restrict__ ph_slice, const BlockIdx &b, Phases<T2> &P) {
    P.p4[0] = __ldg(ph_slice + b.p4[0]); P.p4[1] = __ldg(ph_slice + b.p4[1]);
    P.p3[0] = __ldg(ph_slice + b.p3[0]); P.p3[1] = __ldg(ph_slice + b.p3[1]);
    P.p2[0] = __ldg(ph_slice + b.p2[0]); P.p2[1] = __ldg(ph_slice + b.p2[1]);
    P.p1[0] = __ldg(ph_slice + b.p1[0]); P.p1[1] = __ldg(ph_slice + b.p1[1]);
}

template <typename T2>
__device__ __forceinline__ void load_block(const T2 *__restrict__ slice, const BlockIdx &b, T2 (&v)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) v[i] = slice[b.o[i]];
}
template <typename T2>
__device__ __forceinline__ void store_block(T2 *__restrict__ slice, const BlockIdx &b, const T2 (&v)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) slice[b.o[i]] = v[i];
}

// Exchange buffers: ex[parity][slot][nb].  One __syncthreads per re-alignment (a buffer
// is rewritten only two barriers after it was read).
template <typename T2> struct Exch {
    T2 *buf;     // 4*nb elements
    int nb;
    int parity;
    __device__ __forceinline__ T2 *slot(int s) { return buf + (parity * 2 + s) * nb; }
};

// Re-alignments for BPT blocks per thread.  kind: 0 = OO->OE (y down), 1 = OE->EE (x down),
// 2 = EE->OE (x up), 3 = OE->OO (y up).
template <int BPT, typename T2>
__device__ __forceinline__ void realign(int kind, Exch<T2> &ex, const BlockIdx (&b)[BPT], T2 (&v)[BPT][4]) {
    T2 *s0 = ex.slot(0), *s1 = ex.slot(1);
#pragma unroll
    for (int k = 0; k < BPT; ++k) {
        if (!b[k].act) continue;
        if (kind == 0)      { s0[b[k].d_yd] = v[k][2]; s1[b[k].d_yd] = v[k][3]; }
        else if (kind == 1) { s0[b[k].d_xd] = v[k][1]; s1[b[k].d_xd] = v[k][3]; }
        else if (kind == 2) { s0[b[k].d_xu] = v[k][0]; s1[b[k].d_xu] = v[k][2]; }
        else                { s0[b[k].d_yu] = v[k][0]; s1[b[k].d_yu] = v[k][1]; }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < BPT; ++k) {
        if (!b[k].act) continue;
        T2 r0 = s0[b[k].q], r1 = s1[b[k].q];
        if (kind == 0)      { v[k][2] = v[k][0]; v[k][3] = v[k][1]; v[k][0] = r0; v[k][1] = r1; }
        else if (kind == 1) { v[k][1] = v[k][0]; v[k][3] = v[k][2]; v[k][0] = r0; v[k][2] = r1; }
        else if (kind == 2) { v[k][0] = v[k][1]; v[k][2] = v[k][3]; v[k][1] = r0; v[k][3] = r1; }
        else                { v[k][0] = v[k][2]; v[k][1] = v[k][3]; v[k][2] = r0; v[k][3] = r1; }
    }
    ex.parity ^= 1;
}

template <typename T2> __device__ __forceinline__ void sweep_y(T2 (&v)[4], const T2 (&P)[2]) {
    rot(v[0], v[2], P[0]);   // bond at (xa, ya)
    rot(v[1], v[3], P[1]);   // bond at (xb, ya)
}
template <typename T2> __device__ __forceinline__ void sweep_x(T2 (&v)[4], const T2 (&P)[2]) {
    rot(v[0], v[1], P[0]);   // bond at (xa, ya)
    rot(v[2], v[3], P[1]);   // bond at (xa, yb)
}

// v <- prod_k (1 + t_k T_k) v : B without its scalar C.  Starts and ends in the OO layout.
template <int BPT, typename T2>
__device__ __forceinline__ void apply_B_norm(Exch<T2> &ex, const BlockIdx (&b)[BPT], const Phases<T2> (&P)[BPT],
                                             T2 (&v)[BPT][4]) {
#pragma unroll
    for (int k = 0; k < BPT; ++k) sweep_y(v[k], P[k].p4);
    realign<BPT>(0, ex, b, v);
#pragma unroll
    for (int k = 0; k < BPT; ++k) { sweep_y(v[k], P[k].p3); sweep_x(v[k], P[k].p2); }
    realign<BPT>(1, ex, b, v);
#pragma unroll
    for (int k = 0; k < BPT; ++k) sweep_x(v[k], P[k].p1);
    realign<BPT>(2, ex, b, v);
#pragma unroll
    for (int k = 0; k < BPT; ++k) { sweep_x(v[k], P[k].p2); sweep_y(v[k], P[k].p3); }
    realign<BPT>(3, ex, b, v);
#pragma unroll
    for (int k = 0; k < BPT; ++k) sweep_y(v[k], P[k].p4);
}

// ---- deterministic block reduction of a double (fixed tree), result valid in thread 0 -------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}
// red must hold >= 32 doubles of shared memory.
__device__ __forceinline__ double block_sum(double v, double *red) {
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) red[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        r = (lane < nw) ? red[lane] : 0.0;
        r = warp_sum(r);
    }
    return r;
}
// Lane-strided sum of n partials in a fixed order (16 independent loads in flight per lane, so a few hundred
// partials cost one or two L2 round trips instead of one per element), then the shuffle tree; all 32 lanes of the
// calling warp get the result.
__device__ __forceinline__ double sum_partials_lanes(const double *__restrict__ part, int n, int lane) {
    double s = 0.0;
    int i = lane;
    for (; i + 15 * 32 < n; i += 16 * 32) {
        double a[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) a[k] = part[i + 32 * k];
#pragma unroll
        for (int k = 0; k < 16; ++k) s += a[k];
    }
    {
        double a[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) a[k] = (i + 32 * k < n) ? part[i + 32 * k] : 0.0;
#pragma unroll
        for (int k = 0; k < 16; ++k) s += a[k];
    }
    s = warp_sum(s);
    return __shfl_sync(0xffffffffu, s, 0);
}
// Sum n partials in a fixed order; every thread of the FIRST WARP gets the result (others get 0).
__device__ __forceinline__ double sum_partials_warp0(const double *__restrict__ part, int n) {
    return (threadIdx.x < 32) ? sum_partials_lanes(part, n, threadIdx.x) : 0.0;
}

// Sum n partials with the WHOLE CTA (thread tid of nthreads takes elements tid, tid + nthreads, ... in order, then a
// fixed shuffle/shared-memory tree): one L2 round trip instead of one per 32 elements.  Every thread gets the result.
// red: >= 33 doubles of shared memory.  Contains __syncthreads: call from all threads of the CTA.
__device__ __forceinline__ double cta_sum_partials(const double *__restrict__ part, int n, int tid, int nthreads, double *red) {
    double s = 0.0;
    for (int i = tid; i < n; i += nthreads) s += __ldcg(part + i);
    const int lane = tid & 31, w = tid >> 5, nw = (nthreads + 31) >> 5;
    s = warp_sum(s);
    __syncthreads();
    if (lane == 0) red[w] = s;
    __syncthreads();
    if (w == 0) {
        double r = (lane < nw) ? red[lane] : 0.0;
        r = warp_sum(r);
        if (lane == 0) red[32] = r;
    }
    __syncthreads();
    return red[32];
}

}  // namespace hqmc
