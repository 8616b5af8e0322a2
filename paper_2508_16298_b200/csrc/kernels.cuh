// kernels.cuh -- CUDA kernels of the HQMC hot path (sm_100a).  See include/hqmc.h for the operations
// and DESIGN.md for the data layout, traffic counts and rooflines.
#pragma once
#include "block_engine.cuh"

namespace hqmc {

#define HQMC_MAX_W 32
#define HQMC_MAX_PART 4096

// Device-resident CG bookkeeping (one per context; mirrored to pinned host memory after each chunk).
struct CgState {
    double bb;          // ||rhs||^2
    double rr;          // ||r||^2 after the last completed iteration
    double tol2;        // tol^2 (<= 0: fixed-count mode)
    long long iters;
    long long max_iter;
    int done;
    int pad;
};

struct Taps { double p[HQMC_MAX_W + 1]; int W; };

// ------------------------------------------------------------------------------------------------
// S1: link-phase table.  ph[t][mu][y][x] = tanh(a_fam) (cos theta, sin theta); a = dtau*t for family 1
// (x-bonds with x even: the merged middle factor e^{V1}), dtau*t/2 otherwise (reading C5).
// FUSE_DRIFT: theta += 2 p eps first (Eq.16, 190 Eq.14).
// ------------------------------------------------------------------------------------------------
template <typename T, bool FUSE_DRIFT>
__global__ void k_phase(Geo g, double *__restrict__ theta, const double *__restrict__ p, double two_eps,
                        typename Cx<T>::type *__restrict__ ph, double th_full, double th_half) {
    typedef typename Cx<T>::type T2;
    size_t n = (size_t)2 * g.Vs * g.Nt;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        double th = theta[i];
        if (FUSE_DRIFT) { th = fma(two_eps, p[i], th); theta[i] = th; }
        int r = (int)(i % (size_t)(2 * g.Vs));
        int mu = r / g.Vs;
        int x = (r - mu * g.Vs) % g.L;
        double sc = (mu == 0 && (x & 1) == 0) ? th_full : th_half;
        double s, c;
        sincos(th, &s, &c);
        T2 o; o.x = (T)(sc * c); o.y = (T)(sc * s);
        ph[i] = o;
    }
}

// ------------------------------------------------------------------------------------------------
// S4: out[dst] = in[dst] - sigma C B_tb in[src]   (one CTA per slice tb)
//   M  : src = tb, dst = tb+1;   M^+ : src = tb+1, dst = tb;   sigma = -1 for tb = Nt-1.
// ------------------------------------------------------------------------------------------------
template <typename T, int BPT, int MAXT>
__global__ void __launch_bounds__(MAXT) k_apply_M(Geo g, const typename Cx<T>::type *__restrict__ ph, const typename Cx<T>::type *__restrict__ in,
                          typename Cx<T>::type *__restrict__ out, int dagger, T C) {
    typedef typename Cx<T>::type T2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Exch<T2> ex; ex.buf = reinterpret_cast<T2 *>(smem_raw); ex.nb = g.nb; ex.parity = 0;
    BlockIdx b[BPT];
#pragma unroll
    for (int k = 0; k < BPT; ++k) make_block(g, threadIdx.x + k * blockDim.x, b[k]);
    in += (size_t)blockIdx.y * g.Vs * g.Nt; out += (size_t)blockIdx.y * g.Vs * g.Nt;   // blockIdx.y: vector of a batch
    const int tb = blockIdx.x, tnx = (tb + 1 == g.Nt) ? 0 : tb + 1;
    const int src = dagger ? tnx : tb, dst = dagger ? tb : tnx;
    const T sC = (tb == g.Nt - 1) ? C : -C;     // -sigma*C
    T2 v[BPT][4];
    Phases<T2> P[BPT];
#pragma unroll
    for (int k = 0; k < BPT; ++k)
        if (b[k].act) { load_phases(ph + (size_t)tb * 2 * g.Vs, b[k], P[k]); load_block(in + (size_t)src * g.Vs, b[k], v[k]); }
    apply_B_norm<BPT>(ex, b, P, v);
#pragma unroll
    for (int k = 0; k < BPT; ++k)
        if (b[k].act) {
            T2 w[4];
            load_block(in + (size_t)dst * g.Vs, b[k], w);
#pragma unroll
            for (int i = 0; i < 4; ++i) { w[i].x = fma(sC, v[k][i].x, w[i].x); w[i].y = fma(sC, v[k][i].y, w[i].y); }
            store_block(out + (size_t)dst * g.Vs, b[k], w);
        }
}

// ------------------------------------------------------------------------------------------------
// S5: fused O v = M^+ M v over a time tile [t0, t0+Tt) per CTA.
//   w_t = v_t - sigma_{t-1} B_{t-1} v_{t-1};   out_t = w_t - sigma_t B_t w_{t+1}
// Everything stays in registers: per slice the CTA applies B_t twice (to v_t and to w_{t+1}) with ONE
// load of the slice's phases, reads v_{t+1} once and writes out_t once; one extra B per tile for the
// halo (2 Tt + 1 applications for Tt slices).  DOT: part[blockIdx] = sum_t ||w_t||^2 = <v, O v> share.
// ------------------------------------------------------------------------------------------------
template <typename T, int BPT, int MAXT, bool DOT>
__global__ void __launch_bounds__(MAXT) k_mdagm(Geo g, int Tt, const typename Cx<T>::type *__restrict__ ph,
                        const typename Cx<T>::type *__restrict__ in, typename Cx<T>::type *__restrict__ out, T C,
                        double *__restrict__ part, const CgState *__restrict__ st, int part_stride,
                        size_t ph_stride) {
    typedef typename Cx<T>::type T2;
    // blockIdx.y: vector of a batch (cg_batched.cuh) with its own CgState and its own row of partials, part_stride apart
    if (st != nullptr) { st += blockIdx.y; if (*(volatile const int *)&st->done) return; }
    in += (size_t)blockIdx.y * g.Vs * g.Nt; out += (size_t)blockIdx.y * g.Vs * g.Nt;
    ph += (size_t)blockIdx.y * ph_stride;      // 0: the batch shares one gauge field; 2N: one field per vector (chains)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Exch<T2> ex; ex.buf = reinterpret_cast<T2 *>(smem_raw); ex.nb = g.nb; ex.parity = 0;
    double *red = reinterpret_cast<double *>(smem_raw + sizeof(T2) * 4 * g.nb);
    BlockIdx b[BPT];
#pragma unroll
    for (int k = 0; k < BPT; ++k) make_block(g, threadIdx.x + k * blockDim.x, b[k]);
    const int t0 = blockIdx.x * Tt;
    const int t1 = min(t0 + Tt, g.Nt);
    const size_t Vs = g.Vs;
    T2 vc[BPT][4], wc[BPT][4], wn[BPT][4];
    Phases<T2> P[BPT];
    double acc = 0.0;
    // prologue: w_{t0} = v_{t0} - sigma_{tp} C B_{tp} v_{tp},  tp = t0 - 1
    {
        const int tp = (t0 == 0) ? g.Nt - 1 : t0 - 1;
        const T sC = (tp == g.Nt - 1) ? C : -C;
#pragma unroll
        for (int k = 0; k < BPT; ++k)
            if (b[k].act) { load_phases(ph + (size_t)tp * 2 * Vs, b[k], P[k]); load_block(in + (size_t)tp * Vs, b[k], wc[k]); }
        apply_B_norm<BPT>(ex, b, P, wc);
#pragma unroll
        for (int k = 0; k < BPT; ++k)
            if (b[k].act) {
                load_block(in + (size_t)t0 * Vs, b[k], vc[k]);
#pragma unroll
                for (int i = 0; i < 4; ++i) { wc[k][i].x = fma(sC, wc[k][i].x, vc[k][i].x); wc[k][i].y = fma(sC, wc[k][i].y, vc[k][i].y); }
            }
    }
    for (int t = t0; t < t1; ++t) {
        const int tn = (t + 1 == g.Nt) ? 0 : t + 1;
        const T sC = (t == g.Nt - 1) ? C : -C;
#pragma unroll
        for (int k = 0; k < BPT; ++k)
            if (b[k].act) load_phases(ph + (size_t)t * 2 * Vs, b[k], P[k]);
        apply_B_norm<BPT>(ex, b, P, vc);                      // vc = B_t v_t / C
#pragma unroll
        for (int k = 0; k < BPT; ++k)
            if (b[k].act) {
                T2 vn[4];
                load_block(in + (size_t)tn * Vs, b[k], vn);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    wn[k][i].x = fma(sC, vc[k][i].x, vn[i].x);   // w_{t+1}
                    wn[k][i].y = fma(sC, vc[k][i].y, vn[i].y);
                    vc[k][i] = vn[i];                            // v_{t+1} for the next slice
                }
            }
        T2 q[BPT][4];
#pragma unroll
        for (int k = 0; k < BPT; ++k)
#pragma unroll
            for (int i = 0; i < 4; ++i) q[k][i] = wn[k][i];
        apply_B_norm<BPT>(ex, b, P, q);                       // q = B_t w_{t+1} / C
#pragma unroll
        for (int k = 0; k < BPT; ++k)
            if (b[k].act) {
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    if (DOT) acc += (double)wc[k][i].x * (double)wc[k][i].x + (double)wc[k][i].y * (double)wc[k][i].y;
                    q[k][i].x = fma(sC, q[k][i].x, wc[k][i].x);  // out_t = w_t - sigma_t C q
                    q[k][i].y = fma(sC, q[k][i].y, wc[k][i].y);
                    wc[k][i] = wn[k][i];
                }
                store_block(out + (size_t)t * Vs, b[k], q[k]);
            }
    }
    if (DOT) {
        double s = block_sum(acc, red);
        if (threadIdx.x == 0) part[(size_t)blockIdx.y * part_stride + blockIdx.x] = s;
    }
}

// out = C * B(ph_slice) in  on ONE slice (used to build the preconditioner taps at pi-flux, reading C10).
template <typename T, int BPT, int MAXT>
__global__ void __launch_bounds__(MAXT) k_apply_B(Geo g, const typename Cx<T>::type *__restrict__ ph_slice,
                                                  const typename Cx<T>::type *__restrict__ in,
                                                  typename Cx<T>::type *__restrict__ out, T C) {
    typedef typename Cx<T>::type T2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Exch<T2> ex; ex.buf = reinterpret_cast<T2 *>(smem_raw); ex.nb = g.nb; ex.parity = 0;
    BlockIdx b[BPT];
    T2 v[BPT][4];
    Phases<T2> P[BPT];
#pragma unroll
    for (int k = 0; k < BPT; ++k) {
        make_block(g, threadIdx.x + k * blockDim.x, b[k]);
        if (b[k].act) { load_phases(ph_slice, b[k], P[k]); load_block(in, b[k], v[k]); }
    }
    apply_B_norm<BPT>(ex, b, P, v);
#pragma unroll
    for (int k = 0; k < BPT; ++k)
        if (b[k].act) {
#pragma unroll
            for (int i = 0; i < 4; ++i) { v[k][i].x *= C; v[k][i].y *= C; }
            store_block(out, b[k], v[k]);
        }
}

}  // namespace hqmc
