// precond_tma.cuh -- tau-banded preconditioner z = P r (reading C10) as a TMA-tiled kernel.
//
// The paper's kernel stages "a chunk of v plus halo" in shared memory.  Here one CTA of 128
// threads owns 128 consecutive spatial sites x a run of TR slices: one thread issues ALL (TR + 2W) row copies
// of the tile (1-D TMA bulk copies, 2 KB each in complex128) up front, grouped eight rows per mbarrier, so the
// whole tile is in flight at once and no thread ever waits on HBM; each thread then marches its site through
// the run with the 2W+1 slices it needs in a register ring fed from shared memory.  Every r element is read
// from L2/HBM once per run (+2W halo rows per run) and z is written once, coalesced (512 B per warp store).
// Same modes / bookkeeping as k_precond (cg_kernels.cuh).  grid = (ceil(Vs/128), ceil(Nt/TR)).
#pragma once
#include "cg_kernels.cuh"
#include "tma.cuh"

namespace hqmc {

#define HQMC_PC_ROWS_PER_BAR 8
#define HQMC_PC_MAX_BARS 16          // (TR + 2W) <= 128 rows

template <typename T, int W>
__global__ void __launch_bounds__(128) k_precond_tma(Geo g, Taps taps, const typename Cx<T>::type *__restrict__ r,
                                                     typename Cx<T>::type *__restrict__ z, double *__restrict__ part_rz,
                                                     const double *__restrict__ part_rr, int n_rr, CgState *st, int mode, int TR) {
    typedef typename Cx<T>::type T2;
    static_assert(W >= 1 && W <= 12, "register ring of 2W+1 <= 25 slots");
    constexpr int RING = 2 * W + 1;
    pdl_wait();
    if (mode != 0 && *(volatile const int *)&st->done) return;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ double red[32];
    __shared__ __align__(8) uint64_t bars[HQMC_PC_MAX_BARS];
    const int Vs = g.Vs, Nt = g.Nt;
    const int s0 = blockIdx.x * 128, s = s0 + threadIdx.x;
    const bool act = s < Vs;
    const int ncol = min(128, Vs - s0);
    const int ta = blockIdx.y * TR, tb = min(ta + TR, Nt);
    const int nrows = (tb - ta) + 2 * W;                    // rows ta-W .. tb-1+W
    const int nbar = (nrows + HQMC_PC_ROWS_PER_BAR - 1) / HQMC_PC_ROWS_PER_BAR;
    T2 *tile = reinterpret_cast<T2 *>(smem_raw);            // [nrows][128]
    const uint32_t row_bytes = (uint32_t)ncol * sizeof(T2);
    if (threadIdx.x == 0) {
        for (int b = 0; b < nbar; ++b) mbar_init(&bars[b], 1);
        mbar_fence_init();
        for (int b = 0; b < nbar; ++b) {
            const int r0 = b * HQMC_PC_ROWS_PER_BAR, r1 = min(r0 + HQMC_PC_ROWS_PER_BAR, nrows);
            mbar_expect_tx(&bars[b], row_bytes * (uint32_t)(r1 - r0));
            for (int i = r0; i < r1; ++i) {
                int u = ta - W + i;
                if (u < 0) u += Nt; else if (u >= Nt) u -= Nt;
                bulk_g2s(tile + (size_t)i * 128, r + (size_t)u * Vs + s0, row_bytes, &bars[b]);
            }
        }
    }
    __syncthreads();
    // row i of the tile = time ta - W + i, with the antiperiodic sign of the wrap
    // the ring holds doubles whatever T is: a complex64 row is widened once, when it enters the ring
    auto ld = [&](int i) -> double2 {
        if ((i & (HQMC_PC_ROWS_PER_BAR - 1)) == 0) mbar_wait(&bars[i / HQMC_PC_ROWS_PER_BAR], 0);
        const int u = ta - W + i;
        const double sg = (u < 0 || u >= Nt) ? -1.0 : 1.0;
        const T2 v = tile[(size_t)i * 128 + threadIdx.x];
        return make_double2(sg * (double)v.x, sg * (double)v.y);
    };
    double2 ring[RING];
#pragma unroll
    for (int j = 0; j < 2 * W; ++j) ring[j] = ld(j);       // times ta-W .. ta+W-1
    double acc = 0.0;
    T2 *zs = z + (act ? s : 0);
    for (int t = ta; t < tb; t += RING) {
#pragma unroll
        for (int j = 0; j < RING; ++j) {
            const int tt = t + j;
            if (tt < tb) {
                ring[(j + 2 * W) % RING] = ld(tt - ta + 2 * W);            // time tt + W
                const double2 c = ring[(j + W) % RING];
                double zx = taps.p[0] * c.x, zy = taps.p[0] * c.y;
#pragma unroll
                for (int m = 1; m <= W; ++m) {
                    const double2 a = ring[(j + W + m) % RING], b = ring[(j + W - m) % RING];
                    zx = fma(taps.p[m], a.x + b.x, zx);
                    zy = fma(taps.p[m], a.y + b.y, zy);
                }
                T2 zi; zi.x = (T)zx; zi.y = (T)zy;
                if (act) {
                    zs[(size_t)tt * Vs] = zi;
                    acc += c.x * (double)zi.x + c.y * (double)zi.y;
                }
            }
        }
    }
    pdl_launch_dependents();
    double sblk = block_sum(acc, red);
    const int bid = blockIdx.y * gridDim.x + blockIdx.x;
    if (threadIdx.x == 0 && part_rz != nullptr) part_rz[bid] = sblk;
    if (mode != 0 && bid == 0) {
        double rr = sum_partials_warp0(part_rr, n_rr);
        if (threadIdx.x == 0) {
            if (mode == 1) {
                st->bb = rr; st->rr = rr; st->iters = 0;
                st->done = (rr == 0.0 || st->max_iter <= 0) ? 2 : 0;     // 2: finished, no iterate update pending
            } else {
                long long it = st->iters + 1;
                st->iters = it; st->rr = rr;
                if ((st->tol2 > 0.0 && rr <= st->tol2 * st->bb) || it >= st->max_iter) st->done = 1;
            }
        }
    }
}


// ------------------------------------------------------------------------------------------------
// Fused PCG vector kernels (Eq.20), used when the TMA-tiled preconditioner applies (W = 1..6):
//
//   k_cg_rz :  alpha = <r,z>/<d,Od>;  r' = r - alpha Od;  z = P r';  partials ||r'||^2, <r',z>
//   k_cg_xd :  x += alpha d;  beta = <r',z>/<r,z>;  d = z + beta d;  bookkeeping (iteration count, done flag)
//
// k_cg_rz is k_precond_tma with TWO tiles (r and Od, both with the 2W halo rows): the residual update is applied
// to every row as it enters the register ring, so r' never makes a round trip through HBM before P sees it.  r' is
// written to a SECOND buffer (the halo rows of a neighbouring CTA must still see the old r).  One PCG iteration
// then moves 48 (M^+M) + ~82 (rz, halo included) + 80 (xd) B/site instead of 48 + 96 + ~48 + 48.
// SITES = sites per CTA (= threads); grid = (ceil(Vs/SITES), ceil(Nt/TR)).
// ------------------------------------------------------------------------------------------------
// blockDim = (SITES, TG): thread (s, g) produces the 4 consecutive slices ta + 4g .. ta + 4g + 3 of site s, streaming
// the 4 + 2W tile rows it needs through 8 accumulators (no register ring, ~50 registers, 3 CTAs per SM).
__device__ __forceinline__ double block_sum_lin(double v, double *red, int tid, int nthreads) {
    const int lane = tid & 31, w = tid >> 5, nw = (nthreads + 31) >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) red[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) { r = (lane < nw) ? red[lane] : 0.0; r = warp_sum(r); }
    return r;
}

template <typename T, int W, int SITES>
__global__ void __launch_bounds__(SITES * 6, 3) k_cg_rz(Geo g, Taps taps, const typename Cx<T>::type *__restrict__ r_in,
                                                 const typename Cx<T>::type *__restrict__ Od, typename Cx<T>::type *__restrict__ r_out,
                                                 typename Cx<T>::type *__restrict__ z, const double *__restrict__ part_rz_old, int n_rz,
                                                 const double *__restrict__ part_dOd, int n_dOd, double *__restrict__ part_rr,
                                                 double *__restrict__ part_rz, const CgState *__restrict__ st, int TR) {
    typedef typename Cx<T>::type T2;
    static_assert(W >= 1 && W <= 6, "4 + 2W <= 16 tile rows per thread");
    if (*(volatile const int *)&st->done) return;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ double red[34];
    __shared__ __align__(8) uint64_t bars[HQMC_PC_MAX_BARS];
    const int Vs = g.Vs, Nt = g.Nt;
    const int tid = threadIdx.y * SITES + threadIdx.x, nthreads = SITES * blockDim.y;
    const int s0 = blockIdx.x * SITES, s = s0 + threadIdx.x;
    const bool act = s < Vs;
    const int ncol = min(SITES, Vs - s0);
    const int ta = blockIdx.y * TR, tb = min(ta + TR, Nt);
    const int nrows = (tb - ta) + 2 * W;
    const int nbar = (nrows + HQMC_PC_ROWS_PER_BAR - 1) / HQMC_PC_ROWS_PER_BAR;
    T2 *tile_r = reinterpret_cast<T2 *>(smem_raw);                       // [nrows][SITES]
    T2 *tile_o = tile_r + (size_t)nrows * SITES;
    const uint32_t row_bytes = (uint32_t)ncol * sizeof(T2);
    if (tid == 0) {
        for (int b = 0; b < nbar; ++b) mbar_init(&bars[b], 1);
        mbar_fence_init();
        for (int b = 0; b < nbar; ++b) {
            const int r0 = b * HQMC_PC_ROWS_PER_BAR, r1 = min(r0 + HQMC_PC_ROWS_PER_BAR, nrows);
            mbar_expect_tx(&bars[b], 2 * row_bytes * (uint32_t)(r1 - r0));
        }
    }
    __syncthreads();
    if (tid < nrows) {   // one thread per tile row issues that row's two copies: the whole tile is in flight at once
        int u = ta - W + tid;
        if (u < 0) u += Nt; else if (u >= Nt) u -= Nt;
        uint64_t *bar = &bars[tid / HQMC_PC_ROWS_PER_BAR];
        bulk_g2s(tile_r + (size_t)tid * SITES, r_in + (size_t)u * Vs + s0, row_bytes, bar);
        bulk_g2s(tile_o + (size_t)tid * SITES, Od + (size_t)u * Vs + s0, row_bytes, bar);
    }
    // alpha, identical in every CTA (fixed-order sums of the producers' partials, all threads loading at once)
    const double rz_old = cta_sum_partials(part_rz_old, n_rz, tid, nthreads, red);
    const double dOd_tot = cta_sum_partials(part_dOd, n_dOd, tid, nthreads, red);
    const T alpha = (T)(rz_old / dOd_tot);
    const int i0 = 4 * threadIdx.y;                                      // first tile row / first output (relative to ta)
    double zx[4] = {0, 0, 0, 0}, zy[4] = {0, 0, 0, 0};
    T2 cen[4];
#pragma unroll
    for (int o = 0; o < 4; ++o) { cen[o].x = (T)0; cen[o].y = (T)0; }
    if (i0 < tb - ta) {
        // the mbarriers covering rows i0 .. i0 + 3 + 2W (each is used once: phase 0)
        for (int b = i0 / HQMC_PC_ROWS_PER_BAR; b <= min(i0 + 3 + 2 * W, nrows - 1) / HQMC_PC_ROWS_PER_BAR; ++b) mbar_wait(&bars[b], 0);
#pragma unroll
        for (int k = 0; k < 4 + 2 * W; ++k) {
            const int i = i0 + k;                                        // tile row = time ta - W + i
            if (i < nrows) {
                const int u = ta - W + i;
                const T sg = (u < 0 || u >= Nt) ? (T)-1 : (T)1;
                const T2 a = tile_r[(size_t)i * SITES + threadIdx.x], od = tile_o[(size_t)i * SITES + threadIdx.x];
                T2 rp; rp.x = fma(-alpha, od.x, a.x); rp.y = fma(-alpha, od.y, a.y);
                const double vx = (double)(sg * rp.x), vy = (double)(sg * rp.y);
#pragma unroll
                for (int o = 0; o < 4; ++o) {
                    const int m = k - W - o;                             // offset of this row from output o's slice
                    if (m >= -W && m <= W) {
                        zx[o] = fma(taps.p[m < 0 ? -m : m], vx, zx[o]); zy[o] = fma(taps.p[m < 0 ? -m : m], vy, zy[o]);
                        if (m == 0) cen[o] = rp;
                    }
                }
            }
        }
    }
    double acc_rz = 0.0, acc_rr = 0.0;
    if (act) {
#pragma unroll
        for (int o = 0; o < 4; ++o) {
            const int tt = ta + i0 + o;
            if (tt < tb) {
                T2 zi; zi.x = (T)zx[o]; zi.y = (T)zy[o];
                r_out[(size_t)tt * Vs + s] = cen[o];
                z[(size_t)tt * Vs + s] = zi;
                acc_rr += (double)cen[o].x * (double)cen[o].x + (double)cen[o].y * (double)cen[o].y;
                acc_rz += (double)cen[o].x * (double)zi.x + (double)cen[o].y * (double)zi.y;
            }
        }
    }
    const int bid = blockIdx.y * gridDim.x + blockIdx.x;
    double s1 = block_sum_lin(acc_rr, red, tid, nthreads);
    if (tid == 0) part_rr[bid] = s1;
    double s2 = block_sum_lin(acc_rz, red, tid, nthreads);
    if (tid == 0) part_rz[bid] = s2;
}

// x += alpha d;  d = z + beta d;  CTA 0 also does the iteration's bookkeeping.
template <typename T>
__global__ void __launch_bounds__(256) k_cg_xd(size_t N, typename Cx<T>::type *__restrict__ x, typename Cx<T>::type *__restrict__ d,
                        const typename Cx<T>::type *__restrict__ z, const double *__restrict__ part_rz_old,
                        const double *__restrict__ part_rz_new, int n_rz, const double *__restrict__ part_dOd, int n_dOd,
                        const double *__restrict__ part_rr, CgState *st) {
    typedef typename Cx<T>::type T2;
    if (*(volatile const int *)&st->done) return;
    __shared__ double red[34];
    const double rz_old = cta_sum_partials(part_rz_old, n_rz, threadIdx.x, blockDim.x, red);
    const double rz_new = cta_sum_partials(part_rz_new, n_rz, threadIdx.x, blockDim.x, red);
    const double dOd = cta_sum_partials(part_dOd, n_dOd, threadIdx.x, blockDim.x, red);
    const T alpha = (T)(rz_old / dOd), beta = (T)(rz_new / rz_old);
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + stride < N; i += 2 * stride) {          // two independent elements in flight per thread
        const size_t k = i + stride;
        T2 x0 = x[i], d0 = d[i], z0 = z[i], x1 = x[k], d1 = d[k], z1 = z[k];
        x0.x = fma(alpha, d0.x, x0.x); x0.y = fma(alpha, d0.y, x0.y); d0.x = fma(beta, d0.x, z0.x); d0.y = fma(beta, d0.y, z0.y);
        x1.x = fma(alpha, d1.x, x1.x); x1.y = fma(alpha, d1.y, x1.y); d1.x = fma(beta, d1.x, z1.x); d1.y = fma(beta, d1.y, z1.y);
        x[i] = x0; d[i] = d0; x[k] = x1; d[k] = d1;
    }
    if (i < N) {
        T2 x0 = x[i], d0 = d[i], z0 = z[i];
        x0.x = fma(alpha, d0.x, x0.x); x0.y = fma(alpha, d0.y, x0.y); d0.x = fma(beta, d0.x, z0.x); d0.y = fma(beta, d0.y, z0.y);
        x[i] = x0; d[i] = d0;
    }
    if (blockIdx.x == 0) {
        const double rr = cta_sum_partials(part_rr, n_rz, threadIdx.x, blockDim.x, red);
        if (threadIdx.x == 0) {
            const long long it = st->iters + 1;
            st->iters = it; st->rr = rr;
            if ((st->tol2 > 0.0 && rr <= st->tol2 * st->bb) || it >= st->max_iter) st->done = 1;
        }
    }
}

}  // namespace hqmc
