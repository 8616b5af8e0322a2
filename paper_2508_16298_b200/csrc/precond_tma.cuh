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
                if ((st->tol2 > 0.0 && (rr <= st->tol2 * st->bb || rr != rr)) || it >= st->max_iter) st->done = 1;   // a non-finite residual ends a tolerance-stopped solve (a fixed-count one runs its count)
            }
        }
    }
}


}  // namespace hqmc
