// cg_kernels.cuh -- preconditioned CG pieces (Eq.20; readings C8, C9) and the
// tau-banded preconditioner (reading C10).
//
// Reductions are single pass: every producer CTA writes ONE partial; every consumer CTA re-sums the
// partials in a fixed order (warp 0: lane-strided adds + shuffle tree), so alpha/beta are bitwise equal
// in all CTAs, run-to-run deterministic, with no atomics, no extra kernel and no host round trip.
#pragma once
#include "kernels.cuh"
#include "tma.cuh"

namespace hqmc {

// Device-side reset of the CG bookkeeping (no host buffer is read, so a solve can be replayed inside a CUDA graph).
__global__ void k_cg_state_set(CgState *st, double tol2, long long max_iter) {
    st->bb = 0.0; st->rr = 0.0; st->tol2 = tol2; st->iters = 0; st->max_iter = max_iter; st->done = 0; st->pad = 0;
}

// x = 0, r = rhs, part_rr[b] = partial ||rhs||^2
template <typename T>
__global__ void k_cg_init(size_t N, const typename Cx<T>::type *__restrict__ rhs, typename Cx<T>::type *__restrict__ x,
                          typename Cx<T>::type *__restrict__ r, double *__restrict__ part_rr) {
    typedef typename Cx<T>::type T2;
    __shared__ double red[32];
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        T2 b = rhs[i];
        T2 z; z.x = (T)0; z.y = (T)0;
        x[i] = z;
        r[i] = b;
        acc += (double)b.x * (double)b.x + (double)b.y * (double)b.y;
    }
    double s = block_sum(acc, red);
    if (threadIdx.x == 0) part_rr[blockIdx.x] = s;
}

// alpha = <r,z> / <d,Od>;  x += alpha d;  r -= alpha Od;  part_rr = partial ||r||^2
template <typename T>
__global__ void k_cg_axpy(size_t N, typename Cx<T>::type *__restrict__ x, typename Cx<T>::type *__restrict__ r,
                          const typename Cx<T>::type *__restrict__ d, const typename Cx<T>::type *__restrict__ Od,
                          const double *__restrict__ part_rz, int n_rz, const double *__restrict__ part_dOd, int n_dOd,
                          double *__restrict__ part_rr, const CgState *__restrict__ st) {
    typedef typename Cx<T>::type T2;
    pdl_wait();
    if (*(volatile const int *)&st->done) return;
    __shared__ double red[34];
    const double rz = cta_sum_partials(part_rz, n_rz, threadIdx.x, blockDim.x, red);
    const double dOd = cta_sum_partials(part_dOd, n_dOd, threadIdx.x, blockDim.x, red);
    const T alpha = (T)(rz / dOd);
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        // x is touched once per iteration: streaming (evict-first) accesses keep it from displacing r, d, Od/z and the
        // packed phases, which then stay L2-resident between kernels
        T2 xi = __ldcs(x + i), ri = r[i], di = d[i], oi = Od[i];
        xi.x = fma(alpha, di.x, xi.x); xi.y = fma(alpha, di.y, xi.y);
        ri.x = fma(-alpha, oi.x, ri.x); ri.y = fma(-alpha, oi.y, ri.y);
        __stcs(x + i, xi);
        r[i] = ri;
        acc += (double)ri.x * (double)ri.x + (double)ri.y * (double)ri.y;
    }
    pdl_launch_dependents();
    double s = block_sum(acc, red);
    if (threadIdx.x == 0) part_rr[blockIdx.x] = s;
}

// z = P r (banded in tau, site diagonal, antiperiodic wrap), part_rz = partial Re<r,z>.
// mode 0: plain apply (no bookkeeping, st may be NULL);  mode 1: CG start (bb = sum part_rr, iters = 0);
// mode 2: CG iteration (rr = sum part_rr, ++iters, convergence / fixed-count test -> done).
// Thread i handles spatial site s = i mod Vs for one slice: loads are coalesced along s and the 2W
// neighbouring slices are re-read from L1/L2 (the halo is on-chip reuse, not algorithmic traffic).
template <typename T>
__global__ void k_precond(Geo g, Taps taps, const typename Cx<T>::type *__restrict__ r, typename Cx<T>::type *__restrict__ z,
                          double *__restrict__ part_rz, const double *__restrict__ part_rr, int n_rr, CgState *st, int mode) {
    typedef typename Cx<T>::type T2;
    if (mode != 0 && *(volatile const int *)&st->done) return;
    __shared__ double red[32];
    const size_t N = (size_t)g.Vs * g.Nt;
    const int W = taps.W, Nt = g.Nt;
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        int t = (int)(i / (size_t)g.Vs);
        size_t s = i - (size_t)t * g.Vs;
        T2 ri = r[i];
        double zx = taps.p[0] * (double)ri.x, zy = taps.p[0] * (double)ri.y;
        for (int m = 1; m <= W; ++m) {
            int ta = t + m, tb = t - m;
            double sa = 1.0, sb = 1.0;
            if (ta >= Nt) { ta -= Nt; sa = -1.0; }
            if (tb < 0) { tb += Nt; sb = -1.0; }
            T2 a = r[(size_t)ta * g.Vs + s], b = r[(size_t)tb * g.Vs + s];
            double pm = taps.p[m];
            zx = fma(pm, sa * (double)a.x + sb * (double)b.x, zx);
            zy = fma(pm, sa * (double)a.y + sb * (double)b.y, zy);
        }
        T2 zi; zi.x = (T)zx; zi.y = (T)zy;
        z[i] = zi;
        acc += (double)ri.x * (double)zi.x + (double)ri.y * (double)zi.y;
    }
    double sblk = block_sum(acc, red);
    if (threadIdx.x == 0 && part_rz != nullptr) part_rz[blockIdx.x] = sblk;
    if (mode != 0 && blockIdx.x == 0) {
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

// Sliding-window form of the same operator for the common half bandwidth W (compile time): thread = one spatial
// site, marching through a run of TR consecutive slices with the 2W+1 slices it needs held in registers (a 16-slot
// ring, three slots of which are loads in flight), so every r element is read once per run (+2W halo per run)
// instead of 2W+1 times; lanes = consecutive sites, so each load/store instruction moves 32 contiguous elements.
// Same modes / bookkeeping as k_precond.  grid = (ceil(Vs/128), ceil(Nt/TR)); partial index = y*gridDim.x + x.
template <typename T, int W>
__global__ void __launch_bounds__(128) k_precond_win(Geo g, Taps taps, const typename Cx<T>::type *__restrict__ r,
                                                     typename Cx<T>::type *__restrict__ z, double *__restrict__ part_rz,
                                                     const double *__restrict__ part_rr, int n_rr, CgState *st, int mode, int TR) {
    typedef typename Cx<T>::type T2;
    static_assert(W >= 1 && W <= 6, "ring of 16 slots holds 2W+1 <= 13 live slices + 3 in flight");
    constexpr int RING = 16, PF = RING - (2 * W + 1);
    if (mode != 0 && *(volatile const int *)&st->done) return;
    __shared__ double red[32];
    const int Vs = g.Vs, Nt = g.Nt;
    const int s = blockIdx.x * 128 + threadIdx.x;
    const bool act = s < Vs;
    const int ta = blockIdx.y * TR, tb = min(ta + TR, Nt);
    const T2 *rs = r + (act ? s : 0);
    T2 *zs = z + (act ? s : 0);
    // r at time index u in [ta - W, tb - 1 + W] (a subset of (-Nt, 2 Nt) because W < Nt), with the antiperiodic
    // sign; indices past the last slice this run needs are not touched.
    const int u_max = tb - 1 + W;
    auto ld = [&](int u) -> T2 {
        T sg = (T)1;
        if (u > u_max) { T2 zero; zero.x = (T)0; zero.y = (T)0; return zero; }
        if (u < 0) { u += Nt; sg = (T)-1; } else if (u >= Nt) { u -= Nt; sg = (T)-1; }
        T2 v = rs[(size_t)u * Vs];
        v.x *= sg; v.y *= sg;
        return v;
    };
    T2 ring[RING];
    // slot of time u: (u - ta + W) mod RING.  Preload times ta-W .. ta+W-1+PF.
#pragma unroll
    for (int j = 0; j < 2 * W + PF; ++j) ring[j] = ld(ta - W + j);
    double acc = 0.0;
    for (int t = ta; t < tb; t += RING) {
#pragma unroll
        for (int j = 0; j < RING; ++j) {
            const int tt = t + j;
            if (tt < tb) {
                ring[(j + 2 * W + PF) % RING] = ld(tt + W + PF);          // in flight for PF steps
                const T2 c = ring[(j + W) % RING];
                double zx = taps.p[0] * (double)c.x, zy = taps.p[0] * (double)c.y;
#pragma unroll
                for (int m = 1; m <= W; ++m) {
                    const T2 a = ring[(j + W + m) % RING], b = ring[(j + W - m) % RING];
                    zx = fma(taps.p[m], (double)a.x + (double)b.x, zx);
                    zy = fma(taps.p[m], (double)a.y + (double)b.y, zy);
                }
                T2 zi; zi.x = (T)zx; zi.y = (T)zy;
                if (act) {
                    zs[(size_t)tt * Vs] = zi;
                    acc += (double)c.x * (double)zi.x + (double)c.y * (double)zi.y;
                }
            }
        }
    }
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

// beta = <r,z>_new / <r,z>_old;  d = z + beta d   (first: d = z)
template <typename T>
__global__ void k_cg_dupdate(size_t N, typename Cx<T>::type *__restrict__ d, const typename Cx<T>::type *__restrict__ z,
                             const double *__restrict__ part_new, const double *__restrict__ part_old, int n,
                             int first, const CgState *__restrict__ st) {
    typedef typename Cx<T>::type T2;
    pdl_wait();
    if (*(volatile const int *)&st->done) return;
    __shared__ double red[34];
    double bt = 0.0;
    if (!first) {
        const double a = cta_sum_partials(part_new, n, threadIdx.x, blockDim.x, red);
        const double b = cta_sum_partials(part_old, n, threadIdx.x, blockDim.x, red);
        bt = a / b;
    }
    const T beta = (T)bt;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        T2 zi = z[i];
        if (!first) { T2 di = d[i]; zi.x = fma(beta, di.x, zi.x); zi.y = fma(beta, di.y, zi.y); }
        d[i] = zi;
    }
    pdl_launch_dependents();
}

// ------------------------------------------------------------------------------------------------
// Deferred-x form of the two vector kernels (hqmc_set_cg_variant(HQMC_CG_DEFERRED_X); the default when the live set exceeds the L2): x_{k+1} = x_k + alpha_k d_k is applied when d_k is read anyway
// to form d_{k+1}, so d is streamed once per iteration instead of twice (128 instead of 144 B/site for the pair):
//   k_cg_raxpy   :  alpha = <r,z>/<d,Od>;  r -= alpha Od;  partial ||r||^2                      (48 B/site)
//   k_cg_xdupdate:  x += alpha d;  beta = <r,z>_new/<r,z>_old;  d = z + beta d                 (80 B/site)
// The iterate must still receive its last update when the solve stops, so `done` has three states here:
// 0 running; 1 stop decided by the preconditioner kernel of this iteration, x update pending (k_cg_xdupdate then
// applies x += alpha d only); 2 finished (set by the next k_cg_raxpy, or at start-up when there is nothing to do).
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void k_cg_raxpy(size_t N, typename Cx<T>::type *__restrict__ r, const typename Cx<T>::type *__restrict__ Od,
                           const double *__restrict__ part_rz, int n_rz, const double *__restrict__ part_dOd, int n_dOd,
                           double *__restrict__ part_rr, CgState *st) {
    typedef typename Cx<T>::type T2;
    pdl_wait();
    {
        const int done = *(volatile const int *)&st->done;
        if (done) { if (done == 1 && blockIdx.x == 0 && threadIdx.x == 0) *(volatile int *)&st->done = 2; return; }
    }
    __shared__ double red[34];
    const double rz = cta_sum_partials(part_rz, n_rz, threadIdx.x, blockDim.x, red);
    const double dOd = cta_sum_partials(part_dOd, n_dOd, threadIdx.x, blockDim.x, red);
    const T alpha = (T)(rz / dOd);
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        T2 ri = r[i], oi = Od[i];
        ri.x = fma(-alpha, oi.x, ri.x); ri.y = fma(-alpha, oi.y, ri.y);
        r[i] = ri;
        acc += (double)ri.x * (double)ri.x + (double)ri.y * (double)ri.y;
    }
    pdl_launch_dependents();
    double s = block_sum(acc, red);
    if (threadIdx.x == 0) part_rr[blockIdx.x] = s;
}

template <typename T>
__global__ void k_cg_xdupdate(size_t N, typename Cx<T>::type *__restrict__ x, typename Cx<T>::type *__restrict__ d,
                              const typename Cx<T>::type *__restrict__ z, const double *__restrict__ part_rz_new,
                              const double *__restrict__ part_rz_old, int n_rz, const double *__restrict__ part_dOd, int n_dOd,
                              const CgState *__restrict__ st) {
    typedef typename Cx<T>::type T2;
    pdl_wait();
    const int done = *(volatile const int *)&st->done;
    if (done == 2) return;
    __shared__ double red[34];
    const double rz_old = cta_sum_partials(part_rz_old, n_rz, threadIdx.x, blockDim.x, red);
    const double dOd = cta_sum_partials(part_dOd, n_dOd, threadIdx.x, blockDim.x, red);
    const T alpha = (T)(rz_old / dOd);
    if (done == 1) {                                  // last iteration: only the iterate is completed
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
            T2 xi = __ldcs(x + i); const T2 di = d[i];
            xi.x = fma(alpha, di.x, xi.x); xi.y = fma(alpha, di.y, xi.y);
            __stcs(x + i, xi);
        }
        return;
    }
    const double rz_new = cta_sum_partials(part_rz_new, n_rz, threadIdx.x, blockDim.x, red);
    const T beta = (T)(rz_new / rz_old);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        T2 xi = __ldcs(x + i), di = d[i]; const T2 zi = z[i];
        xi.x = fma(alpha, di.x, xi.x); xi.y = fma(alpha, di.y, xi.y);
        di.x = fma(beta, di.x, zi.x); di.y = fma(beta, di.y, zi.y);
        __stcs(x + i, xi); d[i] = di;
    }
    pdl_launch_dependents();
}

// Generic deterministic reductions for the energies (Eq.12).
// kind 0: sum p^2 over doubles a[0..n);  kind 1: Re <a, b> over complex vectors of n elements.
template <typename T>
__global__ void k_reduce(int kind, size_t n, const void *__restrict__ a_, const void *__restrict__ b_, double *__restrict__ part) {
    typedef typename Cx<T>::type T2;
    __shared__ double red[32];
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        if (kind == 0) { double v = ((const double *)a_)[i]; acc = fma(v, v, acc); }
        else { T2 a = ((const T2 *)a_)[i], b = ((const T2 *)b_)[i]; acc += (double)a.x * (double)b.x + (double)a.y * (double)b.y; }
    }
    double s = block_sum(acc, red);
    if (threadIdx.x == 0) part[blockIdx.x] = s;
}

// out[slot] = sum of n partials (single CTA, fixed order)
__global__ void k_final_sum(const double *__restrict__ part, int n, double *__restrict__ out) {
    double s = sum_partials_warp0(part, n);
    if (threadIdx.x == 0) *out = s;
}

}  // namespace hqmc
