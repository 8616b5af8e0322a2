// cg_batched.cuh -- multi-right-hand-side PCG: n_vec independent solves of M^+M x_b = phi_b that share one theta
// (the N_rv noise vectors of the stochastic estimator; Eq.20).
//
// Every kernel of the iteration takes the vector index from blockIdx.y; vector b owns lattice vectors at offset b*N, its
// own CgState (alpha, beta, iteration count and `done` flag stay per vector: each solve stops on its own residual) and
// its own partial-sum rows at offset b*pstride.  One launch therefore carries n_vec solves: on lattices whose single solve
// cannot fill 148 SMs ("launch overhead dominates for L < 30") the launch count per solved vector drops by
// n_vec and the link phases of a slice are fetched once into L2 for all vectors.  The iterates of vector b are the ones the
// one-vector solver produces up to the summation order of the partial sums.
#pragma once
#include "cg_kernels.cuh"

namespace hqmc {

template <typename T>
__global__ void k_cgb_init(size_t N, const typename Cx<T>::type *__restrict__ rhs, typename Cx<T>::type *__restrict__ x,
                           typename Cx<T>::type *__restrict__ r, double *__restrict__ part_rr, int pstride) {
    typedef typename Cx<T>::type T2;
    const size_t off = (size_t)blockIdx.y * N;
    rhs += off; x += off; r += off; part_rr += (size_t)blockIdx.y * pstride;
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

// alpha_b = <r,z>_b / <d,Od>_b;  x_b += alpha_b d_b;  r_b -= alpha_b Od_b;  part_rr = partial ||r_b||^2
template <typename T>
__global__ void __launch_bounds__(256, 8) k_cgb_axpy(size_t N, typename Cx<T>::type *__restrict__ x, typename Cx<T>::type *__restrict__ r,
                           const typename Cx<T>::type *__restrict__ d, const typename Cx<T>::type *__restrict__ Od,
                           const double *__restrict__ part_rz, int n_rz, const double *__restrict__ part_dOd, int n_dOd,
                           double *__restrict__ part_rr, int pstride, const CgState *__restrict__ st) {
    typedef typename Cx<T>::type T2;
    st += blockIdx.y;
    if (*(volatile const int *)&st->done) return;
    const size_t off = (size_t)blockIdx.y * N, poff = (size_t)blockIdx.y * pstride;
    x += off; r += off; d += off; Od += off;
    __shared__ double red[34];
    const double rz = cta_sum_partials(part_rz + poff, n_rz, threadIdx.x, blockDim.x, red);
    const double dOd = cta_sum_partials(part_dOd + poff, n_dOd, threadIdx.x, blockDim.x, red);
    const T alpha = (T)(rz / dOd);
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        // x is touched once per iteration: streamed (evict-first) so that r, d and Od|z of the whole batch stay L2-resident
        T2 xi = __ldcs(x + i), ri = r[i], di = d[i], oi = Od[i];
        xi.x = fma(alpha, di.x, xi.x); xi.y = fma(alpha, di.y, xi.y);
        ri.x = fma(-alpha, oi.x, ri.x); ri.y = fma(-alpha, oi.y, ri.y);
        __stcs(x + i, xi);
        r[i] = ri;
        acc += (double)ri.x * (double)ri.x + (double)ri.y * (double)ri.y;
    }
    double s = block_sum(acc, red);
    if (threadIdx.x == 0) part_rr[poff + blockIdx.x] = s;
}

// z_b = P r_b (reading C10): thread = one spatial site marching through a run of TR consecutive slices
// with the 2W+1 rows it needs in a register ring (the one-vector k_precond_win scheme), grid = (ceil(Vs/blockDim.x), ceil(Nt/TR),
// n_vec), blockDim.x <= 128.  part_rz = partial Re<r,z>; mode 1: CG start (bb = ||r||^2, iters = 0); mode 2: iteration bookkeeping
// (rr, ++iters, stop test on ||r|| <= tol ||phi|| or the fixed count; reading C9).
template <typename T, int W>
__global__ void __launch_bounds__(128) k_cgb_precond(Geo g, Taps taps, const typename Cx<T>::type *__restrict__ r,
                                                     typename Cx<T>::type *__restrict__ z, double *__restrict__ part_rz,
                                                     const double *__restrict__ part_rr, int n_rr, int pstride, CgState *st,
                                                     int mode, int TR) {
    typedef typename Cx<T>::type T2;
    constexpr int RING = 2 * W + 1;
    st += blockIdx.z;
    if (*(volatile const int *)&st->done) return;
    __shared__ double red[32];
    const int Vs = g.Vs, Nt = g.Nt;
    const size_t off = (size_t)blockIdx.z * Vs * Nt, poff = (size_t)blockIdx.z * pstride;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    const bool act = s < Vs;
    const int ta = blockIdx.y * TR, tb = min(ta + TR, Nt);
    const T2 *rs = r + off + (act ? s : 0);
    T2 *zs = z + off + (act ? s : 0);
    auto ld = [&](int u) -> T2 {       // r at time u in (-Nt, 2 Nt) with the antiperiodic sign
        T sg = (T)1;
        if (u < 0) { u += Nt; sg = (T)-1; } else if (u >= Nt) { u -= Nt; sg = (T)-1; }
        T2 v = rs[(size_t)u * Vs];
        v.x *= sg; v.y *= sg;
        return v;
    };
    T2 ring[RING];                     // slot of time u: (u - ta + W) mod RING
#pragma unroll
    for (int j = 0; j < 2 * W; ++j) ring[j] = ld(ta - W + j);
    double acc = 0.0;
    for (int t = ta; t < tb; t += RING) {
#pragma unroll
        for (int j = 0; j < RING; ++j) {
            const int tt = t + j;
            if (tt < tb) {
                ring[(j + 2 * W) % RING] = ld(tt + W);
                const T2 c = ring[(j + W) % RING];
                double zx = taps.p[0] * (double)c.x, zy = taps.p[0] * (double)c.y;
#pragma unroll
                for (int m = 1; m <= W; ++m) {
                    const T2 a = ring[(j + W + m) % RING], b = ring[(j + W - m + RING) % RING];
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
    if (threadIdx.x == 0) part_rz[poff + bid] = sblk;
    if (bid == 0) {
        double rr = sum_partials_warp0(part_rr + poff, n_rr);
        if (threadIdx.x == 0) {
            if (mode == 1) {
                st->bb = rr; st->rr = rr; st->iters = 0;
                st->done = (rr == 0.0 || st->max_iter <= 0) ? 2 : 0;
            } else {
                long long it = st->iters + 1;
                st->iters = it; st->rr = rr;
                if ((st->tol2 > 0.0 && (rr <= st->tol2 * st->bb || rr != rr)) || it >= st->max_iter) st->done = 1;   // a non-finite residual ends a tolerance-stopped solve (a fixed-count one runs its count)
            }
        }
    }
}

// Any half bandwidth (and W = 0: identity): one thread per site and slice, the 2W neighbouring rows re-read through L1/L2.
template <typename T>
__global__ void k_cgb_precond_gen(Geo g, Taps taps, const typename Cx<T>::type *__restrict__ r, typename Cx<T>::type *__restrict__ z,
                                  double *__restrict__ part_rz, const double *__restrict__ part_rr, int n_rr, int pstride,
                                  CgState *st, int mode) {
    typedef typename Cx<T>::type T2;
    st += blockIdx.y;
    if (*(volatile const int *)&st->done) return;
    __shared__ double red[32];
    const size_t N = (size_t)g.Vs * g.Nt, poff = (size_t)blockIdx.y * pstride;
    r += (size_t)blockIdx.y * N; z += (size_t)blockIdx.y * N;
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
    if (threadIdx.x == 0) part_rz[poff + blockIdx.x] = sblk;
    if (blockIdx.x == 0) {
        double rr = sum_partials_warp0(part_rr + poff, n_rr);
        if (threadIdx.x == 0) {
            if (mode == 1) {
                st->bb = rr; st->rr = rr; st->iters = 0;
                st->done = (rr == 0.0 || st->max_iter <= 0) ? 2 : 0;
            } else {
                long long it = st->iters + 1;
                st->iters = it; st->rr = rr;
                if ((st->tol2 > 0.0 && (rr <= st->tol2 * st->bb || rr != rr)) || it >= st->max_iter) st->done = 1;   // a non-finite residual ends a tolerance-stopped solve (a fixed-count one runs its count)
            }
        }
    }
}

// beta_b = <r,z>_new / <r,z>_old;  d_b = z_b + beta_b d_b   (first: d_b = z_b)
template <typename T>
__global__ void __launch_bounds__(256, 8) k_cgb_dupdate(size_t N, typename Cx<T>::type *__restrict__ d, const typename Cx<T>::type *__restrict__ z,
                              const double *__restrict__ part_new, const double *__restrict__ part_old, int n, int pstride,
                              int first, const CgState *__restrict__ st) {
    typedef typename Cx<T>::type T2;
    st += blockIdx.y;
    if (*(volatile const int *)&st->done) return;
    const size_t off = (size_t)blockIdx.y * N, poff = (size_t)blockIdx.y * pstride;
    d += off; z += off;
    __shared__ double red[34];
    double bt = 0.0;
    if (!first) {
        const double a = cta_sum_partials(part_new + poff, n, threadIdx.x, blockDim.x, red);
        const double b = cta_sum_partials(part_old + poff, n, threadIdx.x, blockDim.x, red);
        bt = a / b;
    }
    const T beta = (T)bt;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        T2 zi = z[i];
        if (!first) { T2 di = d[i]; zi.x = fma(beta, di.x, zi.x); zi.y = fma(beta, di.y, zi.y); }
        d[i] = zi;
    }
}

}  // namespace hqmc
