// pcg_persist.cuh -- a whole preconditioned CG solve (Eq.20; readings C8, C9) as ONE persistent kernel, for
// lattices too small to fill the GPU (the regime PAPER.md:350 calls launch-bound, L < 30): there the four kernels of an
// iteration cost ~3.7 us each whatever the size, i.e. their launch and drain.
//
// One CTA per time slice (cooperative launch: all Ntau CTAs are resident), one thread per 2x2 block of sites
// (block_engine.cuh).  A thread keeps ITS four sites of x, r, d and z = P r | O d in registers for the whole solve, and the
// decoded links of its slice and of the slice below as well; global memory carries only what the neighbours need -- d (read one
// slice up and down by M^+M) and r (read W slices up and down by the preconditioner) -- and x at the end.  Per iteration:
//     [a = B_{t-1} d_{t-1}, b = B_t d_t, w_t = d_t - s a, w_{t+1} = d_{t+1} - s b, Od_t = w_t - s B_t w_{t+1}, <d,Od> share]
//     EXCHANGE       [alpha; x += alpha d; r -= alpha Od; r -> global]
//     neighbours     [z = P r; shares of ||r||^2 and <r,z>]                 (wait for the r of the W slices either side)
//     EXCHANGE       [stopping test; beta; d = z + beta d; d -> global]
//     neighbours                                                            (wait for the d of slices t - 1 and t + 1)
// Every CTA sums the per-CTA shares itself, in the same fixed order, so alpha, beta and the stopping decision are bitwise
// identical everywhere and the result is deterministic run to run (no atomics anywhere).  The two EXCHANGES are the two global
// sums of Eq.20, done as an all-to-all of tagged words (exchange_sum below: 0.8 us against 2.7 us for partials + an atomic grid
// barrier + re-read, measured on a B200); the two halo hand-overs are point to point (a flag per CTA, polled by the CTAs that
// read its slice).  All CTAs are resident, so no spin can starve anyone.  A buffer is rewritten only after an exchange that
// follows its last read (r: read before the second exchange, rewritten after the first of the next iteration; d likewise):
// a CTA's share depends on everything it has read, so whoever has seen every share knows those reads are done.
#pragma once
#include "cg_kernels.cuh"

namespace hqmc {

__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_volatile_u64(unsigned long long *p, unsigned long long v) {
    asm volatile("st.volatile.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void st_release_u64(unsigned long long *p, unsigned long long v) {
    asm volatile("st.release.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}

// Layout of the sync words (all zero at launch): [0, 8 G): the exchange slots, 2 buffers x G CTAs x 2 values x 2 words;
// then 2 G flags: CTA t has published r / d of iteration n.
#define HQMC_SYNC_WORDS(G) (10 * (size_t)(G))

// All-to-all exchange of up to two doubles per CTA, which is BOTH global sums of Eq.20 and the only grid-wide synchronisation of
// the iteration.  Every value travels as two self-validating 8-byte words {32 bits of the double, 32-bit round tag} (8-byte
// stores are single-copy atomic, so a reader never sees half a word): no fence, no atomic, no separate barrier -- a reader
// polls the words of CTA j until their tag is the current round.  Two buffers alternate by round: a CTA writes round n + 2 into
// the buffer of round n only after it has read every CTA's round n + 1 words, which those wrote after reading all of round n.
// Thread 0 publishes (v0, v1); thread j gathers CTA j, j + nthr, ... in order, then the fixed tree of cta_sum: every CTA gets the
// same bits.  red: >= 34 doubles.
template <int NV>
__device__ __forceinline__ void exchange_sum(unsigned long long *slots, unsigned G, unsigned &round, double v0, double v1,
                                             int tid, int nthr, double *red, double &s0, double &s1) {
    ++round;
    unsigned long long *buf = slots + (size_t)(round & 1u) * 4 * G;
    if (tid == 0) {
        const unsigned long long a = (unsigned long long)__double_as_longlong(v0), c = (unsigned long long)__double_as_longlong(v1);
        unsigned long long *mine = buf + 4 * blockIdx.x;
        st_volatile_u64(mine, (a & 0xffffffff00000000ull) | round);
        st_volatile_u64(mine + 1, (a << 32) | round);
        if (NV > 1) { st_volatile_u64(mine + 2, (c & 0xffffffff00000000ull) | round); st_volatile_u64(mine + 3, (c << 32) | round); }
    }
    // gather: all of a thread's slots are requested in one pass (independent 16-byte loads), passes repeat for the late ones
    constexpr int JMAX = 8;                                 // G <= 8 nthr (checked on the host)
    double v0s[JMAX], v1s[JMAX];
    unsigned pending = 0;
#pragma unroll
    for (int k = 0; k < JMAX; ++k) { v0s[k] = 0.0; v1s[k] = 0.0; if (tid + k * nthr < (int)G) pending |= 1u << k; }
    while (pending) {
#pragma unroll
        for (int k = 0; k < JMAX; ++k) {
            if (!((pending >> k) & 1u)) continue;
            const unsigned long long *w = buf + 4 * (size_t)(tid + k * nthr);
            unsigned long long h, l, h2 = round, l2 = round;
            asm volatile("ld.volatile.global.v2.u64 {%0, %1}, [%2];" : "=l"(h), "=l"(l) : "l"(w) : "memory");
            if (NV > 1) asm volatile("ld.volatile.global.v2.u64 {%0, %1}, [%2];" : "=l"(h2), "=l"(l2) : "l"(w + 2) : "memory");
            if ((h & 0xffffffffull) == round && (l & 0xffffffffull) == round && (h2 & 0xffffffffull) == round && (l2 & 0xffffffffull) == round) {
                v0s[k] = __longlong_as_double((long long)((h & 0xffffffff00000000ull) | (l >> 32)));
                if (NV > 1) v1s[k] = __longlong_as_double((long long)((h2 & 0xffffffff00000000ull) | (l2 >> 32)));
                pending &= ~(1u << k);
            }
        }
    }
    double a0 = 0.0, a1 = 0.0;
#pragma unroll
    for (int k = 0; k < JMAX; ++k) { a0 += v0s[k]; a1 += v1s[k]; }
    const int lane = tid & 31, wq = tid >> 5, nw = (nthr + 31) >> 5;
    a0 = warp_sum(a0);
    if (NV > 1) a1 = warp_sum(a1);
    __syncthreads();
    if (lane == 0) { red[wq] = a0; if (NV > 1) red[16 + wq] = a1; }
    __syncthreads();
    if (wq == 0) {
        double r0 = (lane < nw) ? red[lane] : 0.0, r1 = (NV > 1 && lane < nw) ? red[16 + lane] : 0.0;
        r0 = warp_sum(r0);
        if (NV > 1) r1 = warp_sum(r1);
        if (lane == 0) { red[32] = r0; red[33] = r1; }
    }
    __syncthreads();
    s0 = red[32]; s1 = red[33];
}

// Point to point: this CTA has stored its slice (flag := n); it needs the slices of the CTAs t +- 1 .. t +- reach.
__device__ __forceinline__ void neighbour_sync(unsigned long long *flags, int which, int t, int Nt, int reach, unsigned long long n) {
    __syncthreads();
    if (threadIdx.x == 0) st_release_u64(flags + 2 * t + which, n);
    for (int k = threadIdx.x; k < 2 * reach; k += blockDim.x) {
        const int m = (k >> 1) + 1;
        int tt = ((k & 1) ? t + m : t - m) % Nt;
        if (tt < 0) tt += Nt;
        while (ld_volatile_u64(flags + 2 * tt + which) < n) { }
        __threadfence();
    }
    __syncthreads();
}

template <typename T2>
__device__ __forceinline__ void load_block_cg(const T2 *__restrict__ slice, const BlockIdx &b, T2 (&v)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) v[i] = __ldcg(slice + b.o[i]);
}

// ctr: HQMC_SYNC_WORDS(gridDim.x) words, zero at launch; rbuf, dbuf: lattice vectors (workspace).
template <typename T>
__global__ void __launch_bounds__(256) k_pcg_persist(Geo g, Taps taps, const typename Cx<T>::type *__restrict__ ph,
                        const typename Cx<T>::type *__restrict__ rhs, typename Cx<T>::type *__restrict__ x,
                        typename Cx<T>::type *rbuf, typename Cx<T>::type *dbuf, T C, unsigned long long *ctr,
                        CgState *st, double tol2, long long max_iter) {
    typedef typename Cx<T>::type T2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Exch<T2> ex; ex.buf = reinterpret_cast<T2 *>(smem_raw); ex.nb = g.nb; ex.parity = 0;
    double *red = reinterpret_cast<double *>(smem_raw + sizeof(T2) * 4 * g.nb);
    const unsigned G = gridDim.x;
    const int Nt = g.Nt, t = blockIdx.x, tid = threadIdx.x, nthr = blockDim.x;
    const size_t Vs = g.Vs;
    const int tp = (t == 0) ? Nt - 1 : t - 1, tn = (t + 1 == Nt) ? 0 : t + 1;
    const T sCt = (t == Nt - 1) ? C : -C, sCp = (tp == Nt - 1) ? C : -C;        // -sigma C of slices t and t-1
    BlockIdx b[1];
    make_block(g, tid, b[0]);
    const bool act = b[0].act;
    Phases<T2> Pp[1], Pt[1];
    if (act) { load_phases(ph + (size_t)tp * 2 * Vs, b[0], Pp[0]); load_phases(ph + (size_t)t * 2 * Vs, b[0], Pt[0]); }
    unsigned round = 0;
    unsigned long long *flags = ctr + 8 * (size_t)G;
    const int W = taps.W;
    T2 xv[4], rv[4], dv[4], zv[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) { xv[i].x = xv[i].y = 0; rv[i] = xv[i]; dv[i] = xv[i]; zv[i] = xv[i]; }

    // z = P r on this thread's sites of slice t: own slice from registers, the others from global memory (L2)
    auto precond = [&](const T2 *src) {
        const T p0 = (T)taps.p[0];
#pragma unroll
        for (int i = 0; i < 4; ++i) { zv[i].x = p0 * rv[i].x; zv[i].y = p0 * rv[i].y; }
        if (!act) return;
        for (int m = 1; m <= W; ++m) {
            int ta = t + m, tb = t - m;
            T pa = (T)taps.p[m], pb = pa;
            if (ta >= Nt) { ta -= Nt; pa = -pa; }
            if (tb < 0) { tb += Nt; pb = -pb; }
            T2 u[4], w[4];
            load_block_cg(src + (size_t)ta * Vs, b[0], u);
            load_block_cg(src + (size_t)tb * Vs, b[0], w);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                zv[i].x = fma(pa, u[i].x, fma(pb, w[i].x, zv[i].x));
                zv[i].y = fma(pa, u[i].y, fma(pb, w[i].y, zv[i].y));
            }
        }
    };
    auto dot4 = [&](const T2 (&a)[4], const T2 (&c)[4]) {
        double s = 0.0;
#pragma unroll
        for (int i = 0; i < 4; ++i) s += (double)a[i].x * (double)c[i].x + (double)a[i].y * (double)c[i].y;
        return act ? s : 0.0;
    };

    // ---- start: x_0 = 0, r_0 = rhs, z_0 = P r_0, d_0 = z_0
    if (act) load_block(rhs + (size_t)t * Vs, b[0], rv);
    precond(rhs);
    double bb, rz;
    {
        const double s1 = block_sum(dot4(rv, rv), red), s2 = block_sum(dot4(rv, zv), red);
        exchange_sum<2>(ctr, G, round, s1, s2, tid, nthr, red, bb, rz);
    }
    double rr = bb;
#pragma unroll
    for (int i = 0; i < 4; ++i) dv[i] = zv[i];
    if (act) store_block(dbuf + (size_t)t * Vs, b[0], dv);
    neighbour_sync(flags, 1, t, Nt, 1, 1ull);

    long long it = 0;
    while (it < max_iter) {
        // ---- O d on slice t (Eq.8, 284-314) and this CTA's share of <d, O d> = ||M d||^2
        T2 a[1][4], q[1][4], wn[4], wt[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) { a[0][i] = dv[i]; q[0][i] = dv[i]; wn[i] = dv[i]; }
        if (act) { load_block_cg(dbuf + (size_t)tp * Vs, b[0], a[0]); load_block_cg(dbuf + (size_t)tn * Vs, b[0], wn); }
        apply_B_norm<1>(ex, b, Pp, a);                          // B_{t-1} d_{t-1} / C
        apply_B_norm<1>(ex, b, Pt, q);                          // B_t d_t / C
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            wt[i].x = fma(sCp, a[0][i].x, dv[i].x); wt[i].y = fma(sCp, a[0][i].y, dv[i].y);       // w_t
            q[0][i].x = fma(sCt, q[0][i].x, wn[i].x); q[0][i].y = fma(sCt, q[0][i].y, wn[i].y);   // w_{t+1}
        }
        apply_B_norm<1>(ex, b, Pt, q);                          // B_t w_{t+1} / C
#pragma unroll
        for (int i = 0; i < 4; ++i) { zv[i].x = fma(sCt, q[0][i].x, wt[i].x); zv[i].y = fma(sCt, q[0][i].y, wt[i].y); }   // (O d)_t
        double dOd, unused;
        {
            const double s = block_sum(dot4(wt, wt), red);
            exchange_sum<1>(ctr, G, round, s, 0.0, tid, nthr, red, dOd, unused);
        }
        // ---- alpha = <r,z> / <d,Od>;  x += alpha d;  r -= alpha O d
        const T alpha = (T)(rz / dOd);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            xv[i].x = fma(alpha, dv[i].x, xv[i].x); xv[i].y = fma(alpha, dv[i].y, xv[i].y);
            rv[i].x = fma(-alpha, zv[i].x, rv[i].x); rv[i].y = fma(-alpha, zv[i].y, rv[i].y);
        }
        if (act) store_block(rbuf + (size_t)t * Vs, b[0], rv);
        const double rr_share = dot4(rv, rv);
        neighbour_sync(flags, 0, t, Nt, W, (unsigned long long)it + 1);      // r of the W slices either side
        // ---- z = P r, shares of ||r||^2 and <r,z>
        precond(rbuf);
        double rz_new;
        {
            const double s1 = block_sum(rr_share, red), s2 = block_sum(dot4(rv, zv), red);
            exchange_sum<2>(ctr, G, round, s1, s2, tid, nthr, red, rr, rz_new);
        }
        ++it;
        if ((tol2 > 0.0 && rr <= tol2 * bb) || it >= max_iter || !(rr == rr) || !(rz_new == rz_new)) break;
        // ---- beta = <r,z>_new / <r,z>_old;  d = z + beta d
        const T beta = (T)(rz_new / rz);
        rz = rz_new;
#pragma unroll
        for (int i = 0; i < 4; ++i) { dv[i].x = fma(beta, dv[i].x, zv[i].x); dv[i].y = fma(beta, dv[i].y, zv[i].y); }
        if (act) store_block(dbuf + (size_t)t * Vs, b[0], dv);
        neighbour_sync(flags, 1, t, Nt, 1, (unsigned long long)it + 1);      // d of the slices t - 1 and t + 1
    }
    if (act) store_block(x + (size_t)t * Vs, b[0], xv);
    if (blockIdx.x == 0 && tid == 0) {
        st->bb = bb; st->rr = rr; st->tol2 = tol2; st->iters = it; st->max_iter = max_iter; st->done = 1; st->pad = 0;
    }
}

}  // namespace hqmc
