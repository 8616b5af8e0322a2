// mdagm_cluster.cuh -- streaming O v = M^+ M v for lattices whose slice does not fit one SM (L = 64 in complex128).
//
//   w_t = v_t - sigma_{t-1} B_{t-1} v_{t-1};   out_t = w_t - sigma_t B_t w_{t+1}      (Eq.8, 284-314)
//
// k_mdagm_stream needs the whole L x L slice (registers: one thread per 2x2 block, 96 registers; shared memory: five
// slice-sized staging buffers) on ONE SM, which stops at L = 48.  Here a thread-block CLUSTER of R CTAs (R SMs) shares
// a slice: CTA `rank` owns the horizontal strip of h/R block-rows, with the same TMA pipeline on its part of v, of the
// packed links and of out.  The x re-alignments never leave a block-row; of the y re-alignments only the strip's edge
// block-row crosses to the neighbouring CTA: those two complex numbers per thread are written straight into the
// neighbour's shared memory (distributed shared memory, st.shared::cluster) and announced on an mbarrier in the
// neighbour's shared memory (mbarrier.arrive.release.cluster); only the receiving edge threads wait on it.  No
// cluster-wide barrier in steady state, no halo recomputation in space, one halo slice per time run as before.
#pragma once
#include "mdagm_stream.cuh"

namespace hqmc {

__device__ __forceinline__ uint32_t cluster_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t cluster_size() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t map_to_cta(const void *local_smem, uint32_t cta) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(local_smem)), "r"(cta));
    return r;
}
__device__ __forceinline__ void st_remote(uint32_t addr, double2 v) {
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void st_remote(uint32_t addr, float2 v) {
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t bar_addr) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(bar_addr) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

template <typename T> struct ClusterSmem {
    size_t tab, vbuf, vbuf2, pbuf, obuf, exch, edge, red, bars, total;
    __host__ __device__ ClusterSmem(int L, int h, int R, int nbp) {
        typedef typename Cx<T>::type T2;
        const size_t part = (size_t)(2 * (h / R)) * L * sizeof(T2);     // this CTA's rows of a slice
        size_t o = 0;
        tab = o;  o += (sizeof(T) == 8) ? (size_t)2 * HQMC_PHASE_TAB * sizeof(double2) : 0;
        vbuf = o; o += part;
        vbuf2 = o; o += part;
        pbuf = o; o += (size_t)4 * (h / R) * h * 16;                     // 4 link pairs x 16 B per block
        obuf = o; o += part;
        exch = o; o += (size_t)4 * nbp * sizeof(T2);
        edge = o; o += (size_t)2 * 2 * h * sizeof(T2);                  // [K0 | K3][slot][bx]
        red = o;  o += 32 * sizeof(double);
        bars = o; o += 8 * sizeof(uint64_t);
        total = o;
    }
};

// Per-thread description inside one strip of the cluster.
struct ClIdx {
    int o0, o1, o2, o3;           // site offsets inside the CTA's rows of a slice (local row index)
    int d_yd, d_xd, d_xu, d_yu;   // local exchange destinations
    int q, bx;
    int flags;                    // bit0 act, bit1 first block-row of the strip, bit2 last block-row
};

__device__ __forceinline__ void make_cl_idx(const Geo &g, int hr, int q, ClIdx &b) {
    const int nbl = hr * g.h;
    const bool act = q < nbl;
    const int qq = act ? q : 0;
    const int byl = qq / g.h, bx = qq - byl * g.h, L = g.L;
    const int xa = 2 * bx + 1, xb = (xa + 1 == L) ? 0 : xa + 1;
    b.q = q; b.bx = bx;
    b.o0 = (2 * byl) * L + xa; b.o1 = (2 * byl) * L + xb; b.o2 = (2 * byl + 1) * L + xa; b.o3 = (2 * byl + 1) * L + xb;
    const int bxp = (bx + 1 == g.h) ? 0 : bx + 1, bxm = (bx == 0) ? g.h - 1 : bx - 1;
    b.d_xd = act ? bxp + g.h * byl : q; b.d_xu = act ? bxm + g.h * byl : q;
    b.d_yd = (act && byl + 1 < hr) ? bx + g.h * (byl + 1) : q;       // unused (edge path) on the last block-row
    b.d_yu = (act && byl > 0) ? bx + g.h * (byl - 1) : q;            // unused (edge path) on the first block-row
    b.flags = (act ? 1 : 0) | ((act && byl == 0) ? 2 : 0) | ((act && byl == hr - 1) ? 4 : 0);
}

// Addresses a CTA needs for the edge exchange.
template <typename T2> struct ClEdge {
    T2 *in_k0, *in_k3;            // my incoming edge buffers (slot 0; slot 1 = + h)
    uint64_t *bar_k0, *bar_k3;    // my mbarriers (h arrivals each)
    uint32_t out_k0, out_k3;      // neighbours' buffers (cluster shared addresses): K0 goes to rank+1, K3 to rank-1
    uint32_t rbar_k0, rbar_k3;    // neighbours' mbarriers
    int h;
};

template <int KIND, int PAR, typename T2, typename Hook>
__device__ __forceinline__ void cl_realign(T2 *__restrict__ ex, int nbp, const ClIdx &b, const ClEdge<T2> &e, uint32_t parK,
                                           T2 &v0, T2 &v1, T2 &v2, T2 &v3, Hook &&hook) {
    T2 *s0 = ex + (size_t)(PAR * 2) * nbp, *s1 = s0 + nbp;
    if (KIND == 0) {
        if (b.flags & 4) {
            st_remote(e.out_k0 + (uint32_t)(b.bx * sizeof(T2)), v2); st_remote(e.out_k0 + (uint32_t)((e.h + b.bx) * sizeof(T2)), v3);
            mbar_arrive_remote(e.rbar_k0);
        } else { s0[b.d_yd] = v2; s1[b.d_yd] = v3; }
    } else if (KIND == 1) { s0[b.d_xd] = v1; s1[b.d_xd] = v3; }
    else if (KIND == 2)   { s0[b.d_xu] = v0; s1[b.d_xu] = v2; }
    else {
        if (b.flags & 2) {
            st_remote(e.out_k3 + (uint32_t)(b.bx * sizeof(T2)), v0); st_remote(e.out_k3 + (uint32_t)((e.h + b.bx) * sizeof(T2)), v1);
            mbar_arrive_remote(e.rbar_k3);
        } else { s0[b.d_yu] = v0; s1[b.d_yu] = v1; }
    }
    __syncthreads();
    hook();
    T2 r0, r1;
    if (KIND == 0 && (b.flags & 2))      { mbar_wait_cluster(e.bar_k0, parK); r0 = e.in_k0[b.bx]; r1 = e.in_k0[e.h + b.bx]; }
    else if (KIND == 3 && (b.flags & 4)) { mbar_wait_cluster(e.bar_k3, parK); r0 = e.in_k3[b.bx]; r1 = e.in_k3[e.h + b.bx]; }
    else { r0 = s0[b.q]; r1 = s1[b.q]; }
    if (KIND == 0)      { v2 = v0; v3 = v1; v0 = r0; v1 = r1; }
    else if (KIND == 1) { v1 = v0; v3 = v2; v0 = r0; v2 = r1; }
    else if (KIND == 2) { v0 = v1; v2 = v3; v1 = r0; v3 = r1; }
    else                { v0 = v2; v1 = v3; v2 = r0; v3 = r1; }
}

template <typename T2, typename Hook>
__device__ __forceinline__ void cl_apply_B(T2 *__restrict__ ex, int nbp, const ClIdx &b, const ClEdge<T2> &e, const LeanPh<T2> &P,
                                           uint32_t parK, T2 &v0, T2 &v1, T2 &v2, T2 &v3, Hook &&hook) {
    rot(v0, v2, P.a4); rot(v1, v3, P.b4);
    cl_realign<0, 0>(ex, nbp, b, e, parK, v0, v1, v2, v3, hook);
    rot(v0, v2, P.a3); rot(v1, v3, P.b3);
    rot(v0, v1, P.a2); rot(v2, v3, P.b2);
    cl_realign<1, 1>(ex, nbp, b, e, parK, v0, v1, v2, v3, []() {});
    rot(v0, v1, P.a1); rot(v2, v3, P.b1);
    cl_realign<2, 0>(ex, nbp, b, e, parK, v0, v1, v2, v3, []() {});
    rot(v0, v1, P.a2); rot(v2, v3, P.b2);
    rot(v0, v2, P.a3); rot(v1, v3, P.b3);
    cl_realign<3, 1>(ex, nbp, b, e, parK, v0, v1, v2, v3, []() {});
    rot(v0, v2, P.a4); rot(v1, v3, P.b4);
}


// ------------------------------------------------------------------------------------------------
// grid = Gc * R CTAs in clusters of R (cluster c = blockIdx.x / R owns slices [c*Nt/Gc, (c+1)*Nt/Gc));
// blockDim.x = (h/R)*h rounded up to 32;  h % R == 0.  packed / tab_g as in k_mdagm_stream.
// DOT: part[blockIdx.x] = this CTA's share of sum_t ||w_t||^2.
// ------------------------------------------------------------------------------------------------
template <typename T, bool DOT, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) k_mdagm_cluster(Geo g, const typename PhasePack<T>::word *__restrict__ packed,
                        const double2 *__restrict__ tab_g, const typename Cx<T>::type *__restrict__ in,
                        typename Cx<T>::type *__restrict__ out, T C, double *__restrict__ part, const CgState *__restrict__ st) {
    typedef typename Cx<T>::type T2;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nbp = blockDim.x;
    const int R = (int)cluster_size(), rank = (int)cluster_rank();
    const int hr = g.h / R, nbl = hr * g.h, L = g.L;
    const ClusterSmem<T> lay(L, g.h, R, nbp);
    const double2 *tab = reinterpret_cast<const double2 *>(smem_raw + lay.tab);
    unsigned char *pbuf = smem_raw + lay.pbuf;
    const T2 *vsA = reinterpret_cast<const T2 *>(smem_raw + lay.vbuf), *vsB = reinterpret_cast<const T2 *>(smem_raw + lay.vbuf2);
    T2 *osm = reinterpret_cast<T2 *>(smem_raw + lay.obuf);
    T2 *ex = reinterpret_cast<T2 *>(smem_raw + lay.exch);
    T2 *edge = reinterpret_cast<T2 *>(smem_raw + lay.edge);
    double *red = reinterpret_cast<double *>(smem_raw + lay.red);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + lay.bars);
    uint64_t *bar_v = bars, *bar_v2 = bars + 1, *bar_p = bars + 2, *bar_t = bars + 3, *bar_k0 = bars + 4, *bar_k3 = bars + 5;
    ClIdx b;
    make_cl_idx(g, hr, threadIdx.x, b);
    ClEdge<T2> e;
    e.in_k0 = edge; e.in_k3 = edge + 2 * g.h; e.bar_k0 = bar_k0; e.bar_k3 = bar_k3; e.h = g.h;
    {
        const uint32_t nxt = (rank + 1 == R) ? 0 : rank + 1, prv = (rank == 0) ? R - 1 : rank - 1;
        e.out_k0 = map_to_cta(e.in_k0, nxt); e.rbar_k0 = map_to_cta(bar_k0, nxt);
        e.out_k3 = map_to_cta(e.in_k3, prv); e.rbar_k3 = map_to_cta(bar_k3, prv);
    }
    const int Gc = gridDim.x / R, cid = blockIdx.x / R;
    const int t0 = (int)(((long long)cid * g.Nt) / Gc), t1 = (int)(((long long)(cid + 1) * g.Nt) / Gc);
    const int nsl = t1 - t0;                                         // >= 1 (host: Gc <= Nt)
    // this CTA's part of a slice: site rows row0 .. row0 + 2 hr - 1 (mod L), i.e. n1 rows from row0 and n2 rows from row 0
    const int row0 = 2 * rank * hr + 1, n1 = min(2 * hr, L - row0), n2 = 2 * hr - n1;
    const uint32_t rowb = (uint32_t)L * sizeof(T2), vbytes = (uint32_t)g.Vs * sizeof(T2), part_bytes = (uint32_t)(2 * hr) * rowb;
    const uint32_t pslice = (uint32_t)g.Vs * 16, pj = (uint32_t)nbl * 16;        // packed bytes per slice / per family here
    const unsigned char *in_b = reinterpret_cast<const unsigned char *>(in);
    const unsigned char *pk_b = reinterpret_cast<const unsigned char *>(packed);
    unsigned char *out_b = reinterpret_cast<unsigned char *>(out);
    const bool leader = threadIdx.x == 0;
    auto wrap = [&](int t) { return t >= g.Nt ? t - g.Nt : t; };
    auto load_v = [&](size_t dst_off, int t, uint64_t *bar) {
        mbar_expect_tx(bar, part_bytes);
        bulk_g2s(smem_raw + dst_off, in_b + (size_t)t * vbytes + (size_t)row0 * rowb, (uint32_t)n1 * rowb, bar);
        if (n2 > 0) bulk_g2s(smem_raw + dst_off + (size_t)n1 * rowb, in_b + (size_t)t * vbytes, (uint32_t)n2 * rowb, bar);
    };
    auto load_p = [&](int t) {
        mbar_expect_tx(bar_p, 4 * pj);
        for (int j = 0; j < 4; ++j)
            bulk_g2s(pbuf + (size_t)j * pj, pk_b + (size_t)t * pslice + ((size_t)j * g.nb + (size_t)rank * nbl) * 16, pj, bar_p);
    };
    auto store_o = [&](int t) {
        bulk_s2g(out_b + (size_t)t * vbytes + (size_t)row0 * rowb, osm, (uint32_t)n1 * rowb);
        if (n2 > 0) bulk_s2g(out_b + (size_t)t * vbytes, reinterpret_cast<unsigned char *>(osm) + (size_t)n1 * rowb, (uint32_t)n2 * rowb);
        bulk_commit();
    };
    uint32_t par_vA = 0, par_vB = 0, par_p = 0, parK = 0;
    const int tp = (t0 == 0) ? g.Nt - 1 : t0 - 1;

    if (leader) {
        mbar_init(bar_v, 1); mbar_init(bar_v2, 1); mbar_init(bar_p, 1); mbar_init(bar_t, 1);
        mbar_init(bar_k0, g.h); mbar_init(bar_k3, g.h);
        mbar_fence_init();
        if (sizeof(T) == 8) bulk_load(smem_raw + lay.tab, tab_g, 2 * HQMC_PHASE_TAB * sizeof(double2), bar_t);
        load_v(lay.vbuf, tp, bar_v);
        load_p(tp);
        load_v(lay.vbuf2, t0, bar_v2);
    }
    const int done = (st != nullptr) ? *(volatile const int *)&st->done : 0;
    cluster_sync_all();                   // every CTA's mbarriers are initialised before anyone writes into a neighbour
    if (sizeof(T) == 8) mbar_wait(bar_t, 0);
    if (done) {                           // (the flag is the same for every CTA) drain my copies, then leave together
        mbar_wait(bar_v, 0); mbar_wait(bar_v2, 0); mbar_wait(bar_p, 0);
        return;
    }

    T2 w0, w1, w2, w3;
    LeanPh<T2> P;
    double acc = 0.0;
    const int qd = (b.flags & 1) ? b.q : 0;

    // ---- prologue: w_{t0} = v_{t0} - sigma_{tp} C B_{tp} v_{tp}
    mbar_wait(bar_v, par_vA); par_vA ^= 1;
    mbar_wait(bar_p, par_p); par_p ^= 1;
    load_block_swz(vsA, b, w0, w1, w2, w3);
    lean_load_phases<T>(pbuf, tab, nbl, qd, P);
    cl_apply_B(ex, nbp, b, e, P, parK, w0, w1, w2, w3, [&]() {
        if (leader) { load_v(lay.vbuf, wrap(t0 + 1), bar_v); load_p(t0); }
    });
    parK ^= 1;
    {
        const T sC = (tp == g.Nt - 1) ? C : -C;
        mbar_wait(bar_v2, par_vB); par_vB ^= 1;
        mbar_wait(bar_p, par_p); par_p ^= 1;
        T2 v0, v1, v2, v3;
        load_block_swz(vsB, b, v0, v1, v2, v3);
        w0.x = fma(sC, w0.x, v0.x); w0.y = fma(sC, w0.y, v0.y); w1.x = fma(sC, w1.x, v1.x); w1.y = fma(sC, w1.y, v1.y);
        w2.x = fma(sC, w2.x, v2.x); w2.y = fma(sC, w2.y, v2.y); w3.x = fma(sC, w3.x, v3.x); w3.y = fma(sC, w3.y, v3.y);
        lean_load_phases<T>(pbuf, tab, nbl, qd, P);
    }
    for (int i = 0; i < nsl; ++i) {
        const int t = t0 + i, tn = wrap(t + 1);
        const T sC = (t == g.Nt - 1) ? C : -C;
        const bool more = (i + 1 < nsl), odd = i & 1;
        const T2 *vcur = odd ? vsA : vsB, *vnxt = odd ? vsB : vsA;
        T2 v0, v1, v2, v3;
        load_block_swz(vcur, b, v0, v1, v2, v3);
        cl_apply_B(ex, nbp, b, e, P, parK, v0, v1, v2, v3, [&]() {
            if (leader) {
                if (i > 0) store_o(t - 1);
                if (more) { load_v(odd ? lay.vbuf : lay.vbuf2, wrap(t + 2), odd ? bar_v : bar_v2); load_p(tn); }
            }
        });
        parK ^= 1;
        if (odd) { mbar_wait(bar_v2, par_vB); par_vB ^= 1; } else { mbar_wait(bar_v, par_vA); par_vA ^= 1; }
        T2 n0, n1v, n2v, n3;
        load_block_swz(vnxt, b, n0, n1v, n2v, n3);
        T2 q0, q1, q2, q3;
        q0.x = fma(sC, v0.x, n0.x); q0.y = fma(sC, v0.y, n0.y); q1.x = fma(sC, v1.x, n1v.x); q1.y = fma(sC, v1.y, n1v.y);
        q2.x = fma(sC, v2.x, n2v.x); q2.y = fma(sC, v2.y, n2v.y); q3.x = fma(sC, v3.x, n3.x); q3.y = fma(sC, v3.y, n3.y);
        const T2 k0 = q0, k1 = q1, k2 = q2, k3 = q3;
        if (leader) bulk_wait_read0();
        cl_apply_B(ex, nbp, b, e, P, parK, q0, q1, q2, q3, []() {});
        parK ^= 1;
        if (DOT && (b.flags & 1))
            acc += ((double)w0.x * w0.x + (double)w0.y * w0.y) + ((double)w1.x * w1.x + (double)w1.y * w1.y) +
                   ((double)w2.x * w2.x + (double)w2.y * w2.y) + ((double)w3.x * w3.x + (double)w3.y * w3.y);
        q0.x = fma(sC, q0.x, w0.x); q0.y = fma(sC, q0.y, w0.y); q1.x = fma(sC, q1.x, w1.x); q1.y = fma(sC, q1.y, w1.y);
        q2.x = fma(sC, q2.x, w2.x); q2.y = fma(sC, q2.y, w2.y); q3.x = fma(sC, q3.x, w3.x); q3.y = fma(sC, q3.y, w3.y);
        w0 = k0; w1 = k1; w2 = k2; w3 = k3;
        if (b.flags & 1) store_block_swz(osm, b, q0, q1, q2, q3);
        fence_async_smem();
        if (more) {
            mbar_wait(bar_p, par_p); par_p ^= 1;
            lean_load_phases<T>(pbuf, tab, nbl, qd, P);
        }
    }
    __syncthreads();
    if (leader) { store_o(t1 - 1); bulk_wait0(); }
    if (DOT) {
        double s = block_sum(acc, red);
        if (threadIdx.x == 0) part[blockIdx.x] = s;
    }
    cluster_sync_all();                   // nobody leaves while a neighbour may still write into its shared memory
}

}  // namespace hqmc
