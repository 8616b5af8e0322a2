// mdagm_ws.cuh -- warp-specialised, strip-decoupled streaming O v = M^+ M v kernel (sm_100a).
//
//   w_t = v_t - sigma_{t-1} B_{t-1} v_{t-1};   out_t = w_t - sigma_t B_t w_{t+1}      (Eq.8, 284-314)
//
// Same data mapping as k_mdagm_stream (one CTA per SM owns a run of whole time slices; one thread per 2x2 block of
// sites in registers; packed 8-byte link phases; every global access a TMA bulk copy), but no CTA-wide barrier in
// steady state:
//  * a dedicated PRODUCER warp issues the bulk copies (v two slices deep, links one slice deep) and the staged store
//    of out_t, talking to the compute warps through full/empty mbarriers (the canonical TMA pipeline);
//  * the compute warps are split into horizontal STRIPS of block-rows (L=48: 6 strips of 4 block-rows = 3 warps).
//    The x re-alignments stay inside a block-row, so they only need the strip's named barrier; the y re-alignments
//    cross a strip edge for one block-row per strip, which is passed through a small edge buffer guarded by an
//    mbarrier the sending threads arrive on -- neighbouring strips hand-shake, nobody else waits.  Strips therefore
//    drift apart by up to a sweep stage and the shared-memory, fp64 and barrier phases of different strips overlap
//    instead of alternating in lock step (the limiter of k_mdagm_stream, profiles/r01_*).
#pragma once
#include "mdagm_stream.cuh"

namespace hqmc {

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// strip geometry chosen by the host (ws_geometry): rs block-rows per strip, ns strips
struct WsGeo { int rs, ns, strip_threads; };

__host__ __device__ inline WsGeo ws_geometry(int h, int nbp) {
    WsGeo w;
    for (int rs = 1; rs < h; ++rs)
        if (h % rs == 0 && (rs * h) % 32 == 0 && h / rs <= 15) { w.rs = rs; w.ns = h / rs; w.strip_threads = rs * h; return w; }
    w.rs = h; w.ns = 1; w.strip_threads = nbp;       // one strip = all compute threads (incl. the ragged tail)
    return w;
}

template <typename T> struct WsSmem {
    size_t tab, vbuf[2], pbuf, obuf, exch, edge, red, bars, total;
    __host__ __device__ WsSmem(int Vs, int nbp, int h, int ns) {
        typedef typename Cx<T>::type T2;
        size_t o = 0;
        tab = o;  o += (sizeof(T) == 8) ? (size_t)2 * HQMC_PHASE_TAB * sizeof(double2) : 0;
        vbuf[0] = o; o += (size_t)Vs * sizeof(T2);
        vbuf[1] = o; o += (size_t)Vs * sizeof(T2);
        pbuf = o; o += (size_t)2 * Vs * 8;
        obuf = o; o += (size_t)Vs * sizeof(T2);
        exch = o; o += (size_t)4 * nbp * sizeof(T2);
        edge = o; o += (size_t)2 * ns * 2 * h * sizeof(T2);     // [K0 | K3][strip][slot][bx]
        red = o;  o += 32 * sizeof(double);
        bars = o; o += (size_t)(12 + 2 * ns) * sizeof(uint64_t);
        total = o;
    }
};

// Per-thread exchange description (compute threads); kept to a few 32-bit registers.
template <typename T2> struct WsIdx {
    int o0, o1, o2, o3;           // OO-layout site offsets inside a slice
    int d_yd, d_xd, d_xu, d_yu;   // local exchange destinations
    int q, bx;
    int strips;                   // my strip | next strip << 4 | previous strip << 8
    int flags;                    // bit0 act, bit1 snd_dn, bit2 rcv_dn, bit3 snd_up, bit4 rcv_up
    int strip_threads, h, ns;
    T2 *edge;                     // [K0 | K3][strip][slot][bx]
    uint64_t *ebar;               // [K0 | K3][strip]
    __device__ __forceinline__ bool act() const { return flags & 1; }
};

template <int KIND, int PAR, typename T2>
__device__ __forceinline__ void ws_realign(T2 *__restrict__ ex, int nbp, const WsIdx<T2> &b, uint32_t parK,
                                           T2 &v0, T2 &v1, T2 &v2, T2 &v3) {
    T2 *s0 = ex + (size_t)(PAR * 2) * nbp, *s1 = s0 + nbp;
    const int me = b.strips & 15, nxt = (b.strips >> 4) & 15, prv = (b.strips >> 8) & 15;
    if (KIND == 0) {
        if (b.flags & 2) { T2 *e = b.edge + (nxt * 2) * b.h + b.bx; e[0] = v2; e[b.h] = v3; mbar_arrive(b.ebar + nxt); }
        else { s0[b.d_yd] = v2; s1[b.d_yd] = v3; }
    } else if (KIND == 1) { s0[b.d_xd] = v1; s1[b.d_xd] = v3; }
    else if (KIND == 2)   { s0[b.d_xu] = v0; s1[b.d_xu] = v2; }
    else {
        if (b.flags & 8) { T2 *e = b.edge + ((b.ns + prv) * 2) * b.h + b.bx; e[0] = v0; e[b.h] = v1; mbar_arrive(b.ebar + b.ns + prv); }
        else { s0[b.d_yu] = v0; s1[b.d_yu] = v1; }
    }
    named_bar_sync(me + 1, b.strip_threads);
    T2 r0, r1;
    if (KIND == 0 && (b.flags & 4))       { mbar_wait(b.ebar + me, parK); const T2 *e = b.edge + (me * 2) * b.h + b.bx; r0 = e[0]; r1 = e[b.h]; }
    else if (KIND == 3 && (b.flags & 16)) { mbar_wait(b.ebar + b.ns + me, parK); const T2 *e = b.edge + ((b.ns + me) * 2) * b.h + b.bx; r0 = e[0]; r1 = e[b.h]; }
    else { r0 = s0[b.q]; r1 = s1[b.q]; }
    if (KIND == 0)      { v2 = v0; v3 = v1; v0 = r0; v1 = r1; }
    else if (KIND == 1) { v1 = v0; v3 = v2; v0 = r0; v2 = r1; }
    else if (KIND == 2) { v0 = v1; v2 = v3; v1 = r0; v3 = r1; }
    else                { v0 = v2; v1 = v3; v2 = r0; v3 = r1; }
}

// v <- prod_k (1 + t_k T_k) v, OO layout in and out.  parK: parity of the edge mbarriers for THIS application
// (each is used once per application); the caller flips it afterwards.
template <typename T2>
__device__ __forceinline__ void ws_apply_B(T2 *__restrict__ ex, int nbp, const WsIdx<T2> &b, const LeanPh<T2> &P, uint32_t parK,
                                           T2 &v0, T2 &v1, T2 &v2, T2 &v3) {
    rot(v0, v2, P.a4); rot(v1, v3, P.b4);
    ws_realign<0, 0>(ex, nbp, b, parK, v0, v1, v2, v3);
    rot(v0, v2, P.a3); rot(v1, v3, P.b3);
    rot(v0, v1, P.a2); rot(v2, v3, P.b2);
    ws_realign<1, 1>(ex, nbp, b, parK, v0, v1, v2, v3);
    rot(v0, v1, P.a1); rot(v2, v3, P.b1);
    ws_realign<2, 0>(ex, nbp, b, parK, v0, v1, v2, v3);
    rot(v0, v1, P.a2); rot(v2, v3, P.b2);
    rot(v0, v2, P.a3); rot(v1, v3, P.b3);
    ws_realign<3, 1>(ex, nbp, b, parK, v0, v1, v2, v3);
    rot(v0, v2, P.a4); rot(v1, v3, P.b4);
}


template <typename T2>
__device__ __forceinline__ void make_ws_idx(const Geo &g, int q, const WsGeo &wg, T2 *edge, uint64_t *ebar, WsIdx<T2> &b) {
    const bool act = q < g.nb;
    const int qq = act ? q : 0;
    const int by = qq / g.h, bx = qq - by * g.h, L = g.L;
    const int xa = 2 * bx + 1, xb = (xa + 1 == L) ? 0 : xa + 1;
    const int ya = 2 * by + 1, yb = (ya + 1 == L) ? 0 : ya + 1;
    b.q = q; b.bx = bx;
    b.o0 = ya * L + xa; b.o1 = ya * L + xb; b.o2 = yb * L + xa; b.o3 = yb * L + xb;
    const int byp = (by + 1 == g.h) ? 0 : by + 1, bym = (by == 0) ? g.h - 1 : by - 1;
    const int bxp = (bx + 1 == g.h) ? 0 : bx + 1, bxm = (bx == 0) ? g.h - 1 : bx - 1;
    b.d_yd = act ? bx + g.h * byp : q; b.d_xd = act ? bxp + g.h * by : q;
    b.d_xu = act ? bxm + g.h * by : q; b.d_yu = act ? bx + g.h * bym : q;
    const int me = act ? by / wg.rs : wg.ns - 1;          // the ragged tail (single-strip mode only) joins the last strip
    const int nxt = (me + 1 == wg.ns) ? 0 : me + 1, prv = (me == 0) ? wg.ns - 1 : me - 1;
    b.strips = me | (nxt << 4) | (prv << 8);
    const bool multi = wg.ns > 1;
    const bool first = multi && act && (by % wg.rs == 0), last = multi && act && (by % wg.rs == wg.rs - 1);
    // K0 (y down): the last block-row of a strip sends to the first block-row of the next strip
    // K3 (y up):   the first block-row of a strip sends to the last block-row of the previous strip
    b.flags = (act ? 1 : 0) | (last ? 2 : 0) | (first ? 4 : 0) | (first ? 8 : 0) | (last ? 16 : 0);
    b.strip_threads = wg.strip_threads; b.h = g.h; b.ns = wg.ns;
    b.edge = edge; b.ebar = ebar;
}

// ------------------------------------------------------------------------------------------------
// S5, warp-specialised form.  grid = G CTAs; CTA i owns slices [i*Nt/G, (i+1)*Nt/G);
// blockDim.x = nbp + 32 (nbp = nb rounded up to 32 compute threads, then one producer warp).
// mbarriers: 0 tab | 1,2 full_v | 3 full_p | 4,5 empty_v | 6 empty_p | 7 full_o | 8 empty_o | 12.. edge [K0|K3][strip]
// ------------------------------------------------------------------------------------------------
template <typename T, bool DOT>
__global__ void __launch_bounds__(608, 1) k_mdagm_ws(Geo g, const typename PhasePack<T>::word *__restrict__ packed,
                        const double2 *__restrict__ tab_g, const typename Cx<T>::type *__restrict__ in,
                        typename Cx<T>::type *__restrict__ out, T C, double *__restrict__ part, const CgState *__restrict__ st) {
    typedef typename Cx<T>::type T2;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nbp = blockDim.x - 32, ncw = nbp >> 5;
    const WsGeo wg = ws_geometry(g.h, nbp);
    const WsSmem<T> lay(g.Vs, nbp, g.h, wg.ns);
    const double2 *tab = reinterpret_cast<const double2 *>(smem_raw + lay.tab);
    unsigned char *pbuf = smem_raw + lay.pbuf;
    T2 *osm = reinterpret_cast<T2 *>(smem_raw + lay.obuf);
    T2 *ex = reinterpret_cast<T2 *>(smem_raw + lay.exch);
    double *red = reinterpret_cast<double *>(smem_raw + lay.red);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + lay.bars);
    uint64_t *bar_t = bars, *full_v = bars + 1, *full_p = bars + 3, *emp_v = bars + 4, *emp_p = bars + 6, *full_o = bars + 7,
             *emp_o = bars + 8, *ebar = bars + 12;
    const int G = gridDim.x;
    const int t0 = (int)(((long long)blockIdx.x * g.Nt) / G), t1 = (int)(((long long)(blockIdx.x + 1) * g.Nt) / G);
    if (t0 >= t1) { if (DOT && threadIdx.x == 0) part[blockIdx.x] = 0.0; return; }
    const int nsl = t1 - t0;
    const uint32_t vbytes = (uint32_t)g.Vs * sizeof(T2), pbytes = (uint32_t)g.Vs * 16;
    const unsigned char *in_b = reinterpret_cast<const unsigned char *>(in);
    const unsigned char *pk_b = reinterpret_cast<const unsigned char *>(packed);
    unsigned char *out_b = reinterpret_cast<unsigned char *>(out);
    const int tp = (t0 == 0) ? g.Nt - 1 : t0 - 1;
    const bool producer = (int)threadIdx.x >= nbp;
    const bool issuer = (int)threadIdx.x == nbp;

    if (issuer) {
        mbar_init(bar_t, 1); mbar_init(full_v, 1); mbar_init(full_v + 1, 1); mbar_init(full_p, 1);
        mbar_init(emp_v, ncw); mbar_init(emp_v + 1, ncw); mbar_init(emp_p, ncw); mbar_init(full_o, ncw); mbar_init(emp_o, 1);
        for (int i = 0; i < 2 * wg.ns; ++i) mbar_init(ebar + i, g.h);
        mbar_fence_init();
        if (sizeof(T) == 8) bulk_load(smem_raw + lay.tab, tab_g, 2 * HQMC_PHASE_TAB * sizeof(double2), bar_t);
        bulk_load(smem_raw + lay.vbuf[0], in_b + (size_t)tp * vbytes, vbytes, full_v);
        bulk_load(pbuf, pk_b + (size_t)tp * pbytes, pbytes, full_p);
        bulk_load(smem_raw + lay.vbuf[1], in_b + (size_t)t0 * vbytes, vbytes, full_v + 1);
    }
    const int done = (st != nullptr) ? *(volatile const int *)&st->done : 0;
    __syncthreads();                      // barrier inits visible to every thread
    if (done) {                           // drain the copies aimed at this CTA's shared memory, then leave
        if (sizeof(T) == 8) mbar_wait(bar_t, 0);
        mbar_wait(full_v, 0); mbar_wait(full_v + 1, 0); mbar_wait(full_p, 0);
        return;
    }
    double acc = 0.0;

    if (producer) {
        if (issuer) {
            // links of slice t0 once the halo's links have been decoded by every compute warp
            mbar_wait(emp_p, 0);
            bulk_load(pbuf, pk_b + (size_t)t0 * pbytes, pbytes, full_p);
            uint32_t n_ev[2] = {0, 0}, n_ep = 1, n_fo = 0;     // completed phases consumed so far on each barrier
            for (int i = 0; i < nsl; ++i) {
                const int t = t0 + i, tn = (t + 1 == g.Nt) ? 0 : t + 1, bsel = i & 1;
                // (a) v_{t+1} into the buffer that held v_{t-1} (v_tp for i = 0): released at the top of iteration i-1
                mbar_wait(emp_v + bsel, n_ev[bsel] & 1); ++n_ev[bsel];
                bulk_load(smem_raw + lay.vbuf[bsel], in_b + (size_t)tn * vbytes, vbytes, full_v + bsel);
                // (b) store out_{t-1} as soon as every compute warp has staged it
                if (i > 0) {
                    mbar_wait(full_o, n_fo & 1); ++n_fo;
                    bulk_s2g(out_b + (size_t)(t - 1) * vbytes, osm, vbytes); bulk_commit(); bulk_wait_read0();
                    mbar_arrive(emp_o);
                }
                // (c) links of slice t+1 once the links of slice t have been decoded
                if (i + 1 < nsl) {
                    mbar_wait(emp_p, n_ep & 1); ++n_ep;
                    bulk_load(pbuf, pk_b + (size_t)tn * pbytes, pbytes, full_p);
                }
            }
            mbar_wait(full_o, n_fo & 1);
            bulk_s2g(out_b + (size_t)(t1 - 1) * vbytes, osm, vbytes); bulk_commit(); bulk_wait0();
        }
    } else {
        WsIdx<T2> b;
        make_ws_idx<T2>(g, threadIdx.x, wg, reinterpret_cast<T2 *>(smem_raw + lay.edge), ebar, b);
        const int lane = threadIdx.x & 31;
        const T2 *vs0 = reinterpret_cast<const T2 *>(smem_raw + lay.vbuf[0]), *vs1 = reinterpret_cast<const T2 *>(smem_raw + lay.vbuf[1]);
        uint32_t pfv0 = 0, pfv1 = 0, pfp = 0, peo = 0, parK = 0;
        const int qd = b.act() ? b.q : 0;
        LeanPh<T2> P;
        T2 w0, w1, w2, w3;
        if (sizeof(T) == 8) mbar_wait(bar_t, 0);
        // ---- prologue: w_{t0} = v_{t0} - sigma_{tp} C B_{tp} v_{tp}
        mbar_wait(full_v, pfv0); pfv0 ^= 1;
        mbar_wait(full_p, pfp); pfp ^= 1;
        w0 = vs0[b.o0]; w1 = vs0[b.o1]; w2 = vs0[b.o2]; w3 = vs0[b.o3];
        lean_load_phases<T>(pbuf, tab, g.nb, qd, P);
        __syncwarp();
        if (lane == 0) { mbar_arrive(emp_v); mbar_arrive(emp_p); }
        ws_apply_B(ex, nbp, b, P, parK, w0, w1, w2, w3); parK ^= 1;
        {
            const T sC = (tp == g.Nt - 1) ? C : -C;
            mbar_wait(full_v + 1, pfv1); pfv1 ^= 1;
            mbar_wait(full_p, pfp); pfp ^= 1;
            const T2 v0 = vs1[b.o0], v1 = vs1[b.o1], v2 = vs1[b.o2], v3 = vs1[b.o3];
            w0.x = fma(sC, w0.x, v0.x); w0.y = fma(sC, w0.y, v0.y); w1.x = fma(sC, w1.x, v1.x); w1.y = fma(sC, w1.y, v1.y);
            w2.x = fma(sC, w2.x, v2.x); w2.y = fma(sC, w2.y, v2.y); w3.x = fma(sC, w3.x, v3.x); w3.y = fma(sC, w3.y, v3.y);
            lean_load_phases<T>(pbuf, tab, g.nb, qd, P);
            __syncwarp();
            if (lane == 0) mbar_arrive(emp_p);
        }
        for (int i = 0; i < nsl; ++i) {
            const int t = t0 + i;
            const T sC = (t == g.Nt - 1) ? C : -C;
            const bool more = (i + 1 < nsl);
            const T2 *vcur = (i & 1) ? vs0 : vs1, *vnxt = (i & 1) ? vs1 : vs0;     // v_t sits in buffer (i+1)&1
            T2 v0 = vcur[b.o0], v1 = vcur[b.o1], v2 = vcur[b.o2], v3 = vcur[b.o3];
            __syncwarp();
            if (lane == 0) mbar_arrive(emp_v + ((i + 1) & 1));
            ws_apply_B(ex, nbp, b, P, parK, v0, v1, v2, v3); parK ^= 1;             // B_t v_t / C
            if (i & 1) { mbar_wait(full_v + 1, pfv1); pfv1 ^= 1; } else { mbar_wait(full_v, pfv0); pfv0 ^= 1; }
            const T2 n0 = vnxt[b.o0], n1 = vnxt[b.o1], n2 = vnxt[b.o2], n3 = vnxt[b.o3];   // v_{t+1}
            T2 q0, q1, q2, q3;
            q0.x = fma(sC, v0.x, n0.x); q0.y = fma(sC, v0.y, n0.y); q1.x = fma(sC, v1.x, n1.x); q1.y = fma(sC, v1.y, n1.y);
            q2.x = fma(sC, v2.x, n2.x); q2.y = fma(sC, v2.y, n2.y); q3.x = fma(sC, v3.x, n3.x); q3.y = fma(sC, v3.y, n3.y);
            const T2 k0 = q0, k1 = q1, k2 = q2, k3 = q3;                             // keep w_{t+1}
            ws_apply_B(ex, nbp, b, P, parK, q0, q1, q2, q3); parK ^= 1;             // B_t w_{t+1} / C
            if (DOT && b.act())
                acc += ((double)w0.x * w0.x + (double)w0.y * w0.y) + ((double)w1.x * w1.x + (double)w1.y * w1.y) +
                       ((double)w2.x * w2.x + (double)w2.y * w2.y) + ((double)w3.x * w3.x + (double)w3.y * w3.y);
            q0.x = fma(sC, q0.x, w0.x); q0.y = fma(sC, q0.y, w0.y); q1.x = fma(sC, q1.x, w1.x); q1.y = fma(sC, q1.y, w1.y);
            q2.x = fma(sC, q2.x, w2.x); q2.y = fma(sC, q2.y, w2.y); q3.x = fma(sC, q3.x, w3.x); q3.y = fma(sC, q3.y, w3.y);
            w0 = k0; w1 = k1; w2 = k2; w3 = k3;
            if (i > 0) { mbar_wait(emp_o, peo); peo ^= 1; }                          // the store of out_{t-1} has read obuf
            if (b.act()) { osm[b.o0] = q0; osm[b.o1] = q1; osm[b.o2] = q2; osm[b.o3] = q3; }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(full_o);
            if (more) {
                mbar_wait(full_p, pfp); pfp ^= 1;
                lean_load_phases<T>(pbuf, tab, g.nb, qd, P);
                __syncwarp();
                if (lane == 0) mbar_arrive(emp_p);
            }
        }
    }
    if (DOT) {
        double s = block_sum(acc, red);
        if (threadIdx.x == 0) part[blockIdx.x] = s;
    }
}

}  // namespace hqmc
