// hqmc.cu -- C ABI of libhqmc.so (host orchestration).  See include/hqmc.h.
#include "hqmc_ctx.h"

#include <type_traits>

namespace hqmc {

thread_local std::string g_last_error;

// ---------------------------------------------------------------------------------------------------
// instrumentation + launch wrapper
// ---------------------------------------------------------------------------------------------------
static int drain_events(hqmc_ctx *c) {
    for (auto &ep : c->pending) {
        CUDA_TRY(cudaEventSynchronize(ep.b));
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, ep.a, ep.b));
        c->ms[ep.kclass] += (double)ms;
        c->pool.push_back(ep);
    }
    c->pending.clear();
    return HQMC_OK;
}

template <typename... KArgs, typename... Args>
static int launch(hqmc_ctx *c, int kclass, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, Args... args) {
    const bool use_pdl = c->pdl_next && ((c->pdl >> kclass) & 1);
    c->pdl_next = false;
    if (c->skip_mask & (1u << kclass)) return HQMC_OK;   // leave-one-out timing (results are then meaningless)
    if (c->capturing) c->graph_nodes[kclass]++; else if (c->capturing_md) c->md_nodes_cur[kclass]++; else c->launches[kclass]++;
    const bool prof = c->profiling && !c->capturing && !c->capturing_md;
    EventPair ep{};
    if (prof) {
        if (c->pending.size() >= 2048) HQ_TRY(drain_events(c));
        if (!c->pool.empty()) { ep = c->pool.back(); c->pool.pop_back(); }
        else { CUDA_TRY(cudaEventCreate(&ep.a)); CUDA_TRY(cudaEventCreate(&ep.b)); }
        ep.kclass = kclass;
        CUDA_TRY(cudaEventRecord(ep.a, c->stream));
    }
    if (use_pdl) {
        // programmatic dependent launch: the PCG kernels call griddepcontrol.launch_dependents at their TAIL and
        // griddepcontrol.wait before touching anything the previous kernel wrote, so the launch latency of kernel k+1
        // (and, for M^+M, its barrier set-up and table fetch) hides under kernel k instead of adding to the iteration
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        CUDA_TRY(cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...));
    } else {
        kernel<<<grid, block, smem, c->stream>>>(static_cast<KArgs>(args)...);
        CUDA_TRY(cudaGetLastError());
    }
    if (prof) { CUDA_TRY(cudaEventRecord(ep.b, c->stream)); c->pending.push_back(ep); }
    return HQMC_OK;
}

// Dispatch on (BPT, MAXT): f(integral_constant<int,BPT>, integral_constant<int,MAXT>)
template <typename F> static int with_cfg(const hqmc_ctx *c, F &&f) {
    using std::integral_constant;
    if (c->cfg.bpt == 1 && c->cfg.maxt == 256) return f(integral_constant<int, 1>(), integral_constant<int, 256>());
    if (c->cfg.bpt == 1 && c->cfg.maxt == 576) return f(integral_constant<int, 1>(), integral_constant<int, 576>());
    if (c->cfg.bpt == 2 && c->cfg.maxt == 576) return f(integral_constant<int, 2>(), integral_constant<int, 576>());
    if (c->cfg.bpt == 4 && c->cfg.maxt == 576) return f(integral_constant<int, 4>(), integral_constant<int, 576>());
    g_last_error = "unsupported kernel configuration";
    return HQMC_EINVAL;
}

static size_t block_smem(const hqmc_ctx *c) { return (size_t)4 * c->g.nb * c->esz + 32 * sizeof(double); }
static size_t force_smem(const hqmc_ctx *c) { return block_smem(c) + (size_t)c->g.Vs * sizeof(double); }     // + sin(curl) per site

template <typename T> static int set_attrs(hqmc_ctx *c) {
    const int smem = (int)block_smem(c);
    return with_cfg(c, [&](auto bpt, auto maxt) -> int {
        constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
        const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
        CUDA_TRY(cudaFuncSetAttribute(k_apply_M<T, B, M>, attr, smem));
        CUDA_TRY(cudaFuncSetAttribute(k_apply_B<T, B, M>, attr, smem));
        CUDA_TRY(cudaFuncSetAttribute(k_mdagm<T, B, M, false>, attr, smem));
        CUDA_TRY(cudaFuncSetAttribute(k_mdagm<T, B, M, true>, attr, smem));
        CUDA_TRY(cudaFuncSetAttribute(k_force<T, B, M, false>, attr, (int)force_smem(c)));
        CUDA_TRY(cudaFuncSetAttribute(k_force<T, B, M, true>, attr, (int)force_smem(c)));
        if (c->use_stream) {
            CUDA_TRY(cudaFuncSetAttribute(k_force_stream<T, false>, attr, (int)c->force_stream_smem));
            CUDA_TRY(cudaFuncSetAttribute(k_force_stream<T, true>, attr, (int)c->force_stream_smem));
            CUDA_TRY(cudaFuncSetAttribute(k_mdagm_back<T, false>, attr, (int)c->stream_smem));
            CUDA_TRY(cudaFuncSetAttribute(k_mdagm_back<T, true>, attr, (int)c->stream_smem));
        }
        return HQMC_OK;
    });
}

template <typename T> static int auto_time_tile(hqmc_ctx *c) {
    int per_sm = 1;
    int s = with_cfg(c, [&](auto bpt, auto maxt) -> int {
        constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_mdagm<T, B, M, true>, c->cfg.threads, block_smem(c)));
        return HQMC_OK;
    });
    if (s != HQMC_OK) return s;
    if (per_sm < 1) per_sm = 1;
    int slots = per_sm * c->n_sm;
    int tt = (c->g.Nt + slots - 1) / slots;
    c->time_tile = tt < 1 ? 1 : tt;
    return HQMC_OK;
}

// ---------------------------------------------------------------------------------------------------
// typed operation launchers
// ---------------------------------------------------------------------------------------------------
template <typename T> static int do_phase(hqmc_ctx *c, const double *p, double two_eps) {
    typedef typename Cx<T>::type T2;
    typedef typename PhasePack<T>::word W;
    if (p) HQ_TRY(launch(c, HQMC_K_PHASE, k_phase<T, true>, dim3(c->grid_ew), dim3(256), 0, c->g, c->d_theta, p, two_eps,
                         (T2 *)c->d_ph, c->th_full, c->th_half));
    else HQ_TRY(launch(c, HQMC_K_PHASE, k_phase<T, false>, dim3(c->grid_ew), dim3(256), 0, c->g, c->d_theta, (const double *)nullptr,
                       0.0, (T2 *)c->d_ph, c->th_full, c->th_half));
    if (c->use_stream || c->use_cluster)
        HQ_TRY(launch(c, HQMC_K_PHASE, k_phase_pack<T>, dim3(c->grid_ew), dim3(256), 0, c->g, (const double *)c->d_theta,
                      (W *)c->d_packed, c->th_full, c->th_half));
    return HQMC_OK;
}

template <typename T> static int do_apply_M(hqmc_ctx *c, const void *in, void *out, int dagger) {
    typedef typename Cx<T>::type T2;
    return with_cfg(c, [&](auto bpt, auto maxt) -> int {
        constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
        return launch(c, HQMC_K_M, k_apply_M<T, B, M>, dim3(c->g.Nt), dim3(c->cfg.threads), block_smem(c), c->g,
                      (const T2 *)c->d_ph, (const T2 *)in, (T2 *)out, dagger, (T)c->C);
    });
}

template <typename T> static int do_mdagm_stream(hqmc_ctx *c, const void *in, void *out, bool dot, const CgState *st) {
    typedef typename Cx<T>::type T2;
    typedef typename PhasePack<T>::word W;
    int G = c->time_tile > 0 ? (c->g.Nt + c->time_tile - 1) / c->time_tile : (c->g.Nt < c->n_sm ? c->g.Nt : c->n_sm);
    c->grid_mdagm = G;
    c->pdl_next = true;                               // k_mdagm_back calls griddepcontrol.wait
    if (dot)
        return launch(c, HQMC_K_MDAGM, k_mdagm_back<T, true>, dim3(G), dim3(c->cfg.threads), c->stream_smem, c->g, (const W *)c->d_packed,
                      (const double2 *)c->d_tab, (const T2 *)in, (T2 *)out, (T)c->C, c->d_part_dOd, st);
    return launch(c, HQMC_K_MDAGM, k_mdagm_back<T, false>, dim3(G), dim3(c->cfg.threads), c->stream_smem, c->g, (const W *)c->d_packed,
                  (const double2 *)c->d_tab, (const T2 *)in, (T2 *)out, (T)c->C, (double *)nullptr, st);
}

// cluster launch (cudaLaunchKernelEx with a cluster dimension); same bookkeeping as launch()
template <typename... KArgs, typename... Args>
static int launch_cluster(hqmc_ctx *c, int kclass, void (*kernel)(KArgs...), int grid, int block, size_t smem, int R, Args... args) {
    if (c->skip_mask & (1u << kclass)) return HQMC_OK;
    if (c->capturing) c->graph_nodes[kclass]++; else if (c->capturing_md) c->md_nodes_cur[kclass]++; else c->launches[kclass]++;
    const bool prof = c->profiling && !c->capturing && !c->capturing_md;
    EventPair ep{};
    if (prof) {
        if (c->pending.size() >= 2048) HQ_TRY(drain_events(c));
        if (!c->pool.empty()) { ep = c->pool.back(); c->pool.pop_back(); }
        else { CUDA_TRY(cudaEventCreate(&ep.a)); CUDA_TRY(cudaEventCreate(&ep.b)); }
        ep.kclass = kclass;
        CUDA_TRY(cudaEventRecord(ep.a, c->stream));
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = R; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    CUDA_TRY(cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...));
    if (prof) { CUDA_TRY(cudaEventRecord(ep.b, c->stream)); c->pending.push_back(ep); }
    return HQMC_OK;
}

template <typename T> static int do_mdagm_cluster(hqmc_ctx *c, const void *in, void *out, bool dot, const CgState *st) {
    typedef typename Cx<T>::type T2;
    typedef typename PhasePack<T>::word W;
    const int R = c->cl_R;
    int Gc = c->time_tile > 0 ? (c->g.Nt + c->time_tile - 1) / c->time_tile : (c->g.Nt < c->n_sm / R ? c->g.Nt : c->n_sm / R);
    if (Gc < 1) Gc = 1;
    c->grid_mdagm = Gc * R;
    auto go = [&](auto kern_dot, auto kern_plain) -> int {
        if (dot) {
            CUDA_TRY(cudaFuncSetAttribute(kern_dot, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->cl_smem));
            return launch_cluster(c, HQMC_K_MDAGM, kern_dot, Gc * R, c->cl_threads, c->cl_smem, R, c->g, (const W *)c->d_packed,
                                  (const double2 *)c->d_tab, (const T2 *)in, (T2 *)out, (T)c->C, c->d_part_dOd, st);
        }
        CUDA_TRY(cudaFuncSetAttribute(kern_plain, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->cl_smem));
        return launch_cluster(c, HQMC_K_MDAGM, kern_plain, Gc * R, c->cl_threads, c->cl_smem, R, c->g, (const W *)c->d_packed,
                              (const double2 *)c->d_tab, (const T2 *)in, (T2 *)out, (T)c->C, (double *)nullptr, st);
    };
    if (c->cl_threads <= 512) return go(k_mdagm_cluster<T, true, 512>, k_mdagm_cluster<T, false, 512>);   // 128 registers per thread
    return go(k_mdagm_cluster<T, true, 576>, k_mdagm_cluster<T, false, 576>);
}

template <typename T> static int do_mdagm(hqmc_ctx *c, const void *in, void *out, bool dot, const CgState *st) {
    typedef typename Cx<T>::type T2;
    if (c->use_cluster && c->cluster_on) return do_mdagm_cluster<T>(c, in, out, dot, st);
    if (c->use_stream && c->stream_on) return do_mdagm_stream<T>(c, in, out, dot, st);
    const int Tt = c->time_tile;
    const int grid = (c->g.Nt + Tt - 1) / Tt;
    c->grid_mdagm = grid;
    return with_cfg(c, [&](auto bpt, auto maxt) -> int {
        constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
        if (dot)
            return launch(c, HQMC_K_MDAGM, k_mdagm<T, B, M, true>, dim3(grid), dim3(c->cfg.threads), block_smem(c), c->g, Tt,
                          (const T2 *)c->d_ph, (const T2 *)in, (T2 *)out, (T)c->C, c->d_part_dOd, st, 0, (size_t)0);
        return launch(c, HQMC_K_MDAGM, k_mdagm<T, B, M, false>, dim3(grid), dim3(c->cfg.threads), block_smem(c), c->g, Tt,
                      (const T2 *)c->d_ph, (const T2 *)in, (T2 *)out, (T)c->C, (double *)nullptr, st, 0, (size_t)0);
    });
}

// choose the preconditioner kernel and its grid; fixes the number of <r,z> partials the CG kernels sum.
// tile > 0: TMA-tiled kernel with runs of `tile` slices; tile < 0: register-ring kernel with runs of -tile; 0: default.
static void precond_cfg(hqmc_ctx *c, int tile) {
    const int W = c->taps.W;
    c->pc_smem = 0;
    if (W < 1 || W > 12) { c->pc_kind = 0; c->pc_tile = 0; c->pc_gx = c->grid_ew; c->pc_gy = 1; c->n_part_rz = c->grid_ew; return; }
    const int gx = (c->g.Vs + 127) / 128;
    c->pc_kind = (tile < 0 && W <= 6) ? 1 : 2;           // the register-ring window kernel exists for W <= 6 only
    if (tile < 0) tile = -tile;
    if (tile == 0) {
        // Default: the shortest run whose CTAs are all resident at once (one wave). With the CG vectors L2-resident the halo
        // re-reads are cheap and many small CTAs pipeline better than few large ones; a second wave costs more than either
        // (measured at L=48, Ntau=480: 15 -> 51.3, 16 (two waves) -> 55.5, 24 -> 52.4 us per PCG iteration; profiles/).
        tile = 24;
        for (int tr = 8; tr <= 32; ++tr) {
            const long long nct = (long long)gx * ((c->g.Nt + tr - 1) / tr);
            const size_t per_cta = (size_t)(tr + 2 * W) * 128 * c->esz + 384 + 1024;     // dynamic + static + reserved
            const long long per_sm = std::min<long long>(16, (long long)(233472 / per_cta));
            if (nct <= HQMC_MAX_PART && nct <= per_sm * c->n_sm) { tile = tr; break; }
        }
    }
    if (tile > c->g.Nt) tile = c->g.Nt;
    const int tmax = 108 - 2 * W;                                // tile rows (tile + 2W <= 108) x 128 sites x 16 B <= 216 KB
    if (c->pc_kind == 2 && tile > tmax) tile = tmax;
    while ((long long)gx * ((c->g.Nt + tile - 1) / tile) > HQMC_MAX_PART) ++tile;
    if (c->pc_kind == 2 && tile > tmax) c->pc_kind = W <= 6 ? 1 : 0;
    if (c->pc_kind == 0) { c->pc_tile = 0; c->pc_gx = c->grid_ew; c->pc_gy = 1; c->n_part_rz = c->grid_ew; return; }
    c->pc_tile = tile; c->pc_gx = gx; c->pc_gy = (c->g.Nt + tile - 1) / tile; c->n_part_rz = c->pc_gx * c->pc_gy;
    if (c->pc_kind == 2) c->pc_smem = (size_t)(tile + 2 * W) * 128 * c->esz;
}

template <typename T, int W> static int launch_precond_win(hqmc_ctx *c, const void *in, void *out, double *part_rz, int mode) {
    typedef typename Cx<T>::type T2;
    if (c->pc_kind == 2) {
        c->pdl_next = true;
        CUDA_TRY(cudaFuncSetAttribute(k_precond_tma<T, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->pc_smem));
        return launch(c, HQMC_K_PRECOND, k_precond_tma<T, W>, dim3(c->pc_gx, c->pc_gy), dim3(128), c->pc_smem, c->g, c->taps,
                      (const T2 *)in, (T2 *)out, part_rz, (const double *)c->d_part_rr, c->grid_ew, c->d_state, mode, c->pc_tile);
    }
    return launch(c, HQMC_K_PRECOND, k_precond_win<T, W>, dim3(c->pc_gx, c->pc_gy), dim3(128), 0, c->g, c->taps, (const T2 *)in,
                  (T2 *)out, part_rz, (const double *)c->d_part_rr, c->grid_ew, c->d_state, mode, c->pc_tile);
}

// W = 7..12 (wider than the paper's 1e-3 truncation gives at dtau = 0.1: a solver upgrade):
// TMA-tiled kernel only, with a ring of up to 25 register slots
template <typename T, int W> static int launch_precond_wide(hqmc_ctx *c, const void *in, void *out, double *part_rz, int mode) {
    typedef typename Cx<T>::type T2;
    c->pdl_next = true;
    CUDA_TRY(cudaFuncSetAttribute(k_precond_tma<T, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->pc_smem));
    return launch(c, HQMC_K_PRECOND, k_precond_tma<T, W>, dim3(c->pc_gx, c->pc_gy), dim3(128), c->pc_smem, c->g, c->taps,
                  (const T2 *)in, (T2 *)out, part_rz, (const double *)c->d_part_rr, c->grid_ew, c->d_state, mode, c->pc_tile);
}

template <typename T> static int do_precond(hqmc_ctx *c, const void *in, void *out, double *part_rz, int mode) {
    typedef typename Cx<T>::type T2;
    if (c->pc_kind == 2) {
        switch (c->taps.W) {
            case 7: return launch_precond_wide<T, 7>(c, in, out, part_rz, mode);
            case 8: return launch_precond_wide<T, 8>(c, in, out, part_rz, mode);
            case 9: return launch_precond_wide<T, 9>(c, in, out, part_rz, mode);
            case 10: return launch_precond_wide<T, 10>(c, in, out, part_rz, mode);
            case 11: return launch_precond_wide<T, 11>(c, in, out, part_rz, mode);
            case 12: return launch_precond_wide<T, 12>(c, in, out, part_rz, mode);
            default: break;
        }
    }
    if (c->pc_kind != 0) {
        switch (c->taps.W) {
            case 1: return launch_precond_win<T, 1>(c, in, out, part_rz, mode);
            case 2: return launch_precond_win<T, 2>(c, in, out, part_rz, mode);
            case 3: return launch_precond_win<T, 3>(c, in, out, part_rz, mode);
            case 4: return launch_precond_win<T, 4>(c, in, out, part_rz, mode);
            case 5: return launch_precond_win<T, 5>(c, in, out, part_rz, mode);
            case 6: return launch_precond_win<T, 6>(c, in, out, part_rz, mode);
            default: break;
        }
    }
    return launch(c, HQMC_K_PRECOND, k_precond<T>, dim3(c->grid_ew), dim3(256), 0, c->g, c->taps, (const T2 *)in, (T2 *)out,
                  part_rz, (const double *)c->d_part_rr, c->grid_ew, c->d_state, mode);
}

template <typename T> static int do_force(hqmc_ctx *c, const void *X, double *out, bool fuse_p, double half_eps, int nkick) {
    typedef typename Cx<T>::type T2;
    typedef typename PhasePack<T>::word W;
    if (c->use_stream && c->stream_on) {             // streaming form: one CTA per SM over a run of slices (force_stream.cuh)
        const int G = c->g.Nt < c->n_sm ? c->g.Nt : c->n_sm;
        if (fuse_p)
            return launch(c, HQMC_K_FORCE, k_force_stream<T, true>, dim3(G), dim3(c->cfg.threads), c->force_stream_smem, c->g,
                          (const W *)c->d_packed, (const double2 *)c->d_tab, (const T2 *)c->d_ph, (const T2 *)X, (T)c->C, out,
                          (const double *)c->d_theta, half_eps, c->prm.c_tau, c->prm.K, c->prm.compact, nkick, c->th_full, c->th_half);
        return launch(c, HQMC_K_FORCE, k_force_stream<T, false>, dim3(G), dim3(c->cfg.threads), c->force_stream_smem, c->g,
                      (const W *)c->d_packed, (const double2 *)c->d_tab, (const T2 *)c->d_ph, (const T2 *)X, (T)c->C, out,
                      (const double *)c->d_theta, 0.0, c->prm.c_tau, c->prm.K, c->prm.compact, 0, c->th_full, c->th_half);
    }
    return with_cfg(c, [&](auto bpt, auto maxt) -> int {
        constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
        if (fuse_p)
            return launch(c, HQMC_K_FORCE, k_force<T, B, M, true>, dim3(c->g.Nt), dim3(c->cfg.threads), force_smem(c), c->g,
                          (const T2 *)c->d_ph, (const T2 *)X, (T)c->C, out, (const double *)c->d_theta, half_eps,
                          c->prm.c_tau, c->prm.K, c->prm.compact, nkick, c->th_full, c->th_half);
        return launch(c, HQMC_K_FORCE, k_force<T, B, M, false>, dim3(c->g.Nt), dim3(c->cfg.threads), force_smem(c), c->g,
                      (const T2 *)c->d_ph, (const T2 *)X, (T)c->C, out, (const double *)c->d_theta, 0.0, c->prm.c_tau,
                      c->prm.K, c->prm.compact, 0, c->th_full, c->th_half);
    });
}

#define DISPATCH_T(c, call_d, call_f) ((c)->prm.prec == HQMC_C128 ? (call_d) : (call_f))

static bool aligned16(const void *p) { return p != nullptr && (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace hqmc

using namespace hqmc;

#include "hqmc_api_setup.inl"
#include "hqmc_api_cg.inl"
#include "hqmc_api_cgb.inl"
#include "hqmc_api_md.inl"
#include "hqmc_api_mdb.inl"
#include "hqmc_api_measure.inl"
#include "hqmc_api_slab.inl"
