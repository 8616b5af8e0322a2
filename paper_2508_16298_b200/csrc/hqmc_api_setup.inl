// hqmc_api_setup.inl -- context lifetime, preconditioner taps, theta / phase table, operator applies.

static int build_default_taps(hqmc_ctx *c) {
    // reading C10: c_k = [B_pi^k]_00 from the library's own B at pi-flux (fp64), p_m = sum_k c_k c_{k+m}
    const int W = c->prm.precond_W, L = c->g.L, Vs = c->g.Vs;
    c->taps.W = W;
    for (int i = 0; i <= HQMC_MAX_W; ++i) c->taps.p[i] = 0.0;
    if (W == 0) { c->taps.p[0] = 1.0; return HQMC_OK; }
    std::vector<double> th((size_t)2 * Vs, 0.0);
    for (int y = 1; y < L; y += 2)
        for (int x = 0; x < L; ++x) th[(size_t)y * L + x] = M_PI;
    double *d_th = nullptr; double2 *d_ph = nullptr, *d_v[2] = {nullptr, nullptr};
    CUDA_TRY(cudaMalloc(&d_th, sizeof(double) * 2 * Vs));
    CUDA_TRY(cudaMalloc(&d_ph, sizeof(double2) * 2 * Vs));
    CUDA_TRY(cudaMalloc(&d_v[0], sizeof(double2) * Vs));
    CUDA_TRY(cudaMalloc(&d_v[1], sizeof(double2) * Vs));
    CUDA_TRY(cudaMemcpyAsync(d_th, th.data(), sizeof(double) * 2 * Vs, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaMemsetAsync(d_v[0], 0, sizeof(double2) * Vs, c->stream));
    const double one[2] = {1.0, 0.0};
    CUDA_TRY(cudaMemcpyAsync(d_v[0], one, sizeof(one), cudaMemcpyHostToDevice, c->stream));
    Geo g1 = c->g; g1.Nt = 1;
    HQ_TRY(launch(c, HQMC_K_PHASE, k_phase<double, false>, dim3(64), dim3(256), 0, g1, d_th, (const double *)nullptr, 0.0, d_ph,
                  c->th_full, c->th_half));
    const size_t smem = (size_t)4 * c->g.nb * sizeof(double2) + 32 * sizeof(double);
    double ck[HQMC_MAX_W + 1];
    int st = with_cfg(c, [&](auto bpt, auto maxt) -> int {
        constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
        CUDA_TRY(cudaFuncSetAttribute(k_apply_B<double, B, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        for (int k = 0; k <= W; ++k) {
            double v0[2];
            CUDA_TRY(cudaMemcpyAsync(v0, d_v[k & 1], sizeof(v0), cudaMemcpyDeviceToHost, c->stream));
            CUDA_TRY(cudaStreamSynchronize(c->stream));
            ck[k] = v0[0];
            HQ_TRY(launch(c, HQMC_K_MISC, k_apply_B<double, B, M>, dim3(1), dim3(c->cfg.threads), smem, g1, (const double2 *)d_ph,
                          (const double2 *)d_v[k & 1], d_v[(k + 1) & 1], c->C));
        }
        return HQMC_OK;
    });
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    cudaFree(d_th); cudaFree(d_ph); cudaFree(d_v[0]); cudaFree(d_v[1]);
    if (st != HQMC_OK) return st;
    for (int m = 0; m <= W; ++m) {
        double s = 0.0;
        for (int k = 0; k + m <= W; ++k) s += ck[k] * ck[k + m];
        c->taps.p[m] = s;
    }
    return HQMC_OK;
}

extern "C" int hqmc_create(const hqmc_params *prm, void *cuda_stream, hqmc_ctx **out) {
    if (!prm || !out) return HQMC_EINVAL;
    *out = nullptr;
    if (prm->L < 4 || (prm->L & 1) || prm->Ntau < 2 || prm->precond_W < 0 || prm->precond_W > HQMC_MAX_W ||
        prm->precond_W >= prm->Ntau || !(prm->dtau > 0.0) || (prm->prec != HQMC_C128 && prm->prec != HQMC_C64))
        return HQMC_EINVAL;
    const int h = prm->L / 2, nb = h * h;
    if (nb > 2304) { g_last_error = "L too large for the register-blocked kernels (L <= 96)"; return HQMC_EINVAL; }
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    hqmc_ctx *c = new hqmc_ctx();
    c->prm = *prm;
    c->g.L = prm->L; c->g.h = h; c->g.nb = nb; c->g.Vs = prm->L * prm->L; c->g.Nt = prm->Ntau;
    c->N = (size_t)c->g.Vs * c->g.Nt;
    c->esz = (prm->prec == HQMC_C128) ? 16 : 8;
    c->own_stream = (cuda_stream == nullptr);
    c->stream = (cudaStream_t)cuda_stream;
    c->cg_graph = nullptr; c->cg_graph_x = nullptr; c->cg_graph_tile = 0; c->cg_graph_defer = false; c->cg_defer_x = false; c->cg_chunk = 32;
    c->profiling = false; c->capturing = false; c->theta_set = false; c->skip_mask = 0; c->pdl = HQMC_PDL_DEFAULT; c->pdl_next = false;
    for (int i = 0; i < HQMC_K_COUNT; ++i) { c->launches[i] = 0; c->graph_nodes[i] = 0; c->ms[i] = 0.0; }
    int st = HQMC_OK;
    auto fail = [&](int s) { hqmc_destroy(c); return s; };
    if (c->own_stream) {
        // a BLOCKING stream: ordered with the legacy default stream, but capturable into CUDA graphs
        cudaError_t e = cudaStreamCreate(&c->stream);
        if (e != cudaSuccess) { g_last_error = cudaGetErrorString(e); c->stream = nullptr; c->own_stream = false; return fail(HQMC_ECUDA); }
    }
    cudaDeviceProp prop;
    { cudaError_t e = cudaGetDeviceProperties(&prop, dev); if (e != cudaSuccess) { g_last_error = cudaGetErrorString(e); return fail(HQMC_ECUDA); } }
    c->n_sm = prop.multiProcessorCount;
    c->l2_bytes = (size_t)prop.l2CacheSize;
    c->cg_defer_x = cg_defer_default(c);
    if (nb <= 256) c->cfg = {1, 256, 0};
    else if (nb <= 576) c->cfg = {1, 576, 0};
    else if (nb <= 1152) c->cfg = {2, 576, 0};
    else c->cfg = {4, 576, 0};
    c->cfg.threads = (((nb + c->cfg.bpt - 1) / c->cfg.bpt) + 31) / 32 * 32;
    const double a = prm->dtau * prm->t;
    c->C = std::pow(std::cosh(0.5 * a), 6) * std::cosh(a);
    c->th_full = std::tanh(a); c->th_half = std::tanh(0.5 * a);
    long long gew = (long long)((c->N + 255) / 256);
    long long cap = (long long)c->n_sm * 8;
    if (cap > HQMC_MAX_PART) cap = HQMC_MAX_PART;
    c->grid_ew = (int)(gew < cap ? gew : cap);
    c->grid_mdagm = 0;
    const size_t vb = c->N * c->esz, tb = sizeof(double) * 2 * c->N;
#define ALLOC(ptr, bytes)                                                                                         \
    do { cudaError_t e = cudaMalloc((void **)&(ptr), (bytes));                                                    \
         if (e != cudaSuccess) { g_last_error = std::string("cudaMalloc: ") + cudaGetErrorString(e); return fail(HQMC_ENOMEM); } } while (0)
    ALLOC(c->d_theta, tb); ALLOC(c->d_ph, 2 * c->N * c->esz);
    {   // streaming M^+M kernel (k_mdagm_back): one thread per 2x2 block and its staging buffers must fit one SM's shared memory
        const size_t need = (prm->prec == HQMC_C128) ? BackSmem<double>(c->g.Vs, c->cfg.threads).total : BackSmem<float>(c->g.Vs, c->cfg.threads).total;
        c->stream_smem = need;
        c->force_stream_smem = (prm->prec == HQMC_C128) ? ForceSmem<double>(c->g.Vs, c->cfg.threads).total : ForceSmem<float>(c->g.Vs, c->cfg.threads).total;
        c->use_stream = (c->cfg.bpt == 1) && need <= (size_t)prop.sharedMemPerBlockOptin && (size_t)c->g.Vs * 16 < (1u << 20);
        c->stream_on = c->use_stream;
        // cluster kernel: the slice split over R SMs (smallest R whose strip fits one SM's threads and shared memory)
        c->use_cluster = false; c->cluster_on = false; c->cl_R = 0;
        for (int R = 2; R <= 8 && !c->use_cluster; R *= 2) {
            if (h % R) continue;
            const int thr = ((h / R) * h + 31) / 32 * 32;
            const size_t sm = (prm->prec == HQMC_C128) ? ClusterSmem<double>(prm->L, h, R, thr).total : ClusterSmem<float>(prm->L, h, R, thr).total;
            if (thr <= 576 && sm <= (size_t)prop.sharedMemPerBlockOptin && (size_t)c->g.Vs * 16 < (1u << 20)) {
                c->use_cluster = true; c->cl_R = R; c->cl_threads = thr; c->cl_smem = sm;
            }
        }
        c->cluster_on = c->use_cluster && !c->use_stream;      // default only where one SM cannot hold the slice
    }
    if (c->use_stream || c->use_cluster) {
        ALLOC(c->d_packed, 2 * c->N * 8);
        ALLOC(c->d_tab, sizeof(double2) * 2 * HQMC_PHASE_TAB);
        std::vector<double2> tab((size_t)2 * HQMC_PHASE_TAB);
        for (int s2 = 0; s2 < 2; ++s2)
            for (int k = 0; k < HQMC_PHASE_K; ++k) {
                const double ang = 2.0 * M_PI * (double)k / (double)HQMC_PHASE_K, sc = s2 ? c->th_full : c->th_half;
                for (int rep = 0; rep < HQMC_PHASE_REP; ++rep)    // 8 replicas: bank-conflict-free lookups (mdagm_stream.cuh)
                    tab[(size_t)s2 * HQMC_PHASE_TAB + (size_t)k * HQMC_PHASE_REP + rep] = make_double2(sc * std::cos(ang), sc * std::sin(ang));
            }
        cudaError_t e = cudaMemcpy(c->d_tab, tab.data(), sizeof(double2) * tab.size(), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { g_last_error = cudaGetErrorString(e); return fail(HQMC_ECUDA); }
    }
    ALLOC(c->d_r, vb); ALLOC(c->d_z, vb); ALLOC(c->d_d, vb); ALLOC(c->d_Od, vb); ALLOC(c->d_X, vb); ALLOC(c->d_phi, vb);
    ALLOC(c->d_p, tb); ALLOC(c->d_force, tb);
    ALLOC(c->d_part_dOd, sizeof(double) * HQMC_MAX_PART); ALLOC(c->d_part_rr, sizeof(double) * HQMC_MAX_PART);
    ALLOC(c->d_part_rz[0], sizeof(double) * HQMC_MAX_PART); ALLOC(c->d_part_rz[1], sizeof(double) * HQMC_MAX_PART);
    ALLOC(c->d_part_misc, sizeof(double) * HQMC_MAX_PART);
    ALLOC(c->d_state, sizeof(CgState)); ALLOC(c->d_scal, sizeof(double) * 8);
#undef ALLOC
    if (cudaMallocHost((void **)&c->h_state, sizeof(CgState)) != cudaSuccess || cudaMallocHost((void **)&c->h_scal, sizeof(double) * 8) != cudaSuccess) {
        g_last_error = "cudaMallocHost failed"; return fail(HQMC_ENOMEM);
    }
    st = DISPATCH_T(c, set_attrs<double>(c), set_attrs<float>(c));
    if (st != HQMC_OK) return fail(st);
    st = DISPATCH_T(c, auto_time_tile<double>(c), auto_time_tile<float>(c));
    if (st != HQMC_OK) return fail(st);
    if (c->use_stream || c->cluster_on) c->time_tile = 0;
    st = build_default_taps(c);
    if (st != HQMC_OK) return fail(st);
    precond_cfg(c, 0);
    c->pdl = pdl_default(c);
    {   // persistent whole-solve kernel: one CTA per slice, all of them resident at once (cooperative launch)
        int coop = 0, per_sm = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        c->persist_smem = block_smem(c) + 8 * sizeof(double);
        if (coop && c->cfg.bpt == 1 && c->cfg.threads <= 256 && c->g.Nt <= 8 * c->cfg.threads) {
            const void *fn = (prm->prec == HQMC_C128) ? (const void *)k_pcg_persist<double> : (const void *)k_pcg_persist<float>;
            cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, c->cfg.threads, c->persist_smem);
            if (e != cudaSuccess) { per_sm = 0; cudaGetLastError(); }
            c->persist_ok = (long long)per_sm * c->n_sm >= c->g.Nt;
        }
        if (c->persist_ok && cudaMalloc((void **)&c->d_ctr, sizeof(unsigned long long) * HQMC_SYNC_WORDS(c->g.Nt)) != cudaSuccess) { cudaGetLastError(); c->persist_ok = false; }
    }
    *out = c;
    return HQMC_OK;
}

extern "C" int hqmc_destroy(hqmc_ctx *c) {
    if (!c) return HQMC_EINVAL;
    if (c->stream || !c->own_stream) cudaStreamSynchronize(c->stream);
    if (c->cg_graph) cudaGraphExecDestroy(c->cg_graph);
    if (c->cgb_graph) cudaGraphExecDestroy(c->cgb_graph);
    for (auto &m : c->md) if (m.exec) cudaGraphExecDestroy(m.exec);
    { void *bp[] = {c->d_cgb_r, c->d_cgb_d, c->d_cgb_Od, c->d_cgb_phi, c->d_cgb_part, c->d_cgb_state, c->d_cgb_ph, c->d_cgb_scal, c->d_cgb_theta0, c->d_cgb_pf}; for (void *p : bp) if (p) cudaFree(p); }
    if (c->h_cgb_state) cudaFreeHost(c->h_cgb_state);
    if (c->h_cgb_scal) cudaFreeHost(c->h_cgb_scal);
    for (auto &ep : c->pending) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
    for (auto &ep : c->pool) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
    if (c->ms_plan_ok) cufftDestroy(c->ms_plan);
    void *ptrs[] = {c->d_ms_a, c->d_ms_b, c->d_ms_acc, c->d_packed, c->d_tab, c->d_theta, c->d_ph, c->d_r, c->d_z, c->d_d, c->d_Od, c->d_X, c->d_phi, c->d_p, c->d_force, c->d_part_dOd,
                    c->d_part_rr, c->d_part_rz[0], c->d_part_rz[1], c->d_part_misc, c->d_state, c->d_scal, c->d_ctr};
    for (void *p : ptrs) if (p) cudaFree(p);
    if (c->h_state) cudaFreeHost(c->h_state);
    if (c->h_scal) cudaFreeHost(c->h_scal);
    if (c->own_stream && c->stream) cudaStreamDestroy(c->stream);
    delete c;
    return HQMC_OK;
}

extern "C" int hqmc_set_precond(hqmc_ctx *c, int W, const double *taps_host) {
    if (!c || W < 0 || W > HQMC_MAX_W || W >= c->g.Nt || (W > 0 && !taps_host)) return HQMC_EINVAL;
    for (int i = 0; i <= HQMC_MAX_W; ++i) c->taps.p[i] = 0.0;
    c->taps.W = W;
    if (W == 0) c->taps.p[0] = taps_host ? taps_host[0] : 1.0;
    else for (int i = 0; i <= W; ++i) c->taps.p[i] = taps_host[i];
    if (c->cg_graph) { cudaGraphExecDestroy(c->cg_graph); c->cg_graph = nullptr; }   // taps are baked into the graph
    if (c->cgb_graph) { cudaGraphExecDestroy(c->cgb_graph); c->cgb_graph = nullptr; }
    precond_cfg(c, 0);
    return HQMC_OK;
}

extern "C" int hqmc_get_precond(hqmc_ctx *c, int *W_out, double *taps_host) {
    if (!c || !W_out || !taps_host) return HQMC_EINVAL;
    *W_out = c->taps.W;
    for (int i = 0; i <= c->taps.W; ++i) taps_host[i] = c->taps.p[i];
    return HQMC_OK;
}

extern "C" int hqmc_set_theta(hqmc_ctx *c, const double *d_theta) {
    if (!c || !aligned16(d_theta)) return HQMC_EINVAL;
    if (d_theta != c->d_theta)
        CUDA_TRY(cudaMemcpyAsync(c->d_theta, d_theta, sizeof(double) * 2 * c->N, cudaMemcpyDeviceToDevice, c->stream));
    HQ_TRY(DISPATCH_T(c, do_phase<double>(c, nullptr, 0.0), do_phase<float>(c, nullptr, 0.0)));
    c->theta_set = true;
    return HQMC_OK;
}

static int check_vec(hqmc_ctx *c, const void *in, const void *out) {
    if (!c || !aligned16(in) || !aligned16(out) || in == out) return HQMC_EINVAL;
    if (!c->theta_set) { g_last_error = "hqmc_set_theta has not been called"; return HQMC_EINVAL; }
    return HQMC_OK;
}

extern "C" int hqmc_apply_M(hqmc_ctx *c, const void *in, void *out) {
    HQ_TRY(check_vec(c, in, out));
    return DISPATCH_T(c, do_apply_M<double>(c, in, out, 0), do_apply_M<float>(c, in, out, 0));
}
extern "C" int hqmc_apply_Mdag(hqmc_ctx *c, const void *in, void *out) {
    HQ_TRY(check_vec(c, in, out));
    return DISPATCH_T(c, do_apply_M<double>(c, in, out, 1), do_apply_M<float>(c, in, out, 1));
}
extern "C" int hqmc_apply_MdagM(hqmc_ctx *c, const void *in, void *out) {
    HQ_TRY(check_vec(c, in, out));
    return DISPATCH_T(c, do_mdagm<double>(c, in, out, false, nullptr), do_mdagm<float>(c, in, out, false, nullptr));
}
extern "C" int hqmc_precond(hqmc_ctx *c, const void *in, void *out) {
    if (!c || !aligned16(in) || !aligned16(out) || in == out) return HQMC_EINVAL;
    return DISPATCH_T(c, do_precond<double>(c, in, out, nullptr, 0), do_precond<float>(c, in, out, nullptr, 0));
}

extern "C" int hqmc_set_profiling(hqmc_ctx *c, int on) {
    if (!c) return HQMC_EINVAL;
    HQ_TRY(drain_events(c));
    c->profiling = on != 0;
    return HQMC_OK;
}
extern "C" int hqmc_reset_stats(hqmc_ctx *c) {
    if (!c) return HQMC_EINVAL;
    HQ_TRY(drain_events(c));
    for (int i = 0; i < HQMC_K_COUNT; ++i) { c->launches[i] = 0; c->ms[i] = 0.0; }
    return HQMC_OK;
}
extern "C" int hqmc_get_kernel_stats(hqmc_ctx *c, int which, long long *launches_out, double *ms_out) {
    if (!c || which < 0 || which >= HQMC_K_COUNT) return HQMC_EINVAL;
    HQ_TRY(drain_events(c));
    if (launches_out) *launches_out = c->launches[which];
    if (ms_out) *ms_out = c->ms[which];
    return HQMC_OK;
}
extern "C" int hqmc_set_time_tile(hqmc_ctx *c, int tt) {
    if (!c || tt < 0 || tt > c->g.Nt) return HQMC_EINVAL;
    if (tt == 0) {
        if ((c->use_stream && c->stream_on) || c->cluster_on) { c->time_tile = 0; return HQMC_OK; }   // one CTA per SM, slices dealt out evenly
        return DISPATCH_T(c, auto_time_tile<double>(c), auto_time_tile<float>(c));
    }
    if ((c->g.Nt + tt - 1) / tt > HQMC_MAX_PART) return HQMC_EINVAL;
    c->time_tile = tt;
    return HQMC_OK;
}
extern "C" int hqmc_set_precond_tile(hqmc_ctx *c, int slices_per_run) {
    if (!c) return HQMC_EINVAL;
    if (c->cg_graph) { cudaGraphExecDestroy(c->cg_graph); c->cg_graph = nullptr; }
    precond_cfg(c, slices_per_run);
    return HQMC_OK;
}
extern "C" int hqmc_set_debug_skip(hqmc_ctx *c, unsigned mask) {
    if (!c) return HQMC_EINVAL;
    c->skip_mask = mask;
    if (c->cg_graph) { cudaGraphExecDestroy(c->cg_graph); c->cg_graph = nullptr; }
    if (c->cgb_graph) { cudaGraphExecDestroy(c->cgb_graph); c->cgb_graph = nullptr; }
    return HQMC_OK;
}
extern "C" int hqmc_set_pdl(hqmc_ctx *c, int on) {
    if (!c) return HQMC_EINVAL;
    c->pdl = on == 1 ? pdl_default(c) : (on >= 16 ? (on & 15) : 0);     // >= 16: per-class mask (timing experiments)
    if (c->cg_graph) { cudaGraphExecDestroy(c->cg_graph); c->cg_graph = nullptr; }
    return HQMC_OK;
}
extern "C" int hqmc_set_md_graph(hqmc_ctx *c, int on) {
    if (!c) return HQMC_EINVAL;
    c->md_graph = on != 0;
    return HQMC_OK;
}
extern "C" int hqmc_set_cg_persistent(hqmc_ctx *c, int mode) {
    if (!c || mode < 0 || mode > 2) return HQMC_EINVAL;
    if (mode == HQMC_PERSIST_ON && !c->persist_ok) { g_last_error = "the persistent PCG kernel cannot run this lattice (one 2x2 block per thread, all Ntau CTAs resident)"; return HQMC_EINVAL; }
    c->persist_mode = mode;
    return HQMC_OK;
}

extern "C" int hqmc_set_cg_variant(hqmc_ctx *c, int which) {
    if (!c || which < HQMC_CG_AUTO || which > HQMC_CG_DEFERRED_X) return HQMC_EINVAL;
    c->cg_defer_x = which == HQMC_CG_DEFERRED_X || (which == HQMC_CG_AUTO && cg_defer_default(c));
    if (c->cg_graph) { cudaGraphExecDestroy(c->cg_graph); c->cg_graph = nullptr; }
    return HQMC_OK;
}
extern "C" int hqmc_set_mdagm_kernel(hqmc_ctx *c, int which) {
    if (!c || which < HQMC_MDAGM_AUTO || which > HQMC_MDAGM_STREAM) return HQMC_EINVAL;
    if ((which == HQMC_MDAGM_CLUSTER && !c->use_cluster) || (which == HQMC_MDAGM_STREAM && !c->use_stream)) return HQMC_EINVAL;
    c->stream_on = which == HQMC_MDAGM_STREAM || (which == HQMC_MDAGM_AUTO && c->use_stream);
    c->cluster_on = which == HQMC_MDAGM_CLUSTER || (which == HQMC_MDAGM_AUTO && c->use_cluster && !c->use_stream);
    if (c->cg_graph) { cudaGraphExecDestroy(c->cg_graph); c->cg_graph = nullptr; }
    return hqmc_set_time_tile(c, 0);
}

extern "C" const char *hqmc_strerror(int s) {
    switch (s) {
        case HQMC_OK: return "ok";
        case HQMC_EINVAL: return "invalid argument";
        case HQMC_ECUDA: return "CUDA error";
        case HQMC_ENOCONV: return "CG did not converge within max_iter";
        case HQMC_ENOMEM: return "out of device memory";
        default: return "unknown status";
    }
}
extern "C" const char *hqmc_last_error(void) { return g_last_error.c_str(); }
extern "C" int hqmc_version(void) { return 100; }
