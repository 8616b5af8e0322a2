// hqmc_api_cgb.inl -- multi-right-hand-side PCG driver (kernels: cg_batched.cuh; Eq.20).
// Included by hqmc.cu.
//
// n_vec solves advance together: one iteration = 4 launches whose grids carry the vector index, captured cg_chunk at a time
// in a CUDA graph like the one-vector solver.  Every vector has its own device-side state and stops on its
// own residual; the host reads the n_vec states once per chunk and replays until all are done.

static bool cgb_supported(const hqmc_ctx *c) { return c->cfg.bpt == 1 && c->g.Nt <= HQMC_MAX_PART && c->taps.W < c->g.Nt; }

static int cgb_reserve(hqmc_ctx *c, int n) {
    if (n <= c->cgb_cap) return HQMC_OK;
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    if (c->cgb_graph) { cudaGraphExecDestroy(c->cgb_graph); c->cgb_graph = nullptr; }
    void **bufs[] = {&c->d_cgb_r, &c->d_cgb_d, &c->d_cgb_Od, &c->d_cgb_phi, (void **)&c->d_cgb_part, (void **)&c->d_cgb_state,
                     &c->d_cgb_ph, (void **)&c->d_cgb_scal};
    for (auto p : bufs) if (*p) { cudaFree(*p); *p = nullptr; }
    if (c->h_cgb_state) { cudaFreeHost(c->h_cgb_state); c->h_cgb_state = nullptr; }
    if (c->h_cgb_scal) { cudaFreeHost(c->h_cgb_scal); c->h_cgb_scal = nullptr; }
    c->cgb_cap = 0;
    c->cgb_pstride = HQMC_MAX_PART;
    const size_t vb = (size_t)n * c->N * c->esz;
    // d_cgb_phi doubles as the solution X of the chains' trajectories; d_cgb_ph: one link-phase table per chain
    const size_t sizes[] = {vb, vb, vb, vb, sizeof(double) * 5 * (size_t)n * c->cgb_pstride, sizeof(CgState) * (size_t)n, 2 * vb,
                            sizeof(double) * 8 * (size_t)n};
    for (int i = 0; i < 8; ++i) {
        cudaError_t e = cudaMalloc(bufs[i], sizes[i]);
        if (e != cudaSuccess) { g_last_error = std::string("cudaMalloc (batched PCG workspace): ") + cudaGetErrorString(e); return HQMC_ENOMEM; }
    }
    if (cudaMallocHost((void **)&c->h_cgb_state, sizeof(CgState) * (size_t)n) != cudaSuccess) { g_last_error = "cudaMallocHost failed"; return HQMC_ENOMEM; }
    if (cudaMallocHost((void **)&c->h_cgb_scal, sizeof(double) * 8 * (size_t)n) != cudaSuccess) { g_last_error = "cudaMallocHost failed"; return HQMC_ENOMEM; }
    c->cgb_cap = n;
    return HQMC_OK;
}

struct CgbGrids { int ge, gm, tt, pgx, pgy, pbs, ptr, n_rz; };

// resident CTAs per SM of the register-ring preconditioner kernel for half bandwidth W (its ring of 2W+1 rows sets the registers)
template <typename T> static int cgb_precond_occupancy(int W, int bs) {
    int per_sm = 0;
    switch (W) {
#define HQ_CASE(w) case w: cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cgb_precond<T, w>, bs, 0); break;
        HQ_CASE(1) HQ_CASE(2) HQ_CASE(3) HQ_CASE(4) HQ_CASE(5) HQ_CASE(6) HQ_CASE(7) HQ_CASE(8) HQ_CASE(9) HQ_CASE(10) HQ_CASE(11) HQ_CASE(12)
#undef HQ_CASE
        default: break;
    }
    return per_sm > 0 ? per_sm : 4;
}

template <typename T> static int cgb_grids(hqmc_ctx *c, int n, CgbGrids &G) {
    // element-wise kernels: at most eight 256-thread CTAs per SM over the whole batch, so that the batch is ONE wave
    long long ge = (long long)((c->N + 255) / 256), cap = std::max<long long>(4, ((long long)c->n_sm * 8) / n);
    G.ge = (int)std::min<long long>(std::min(ge, cap), HQMC_MAX_PART);
    // M^+M: one CTA per (run of tt slices, vector); tt = the shortest run that keeps the batch in one wave of resident CTAs
    int per_sm = 1;
    HQ_TRY(with_cfg(c, [&](auto bpt, auto maxt) -> int {
        constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_mdagm<T, B, M, true>, c->cfg.threads, block_smem(c)));
        return HQMC_OK;
    }));
    const long long slots = (long long)std::max(per_sm, 1) * c->n_sm;
    long long tt = ((long long)n * c->g.Nt + slots - 1) / slots;
    G.tt = (int)std::min<long long>(std::max<long long>(tt, 1), 16);
    G.gm = (c->g.Nt + G.tt - 1) / G.tt;
    // preconditioner: register-ring kernel for W = 1..12, runs long enough to amortise the 2W halo rows
    const int W = c->taps.W, Vs = c->g.Vs, Nt = c->g.Nt;
    if (W >= 1 && W <= 12) {
        G.pgx = (Vs + 127) / 128;
        G.pbs = (((Vs + G.pgx - 1) / G.pgx) + 31) / 32 * 32;
        // runs just long enough for the whole batch to be ONE wave of resident CTAs (a second wave costs more than the halo)
        const long long slots = (long long)c->n_sm * cgb_precond_occupancy<T>(W, G.pbs);
        long long tr = ((long long)n * G.pgx * Nt + slots - 1) / slots;
        tr = std::min<long long>(std::max<long long>(tr, 2 * W + 1), Nt);
        while ((long long)G.pgx * ((Nt + tr - 1) / tr) > HQMC_MAX_PART) ++tr;
        G.ptr = (int)tr; G.pgy = (Nt + G.ptr - 1) / G.ptr; G.n_rz = G.pgx * G.pgy;
    } else {
        G.pgx = G.ge; G.pgy = 1; G.pbs = 256; G.ptr = 0; G.n_rz = G.ge;
    }
    return HQMC_OK;
}

template <typename T, int W> static int cgb_launch_precond_w(hqmc_ctx *c, int n, const CgbGrids &G, const void *r, void *z, double *part_rz,
                                                             const double *part_rr, int mode) {
    typedef typename Cx<T>::type T2;
    return launch(c, HQMC_K_PRECOND, k_cgb_precond<T, W>, dim3(G.pgx, G.pgy, n), dim3(G.pbs), 0, c->g, c->taps, (const T2 *)r, (T2 *)z,
                  part_rz, part_rr, G.ge, c->cgb_pstride, c->d_cgb_state, mode, G.ptr);
}

template <typename T> static int cgb_precond(hqmc_ctx *c, int n, const CgbGrids &G, const void *r, void *z, double *part_rz,
                                             const double *part_rr, int mode) {
    typedef typename Cx<T>::type T2;
    switch (G.ptr > 0 ? c->taps.W : 0) {
#define HQ_CASE(w) case w: return cgb_launch_precond_w<T, w>(c, n, G, r, z, part_rz, part_rr, mode);
        HQ_CASE(1) HQ_CASE(2) HQ_CASE(3) HQ_CASE(4) HQ_CASE(5) HQ_CASE(6) HQ_CASE(7) HQ_CASE(8) HQ_CASE(9) HQ_CASE(10) HQ_CASE(11) HQ_CASE(12)
#undef HQ_CASE
        default: break;
    }
    return launch(c, HQMC_K_PRECOND, k_cgb_precond_gen<T>, dim3(G.ge, n), dim3(256), 0, c->g, c->taps, (const T2 *)r, (T2 *)z, part_rz,
                  part_rr, G.ge, c->cgb_pstride, c->d_cgb_state, mode);
}

// rows of the partial-sum workspace
static double *cgb_row(hqmc_ctx *c, int row) { return c->d_cgb_part + (size_t)row * c->cgb_cap * c->cgb_pstride; }

template <typename T> static int cgb_iteration(hqmc_ctx *c, int n, const CgbGrids &G, void *x, int par, const void *ph, size_t ph_stride) {
    typedef typename Cx<T>::type T2;
    double *p_dOd = cgb_row(c, 0), *p_rr = cgb_row(c, 1), *p_rz[2] = {cgb_row(c, 2), cgb_row(c, 3)};
    HQ_TRY(with_cfg(c, [&](auto bpt, auto maxt) -> int {
        constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
        return launch(c, HQMC_K_MDAGM, k_mdagm<T, B, M, true>, dim3(G.gm, n), dim3(c->cfg.threads), block_smem(c), c->g, G.tt,
                      (const T2 *)ph, (const T2 *)c->d_cgb_d, (T2 *)c->d_cgb_Od, (T)c->C, p_dOd, (const CgState *)c->d_cgb_state, c->cgb_pstride, ph_stride);
    }));
    HQ_TRY(launch(c, HQMC_K_AXPY, k_cgb_axpy<T>, dim3(G.ge, n), dim3(256), 0, c->N, (T2 *)x, (T2 *)c->d_cgb_r, (const T2 *)c->d_cgb_d,
                  (const T2 *)c->d_cgb_Od, (const double *)p_rz[par], G.n_rz, (const double *)p_dOd, G.gm, p_rr, c->cgb_pstride,
                  (const CgState *)c->d_cgb_state));
    HQ_TRY(cgb_precond<T>(c, n, G, c->d_cgb_r, c->d_cgb_Od, p_rz[par ^ 1], p_rr, 2));     // z over the dead Od
    return launch(c, HQMC_K_DUPDATE, k_cgb_dupdate<T>, dim3(G.ge, n), dim3(256), 0, c->N, (T2 *)c->d_cgb_d, (const T2 *)c->d_cgb_Od,
                  (const double *)p_rz[par ^ 1], (const double *)p_rz[par], G.n_rz, c->cgb_pstride, 0, (const CgState *)c->d_cgb_state);
}

template <typename T> static int cgb_build_graph(hqmc_ctx *c, int n, const CgbGrids &G, void *x, const void *ph, size_t ph_stride) {
    if (c->cgb_graph && c->cgb_graph_x == x && c->cgb_graph_ph == ph && c->cgb_graph_phs == ph_stride && c->cgb_graph_n == n && c->cgb_graph_tt == G.tt && c->cgb_graph_W == c->taps.W) return HQMC_OK;
    if (c->cgb_graph) { cudaGraphExecDestroy(c->cgb_graph); c->cgb_graph = nullptr; }
    long long saved[HQMC_K_COUNT];
    for (int i = 0; i < HQMC_K_COUNT; ++i) { saved[i] = c->graph_nodes[i]; c->graph_nodes[i] = 0; }
    cudaGraph_t graph = nullptr;
    CUDA_TRY(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed));
    c->capturing = true;
    int st = HQMC_OK;
    for (int i = 0; i < c->cg_chunk && st == HQMC_OK; ++i) st = cgb_iteration<T>(c, n, G, x, i & 1, ph, ph_stride);
    c->capturing = false;
    cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    for (int i = 0; i < HQMC_K_COUNT; ++i) { c->cgb_nodes[i] = c->graph_nodes[i]; c->graph_nodes[i] = saved[i]; }
    if (st != HQMC_OK) { if (graph) cudaGraphDestroy(graph); return st; }
    CUDA_TRY(e);
    e = cudaGraphInstantiate(&c->cgb_graph, graph, 0);
    cudaGraphDestroy(graph);
    CUDA_TRY(e);
    c->cgb_graph_x = x; c->cgb_graph_ph = ph; c->cgb_graph_phs = ph_stride; c->cgb_graph_n = n; c->cgb_graph_tt = G.tt; c->cgb_graph_W = c->taps.W;
    return HQMC_OK;
}

// ph / ph_stride: link-phase tables of the batch (stride 0: one gauge field shared by all vectors; 2N: one per vector)
template <typename T> static int cgb_solve_t(hqmc_ctx *c, const void *rhs, void *x, int n, double tol, long long max_iter,
                                             long long *iters_out, double *relres_out, const void *ph = nullptr, size_t ph_stride = 0) {
    if (!ph) ph = c->d_ph;
    typedef typename Cx<T>::type T2;
    HQ_TRY(cgb_reserve(c, n));
    CgbGrids G;
    HQ_TRY(cgb_grids<T>(c, n, G));
    for (int b = 0; b < n; ++b) {
        CgState &s = c->h_cgb_state[b];
        s.bb = 0.0; s.rr = 0.0; s.tol2 = tol > 0.0 ? tol * tol : 0.0; s.iters = 0; s.max_iter = max_iter; s.done = 0; s.pad = 0;
    }
    CUDA_TRY(cudaMemcpyAsync(c->d_cgb_state, c->h_cgb_state, sizeof(CgState) * n, cudaMemcpyHostToDevice, c->stream));
    double *p_rr = cgb_row(c, 1), *p_rz0 = cgb_row(c, 2);
    HQ_TRY(launch(c, HQMC_K_MISC, k_cgb_init<T>, dim3(G.ge, n), dim3(256), 0, c->N, (const T2 *)rhs, (T2 *)x, (T2 *)c->d_cgb_r, p_rr,
                  c->cgb_pstride));
    HQ_TRY(cgb_precond<T>(c, n, G, c->d_cgb_r, c->d_cgb_Od, p_rz0, p_rr, 1));
    HQ_TRY(launch(c, HQMC_K_DUPDATE, k_cgb_dupdate<T>, dim3(G.ge, n), dim3(256), 0, c->N, (T2 *)c->d_cgb_d, (const T2 *)c->d_cgb_Od,
                  (const double *)p_rz0, (const double *)p_rz0, G.n_rz, c->cgb_pstride, 1, (const CgState *)c->d_cgb_state));
    const bool use_graph = !c->profiling;
    if (use_graph) HQ_TRY(cgb_build_graph<T>(c, n, G, x, ph, ph_stride));
    long long launched = 0;
    while (true) {
        if (use_graph) {
            CUDA_TRY(cudaGraphLaunch(c->cgb_graph, c->stream));
            for (int i = 0; i < HQMC_K_COUNT; ++i) c->launches[i] += c->cgb_nodes[i];
        } else {
            for (int i = 0; i < c->cg_chunk; ++i) HQ_TRY(cgb_iteration<T>(c, n, G, x, i & 1, ph, ph_stride));
        }
        launched += c->cg_chunk;
        CUDA_TRY(cudaMemcpyAsync(c->h_cgb_state, c->d_cgb_state, sizeof(CgState) * n, cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(cudaStreamSynchronize(c->stream));
        bool all = true;
        for (int b = 0; b < n; ++b) all = all && c->h_cgb_state[b].done != 0;
        if (all) break;
        if (launched > max_iter + c->cg_chunk) { g_last_error = "batched CG bookkeeping failed to terminate"; return HQMC_ECUDA; }
    }
    int st = HQMC_OK;
    for (int b = 0; b < n; ++b) {
        const double bb = c->h_cgb_state[b].bb, rr = c->h_cgb_state[b].rr;
        const double rel = bb > 0.0 ? std::sqrt(rr / bb) : 0.0;
        if (iters_out) iters_out[b] = c->h_cgb_state[b].iters;
        if (relres_out) relres_out[b] = rel;
        if (rel != rel || (tol > 0.0 && !(rel <= tol))) st = HQMC_ENOCONV;
    }
    return st;
}

extern "C" int hqmc_cg_solve_batched(hqmc_ctx *c, const void *d_rhs, void *d_x, int n_vec, double tol, long long max_iter,
                                     long long *iters_out, double *relres_out) {
    if (!c || !c->theta_set || n_vec < 1 || max_iter < 0 || !aligned16(d_rhs) || !aligned16(d_x) || d_rhs == d_x) return HQMC_EINVAL;
    if (!cgb_supported(c)) { g_last_error = "batched PCG needs L <= 48 (one thread per 2x2 block) and Ntau <= 4096"; return HQMC_EINVAL; }
    return DISPATCH_T(c, cgb_solve_t<double>(c, d_rhs, d_x, n_vec, tol, max_iter, iters_out, relres_out),
                      cgb_solve_t<float>(c, d_rhs, d_x, n_vec, tol, max_iter, iters_out, relres_out));
}

extern "C" int hqmc_set_green_batch(hqmc_ctx *c, int n) {
    if (!c || n < 0) return HQMC_EINVAL;
    c->green_batch = n;
    return HQMC_OK;
}

// vectors solved together by hqmc_green_apply
static int green_batch_size(const hqmc_ctx *c, int n_rv) {
    if (!cgb_supported(c)) return 1;
    if (c->green_batch > 0) return std::min(c->green_batch, n_rv);
    // by footprint: while the live sets (r, d, Od|z per vector; x is streamed) of the whole batch stay L2-resident
    const size_t per_vec = 5 * c->N * c->esz;      // one vector of margin: measured best (L=24: 11 vectors 44.0, 14 vectors 46.4 ps per site)
    const long long fit = (long long)(c->l2_bytes / per_vec);
    return (int)std::max<long long>(1, std::min<long long>(fit, n_rv));
}

// R_k = M^+ xi_k for a batch (k_apply_M with the vector index in blockIdx.y), then the batched solve
template <typename T> static int green_batch_t(hqmc_ctx *c, const void *xi, void *g, int n, double tol, long long max_iter,
                                               long long *iters) {
    typedef typename Cx<T>::type T2;
    HQ_TRY(cgb_reserve(c, n));
    HQ_TRY(with_cfg(c, [&](auto bpt, auto maxt) -> int {
        constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
        return launch(c, HQMC_K_M, k_apply_M<T, B, M>, dim3(c->g.Nt, n), dim3(c->cfg.threads), block_smem(c), c->g, (const T2 *)c->d_ph,
                      (const T2 *)xi, (T2 *)c->d_cgb_phi, 1, (T)c->C);
    }));
    return cgb_solve_t<T>(c, c->d_cgb_phi, g, n, tol, max_iter, iters, nullptr);
}
