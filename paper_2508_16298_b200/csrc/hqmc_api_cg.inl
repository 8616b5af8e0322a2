// hqmc_api_cg.inl -- preconditioned CG driver (Eq.20; readings C8, C9).
//
// One iteration = 4 kernels: [O d + <d,Od>] [x,r update + ||r||^2] [z = P r + <r,z> + bookkeeping]
// [d = z + beta d].  All scalars (alpha, beta, convergence flag, iteration count) live on the device,
// so a chunk of iterations is captured ONCE in a CUDA graph and replayed; unlike the
// paper's fixed-count graph every kernel tests the device-side `done` flag and turns
// into a no-op after convergence, so tolerance-based stopping and graph replay coexist.  The host looks
// at the flag once per chunk.

// Deferred-x form (chosen when the loop's live set exceeds the L2): [O d] [r -= alpha Od] [z = P r] [x += alpha d, d = z + beta d].
template <typename T> static int cg_iteration(hqmc_ctx *c, void *x, int par) {
    typedef typename Cx<T>::type T2;
    HQ_TRY(do_mdagm<T>(c, c->d_d, c->d_Od, true, c->d_state));
    // O d is dead once r has been updated, so z = P r is written over it: the iteration's live set is x, r, d, (Od|z) and
    // the packed phases, 88 MB at config 4, and stays largely L2-resident.
    void *zb = c->d_Od;
    if (c->cg_defer_x) {       // x += alpha d rides on the d update: d is streamed once per iteration
        c->pdl_next = true;
        HQ_TRY(launch(c, HQMC_K_AXPY, k_cg_raxpy<T>, dim3(c->grid_ew), dim3(256), 0, c->N, (T2 *)c->d_r, (const T2 *)c->d_Od,
                      (const double *)c->d_part_rz[par], c->n_part_rz, (const double *)c->d_part_dOd, c->grid_mdagm, c->d_part_rr,
                      c->d_state));
        HQ_TRY(do_precond<T>(c, c->d_r, zb, c->d_part_rz[par ^ 1], 2));
        c->pdl_next = true;
        return launch(c, HQMC_K_DUPDATE, k_cg_xdupdate<T>, dim3(c->grid_ew), dim3(256), 0, c->N, (T2 *)x, (T2 *)c->d_d,
                      (const T2 *)zb, (const double *)c->d_part_rz[par ^ 1], (const double *)c->d_part_rz[par], c->n_part_rz,
                      (const double *)c->d_part_dOd, c->grid_mdagm, (const CgState *)c->d_state);
    }
    c->pdl_next = true;
    HQ_TRY(launch(c, HQMC_K_AXPY, k_cg_axpy<T>, dim3(c->grid_ew), dim3(256), 0, c->N, (T2 *)x, (T2 *)c->d_r, (const T2 *)c->d_d,
                  (const T2 *)c->d_Od, (const double *)c->d_part_rz[par], c->n_part_rz, (const double *)c->d_part_dOd,
                  c->grid_mdagm, c->d_part_rr, (const CgState *)c->d_state));
    HQ_TRY(do_precond<T>(c, c->d_r, zb, c->d_part_rz[par ^ 1], 2));
    c->pdl_next = true;
    HQ_TRY(launch(c, HQMC_K_DUPDATE, k_cg_dupdate<T>, dim3(c->grid_ew), dim3(256), 0, c->N, (T2 *)c->d_d, (const T2 *)zb,
                  (const double *)c->d_part_rz[par ^ 1], (const double *)c->d_part_rz[par], c->n_part_rz, 0,
                  (const CgState *)c->d_state));
    return HQMC_OK;
}

template <typename T> static int cg_build_graph(hqmc_ctx *c, void *x) {
    if (c->cg_graph && c->cg_graph_x == x && c->cg_graph_tile == c->time_tile && c->cg_graph_defer == c->cg_defer_x) return HQMC_OK;
    if (c->cg_graph) { cudaGraphExecDestroy(c->cg_graph); c->cg_graph = nullptr; }
    for (int i = 0; i < HQMC_K_COUNT; ++i) c->graph_nodes[i] = 0;
    cudaGraph_t graph = nullptr;
    CUDA_TRY(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed));
    c->capturing = true;
    int st = HQMC_OK;
    for (int i = 0; i < c->cg_chunk && st == HQMC_OK; ++i) st = cg_iteration<T>(c, x, i & 1);
    c->capturing = false;
    cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    if (st != HQMC_OK) { if (graph) cudaGraphDestroy(graph); return st; }
    CUDA_TRY(e);
    e = cudaGraphInstantiate(&c->cg_graph, graph, 0);
    cudaGraphDestroy(graph);
    CUDA_TRY(e);
    c->cfg_epoch++;
    c->cg_graph_x = x;
    c->cg_graph_tile = c->time_tile;
    c->cg_graph_defer = c->cg_defer_x;
    return HQMC_OK;
}

// x_0 = 0, r_0 = rhs, z_0 = P r_0, d_0 = z_0; bookkeeping reset on the device.  Enqueue only.
template <typename T> static int cg_start(hqmc_ctx *c, const void *rhs, void *x, double tol, long long max_iter) {
    typedef typename Cx<T>::type T2;
    HQ_TRY(launch(c, HQMC_K_MISC, k_cg_state_set, dim3(1), dim3(1), 0, c->d_state, tol > 0.0 ? tol * tol : 0.0, max_iter));
    HQ_TRY(launch(c, HQMC_K_MISC, k_cg_init<T>, dim3(c->grid_ew), dim3(256), 0, c->N, (const T2 *)rhs, (T2 *)x, (T2 *)c->d_r,
                  c->d_part_rr));
    HQ_TRY(do_precond<T>(c, c->d_r, c->d_z, c->d_part_rz[0], 1));
    return launch(c, HQMC_K_DUPDATE, k_cg_dupdate<T>, dim3(c->grid_ew), dim3(256), 0, c->N, (T2 *)c->d_d, (const T2 *)c->d_z,
                  (const double *)c->d_part_rz[0], (const double *)c->d_part_rz[0], c->n_part_rz, 1, (const CgState *)c->d_state);
}

// A whole fixed-count solve enqueued without any host round trip: start-up kernels + ceil(max_iter / chunk)
// replays of the chunk graph (its kernels turn into no-ops once the device-side count is reached).  Capturable: inside a
// stream capture the chunk graph becomes a child graph node.  cg_build_graph(c, x) must have been called before.
template <typename T> static int cg_enqueue_fixed(hqmc_ctx *c, const void *rhs, void *x, long long max_iter) {
    HQ_TRY(cg_start<T>(c, rhs, x, 0.0, max_iter));
    const long long nchunk = (max_iter + c->cg_chunk - 1) / c->cg_chunk;
    for (long long k = 0; k < nchunk; ++k) {
        CUDA_TRY(cudaGraphLaunch(c->cg_graph, c->stream));
        for (int i = 0; i < HQMC_K_COUNT; ++i) (c->capturing_md ? c->md_nodes_cur[i] : c->launches[i]) += c->graph_nodes[i];
    }
    return HQMC_OK;
}

// Small lattices (PAPER.md:350's launch-bound regime): the whole solve is ONE cooperative launch of k_pcg_persist.  AUTO takes it
// where an iteration of the four-kernel loop is all launch and drain (measured: profiles/r02_summary.md section 6).
static bool cg_use_persistent(const hqmc_ctx *c) {
    if (!c->persist_ok || c->persist_mode == 1 || c->profiling || c->skip_mask) return false;
    return c->persist_mode == 2 || c->N <= HQMC_PERSIST_AUTO_SITES;
}
template <typename T> static int cg_solve_persistent(hqmc_ctx *c, const void *rhs, void *x, double tol, long long max_iter) {
    typedef typename Cx<T>::type T2;
    CUDA_TRY(cudaMemsetAsync(c->d_ctr, 0, sizeof(unsigned long long) * HQMC_SYNC_WORDS(c->g.Nt), c->stream));
    Geo g = c->g; Taps taps = c->taps; T C = (T)c->C;
    const T2 *ph = (const T2 *)c->d_ph, *b = (const T2 *)rhs;
    T2 *xx = (T2 *)x, *rb = (T2 *)c->d_r, *db = (T2 *)c->d_d;
    double tol2 = tol > 0.0 ? tol * tol : 0.0;
    unsigned long long *ctr = c->d_ctr; CgState *st = c->d_state;
    void *args[] = {&g, &taps, &ph, &b, &xx, &rb, &db, &C, &ctr, &st, &tol2, &max_iter};
    const void *fn = (const void *)k_pcg_persist<T>;
    CUDA_TRY(cudaLaunchCooperativeKernel(fn, dim3(c->g.Nt), dim3(c->cfg.threads), args, c->persist_smem, c->stream));
    c->launches[HQMC_K_MISC]++;
    return HQMC_OK;
}

template <typename T> static int cg_solve_t(hqmc_ctx *c, const void *rhs, void *x, double tol, long long max_iter,
                                            long long *iters_out, double *relres_out) {
    if (cg_use_persistent(c)) {
        const int sp = cg_solve_persistent<T>(c, rhs, x, tol, max_iter);
        if (sp != HQMC_OK) {      // the cooperative launch was refused (e.g. the device is shared): the four-kernel loop from now on
            cudaGetLastError();
            c->persist_ok = false;
            return cg_solve_t<T>(c, rhs, x, tol, max_iter, iters_out, relres_out);
        }
        CUDA_TRY(cudaMemcpyAsync(c->h_state, c->d_state, sizeof(CgState), cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(cudaStreamSynchronize(c->stream));
        const double bb = c->h_state->bb, rr = c->h_state->rr;
        const double rel = bb > 0.0 ? std::sqrt(rr / bb) : 0.0;
        if (iters_out) *iters_out = c->h_state->iters;
        if (relres_out) *relres_out = rel;
        if (rel != rel || (tol > 0.0 && !(rel <= tol))) return HQMC_ENOCONV;
        return HQMC_OK;
    }
    HQ_TRY(cg_start<T>(c, rhs, x, tol, max_iter));
    const bool use_graph = !c->profiling;
    if (use_graph) HQ_TRY(cg_build_graph<T>(c, x));
    long long launched = 0;
    while (true) {
        if (use_graph) {
            CUDA_TRY(cudaGraphLaunch(c->cg_graph, c->stream));
            for (int i = 0; i < HQMC_K_COUNT; ++i) c->launches[i] += c->graph_nodes[i];
        } else {
            for (int i = 0; i < c->cg_chunk; ++i) HQ_TRY(cg_iteration<T>(c, x, i & 1));
        }
        launched += c->cg_chunk;
        CUDA_TRY(cudaMemcpyAsync(c->h_state, c->d_state, sizeof(CgState), cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(cudaStreamSynchronize(c->stream));
        if (c->h_state->done) break;
        if (launched > max_iter + c->cg_chunk) { g_last_error = "CG bookkeeping failed to terminate"; return HQMC_ECUDA; }
    }
    const double bb = c->h_state->bb, rr = c->h_state->rr;
    const double rel = bb > 0.0 ? std::sqrt(rr / bb) : 0.0;
    if (iters_out) *iters_out = c->h_state->iters;
    if (relres_out) *relres_out = rel;
    if (rel != rel || (tol > 0.0 && !(rel <= tol))) return HQMC_ENOCONV;      // also a non-finite residual (x is then meaningless)
    return HQMC_OK;
}

static int cg_solve_any(hqmc_ctx *c, const void *rhs, void *x, double tol, long long max_iter, long long *iters_out,
                        double *relres_out) {
    return DISPATCH_T(c, cg_solve_t<double>(c, rhs, x, tol, max_iter, iters_out, relres_out),
                      cg_solve_t<float>(c, rhs, x, tol, max_iter, iters_out, relres_out));
}

extern "C" int hqmc_cg_solve(hqmc_ctx *c, const void *d_rhs, void *d_x, double tol, long long max_iter, long long *iters_out,
                             double *relres_out) {
    HQ_TRY(check_vec(c, d_rhs, d_x));
    if (max_iter < 0) return HQMC_EINVAL;
    return cg_solve_any(c, d_rhs, d_x, tol, max_iter, iters_out, relres_out);
}
