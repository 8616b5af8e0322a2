// hqmc_api_measure.inl -- C ABI of the stochastic estimator (Eq.17-19; widening row NEXT-2).
// Included by hqmc.cu.

#define CUFFT_TRY(x) do { cufftResult r_ = (x); if (r_ != CUFFT_SUCCESS) { g_last_error = std::string("cuFFT error ") + std::to_string((int)r_) + " at " #x; return HQMC_ECUDA; } } while (0)

// workspace (three lattice vectors) and the 3-D plan over (tau, y, x), created on first use
static int measure_setup(hqmc_ctx *c) {
    if (c->ms_ready) return HQMC_OK;
    const size_t vb = c->N * c->esz;
    void **bufs[3] = {&c->d_ms_a, &c->d_ms_b, &c->d_ms_acc};
    for (auto p : bufs)
        if (!*p) { cudaError_t e = cudaMalloc(p, vb); if (e != cudaSuccess) { g_last_error = std::string("cudaMalloc: ") + cudaGetErrorString(e); return HQMC_ENOMEM; } }
    CUFFT_TRY(cufftPlan3d(&c->ms_plan, c->g.Nt, c->g.L, c->g.L, c->esz == 16 ? CUFFT_Z2Z : CUFFT_C2C));
    c->ms_plan_ok = true;
    CUFFT_TRY(cufftSetStream(c->ms_plan, c->stream));
    c->ms_ready = true;
    return HQMC_OK;
}

template <typename T> static int ms_fft(hqmc_ctx *c, void *inout, int dir) {
    if (sizeof(T) == 8) CUFFT_TRY(cufftExecZ2Z(c->ms_plan, (cufftDoubleComplex *)inout, (cufftDoubleComplex *)inout, dir));
    else CUFFT_TRY(cufftExecC2C(c->ms_plan, (cufftComplex *)inout, (cufftComplex *)inout, dir));
    return HQMC_OK;
}

// D (+)= (1/N^2) F[a]_{-k} F[b]_k with a, b in the workspace (transformed in place); 1/N of Eq.17 times the 1/N cuFFT's
// unnormalised inverse leaves out
template <typename T> static int ms_spectral(hqmc_ctx *c, bool acc, double weight) {
    typedef typename Cx<T>::type T2;
    HQ_TRY(ms_fft<T>(c, c->d_ms_a, CUFFT_FORWARD));
    HQ_TRY(ms_fft<T>(c, c->d_ms_b, CUFFT_FORWARD));
    const T scale = (T)(weight / ((double)c->N * (double)c->N));
    if (acc) return launch(c, HQMC_K_MISC, k_ms_spectral<T, true>, dim3(c->grid_ew), dim3(256), 0, c->g.Nt, c->g.L, (const T2 *)c->d_ms_a,
                           (const T2 *)c->d_ms_b, (T2 *)c->d_ms_acc, scale);
    return launch(c, HQMC_K_MISC, k_ms_spectral<T, false>, dim3(c->grid_ew), dim3(256), 0, c->g.Nt, c->g.L, (const T2 *)c->d_ms_a,
                  (const T2 *)c->d_ms_b, (T2 *)c->d_ms_acc, scale);
}

template <typename T> static int ms_finish(hqmc_ctx *c, void *d_C) {
    HQ_TRY(ms_fft<T>(c, c->d_ms_acc, CUFFT_INVERSE));
    CUDA_TRY(cudaMemcpyAsync(d_C, c->d_ms_acc, c->N * c->esz, cudaMemcpyDeviceToDevice, c->stream));
    return HQMC_OK;
}

template <typename T> static int translation_average_t(hqmc_ctx *c, const void *d_a, const void *d_b, void *d_C) {
    CUDA_TRY(cudaMemcpyAsync(c->d_ms_a, d_a, c->N * c->esz, cudaMemcpyDeviceToDevice, c->stream));
    CUDA_TRY(cudaMemcpyAsync(c->d_ms_b, d_b, c->N * c->esz, cudaMemcpyDeviceToDevice, c->stream));
    HQ_TRY(ms_spectral<T>(c, false, 1.0));
    return ms_finish<T>(c, d_C);
}

template <typename T> static int green_2pt_t(hqmc_ctx *c, const void *d_g, const void *d_xi, int n_rv, void *d_C) {
    typedef typename Cx<T>::type T2;
    for (int k = 0; k < n_rv; ++k) {
        const T2 *g = (const T2 *)d_g + (size_t)k * c->N, *xi = (const T2 *)d_xi + (size_t)k * c->N;
        HQ_TRY(launch(c, HQMC_K_MISC, k_ms_2pt_ab<T>, dim3(c->grid_ew), dim3(256), 0, c->N, g, xi, (T2 *)c->d_ms_a, (T2 *)c->d_ms_b));
        HQ_TRY(ms_spectral<T>(c, k > 0, 1.0 / n_rv));
    }
    return ms_finish<T>(c, d_C);
}

template <typename T> static int pair_correlator_t(hqmc_ctx *c, const void *d_g, const void *d_xi, int n_rv, void *d_C) {
    typedef typename Cx<T>::type T2;
    const double npair = 0.5 * n_rv * (n_rv - 1);
    bool first = true;
    for (int k = 0; k < n_rv; ++k)
        for (int kp = k + 1; kp < n_rv; ++kp) {
            const T2 *g1 = (const T2 *)d_g + (size_t)k * c->N, *g2 = (const T2 *)d_g + (size_t)kp * c->N;
            const T2 *x1 = (const T2 *)d_xi + (size_t)k * c->N, *x2 = (const T2 *)d_xi + (size_t)kp * c->N;
            HQ_TRY(launch(c, HQMC_K_MISC, k_ms_pair_ab<T>, dim3(c->grid_ew), dim3(256), 0, c->N, g1, g2, x1, x2, (T2 *)c->d_ms_a, (T2 *)c->d_ms_b));
            HQ_TRY(ms_spectral<T>(c, !first, 1.0 / npair));
            first = false;
        }
    return ms_finish<T>(c, d_C);
}

extern "C" int hqmc_green_apply(hqmc_ctx *c, const void *d_xi, void *d_g, int n_rv, double tol, long long max_iter,
                                long long *iters_total) {
    if (!c || !c->theta_set || !d_xi || !d_g || d_xi == d_g || n_rv < 1 || max_iter < 0 || !aligned16(d_xi) || !aligned16(d_g)) return HQMC_EINVAL;
    long long total = 0;
    int worst = HQMC_OK;
    int bs = green_batch_size(c, n_rv);
    { const int groups = (n_rv + bs - 1) / bs; bs = (n_rv + groups - 1) / groups; }      // even groups: fewer distinct graphs
    if (bs > 1) {                                  // several vectors per launch (hqmc_api_cgb.inl)
        std::vector<long long> its((size_t)bs);
        for (int k = 0; k < n_rv; k += bs) {
            const int n = std::min(bs, n_rv - k);
            const char *xi = (const char *)d_xi + (size_t)k * c->N * c->esz;
            char *g = (char *)d_g + (size_t)k * c->N * c->esz;
            const int st = DISPATCH_T(c, green_batch_t<double>(c, xi, g, n, tol, max_iter, its.data()),
                                      green_batch_t<float>(c, xi, g, n, tol, max_iter, its.data()));
            for (int b = 0; b < n; ++b) total += its[b];
            if (st == HQMC_ENOCONV) worst = st; else if (st != HQMC_OK) return st;
        }
        if (iters_total) *iters_total = total;
        return worst;
    }
    for (int k = 0; k < n_rv; ++k) {
        const char *xi = (const char *)d_xi + (size_t)k * c->N * c->esz;
        char *g = (char *)d_g + (size_t)k * c->N * c->esz;
        HQ_TRY(DISPATCH_T(c, do_apply_M<double>(c, xi, c->d_phi, 1), do_apply_M<float>(c, xi, c->d_phi, 1)));     // R = M^+ xi
        long long it = 0;
        // solve into the context's own X: the PCG graph (keyed on the solution pointer) is captured once, not once per vector
        const int st = cg_solve_any(c, c->d_phi, c->d_X, tol, max_iter, &it, nullptr);
        CUDA_TRY(cudaMemcpyAsync(g, c->d_X, c->N * c->esz, cudaMemcpyDeviceToDevice, c->stream));
        total += it;
        if (st == HQMC_ENOCONV) worst = st; else if (st != HQMC_OK) return st;
    }
    if (iters_total) *iters_total = total;
    return worst;
}

extern "C" int hqmc_translation_average(hqmc_ctx *c, const void *d_a, const void *d_b, void *d_C) {
    if (!c || !d_a || !d_b || !d_C || !aligned16(d_a) || !aligned16(d_b) || !aligned16(d_C)) return HQMC_EINVAL;
    HQ_TRY(measure_setup(c));
    return DISPATCH_T(c, translation_average_t<double>(c, d_a, d_b, d_C), translation_average_t<float>(c, d_a, d_b, d_C));
}

extern "C" int hqmc_green_2pt(hqmc_ctx *c, const void *d_g, const void *d_xi, int n_rv, void *d_C) {
    if (!c || !d_g || !d_xi || !d_C || n_rv < 1 || !aligned16(d_g) || !aligned16(d_xi) || !aligned16(d_C)) return HQMC_EINVAL;
    HQ_TRY(measure_setup(c));
    return DISPATCH_T(c, green_2pt_t<double>(c, d_g, d_xi, n_rv, d_C), green_2pt_t<float>(c, d_g, d_xi, n_rv, d_C));
}

extern "C" int hqmc_pair_correlator(hqmc_ctx *c, const void *d_g, const void *d_xi, int n_rv, void *d_C) {
    if (!c || !d_g || !d_xi || !d_C || n_rv < 2 || !aligned16(d_g) || !aligned16(d_xi) || !aligned16(d_C)) return HQMC_EINVAL;
    HQ_TRY(measure_setup(c));
    return DISPATCH_T(c, pair_correlator_t<double>(c, d_g, d_xi, n_rv, d_C), pair_correlator_t<float>(c, d_g, d_xi, n_rv, d_C));
}
