// hqmc_api_mdb.inl -- n_chain independent molecular-dynamics trajectories advanced together (Eq.16, 181 Eq.12;
// independent Markov chains are how the method uses more hardware than one lattice fills).
// Included by hqmc.cu.
//
// Chain b has its own gauge field theta_b, momenta p_b and pseudofermion phi_b; all chains share the lattice shape and
// couplings of the context.  Every leapfrog step is the one of hqmc_leapfrog_trajectory, with the chain index in the grid:
// one phase-table launch, one multi-right-hand-side PCG (hqmc_api_cgb.inl, one link-phase table per chain) and one force /
// kick launch for all chains.  On lattices whose kernels cannot fill the GPU the time per step then hardly
// grows with n_chain.  The context's own theta (hqmc_set_theta) is not touched.

template <typename T> static int traj_batched_t(hqmc_ctx *c, double *d_theta, double *d_p, const void *d_pf, int n, int nsteps,
                                                double eps, double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out,
                                                long long *cg_iters_out) {
    typedef typename Cx<T>::type T2;
    HQ_TRY(cgb_reserve(c, n));
    const size_t N = c->N, N2 = 2 * c->N;
    void *X = c->d_cgb_phi;                                   // solutions [n][N]
    std::vector<long long> total((size_t)n, 0), it((size_t)n, 0);
    bool noconv = false;
    // k_phase only needs the position inside a slice: the n fields are n * Ntau slices to it
    Geo gb = c->g; gb.Nt = c->g.Nt * n;
    const int grid_ph = (int)std::min<long long>((long long)((N2 * n + 255) / 256), (long long)c->n_sm * 8);
    auto phase = [&](bool drift) -> int {
        if (drift) return launch(c, HQMC_K_PHASE, k_phase<T, true>, dim3(grid_ph), dim3(256), 0, gb, d_theta, (const double *)d_p,
                                 2.0 * eps, (T2 *)c->d_cgb_ph, c->th_full, c->th_half);
        return launch(c, HQMC_K_PHASE, k_phase<T, false>, dim3(grid_ph), dim3(256), 0, gb, d_theta, (const double *)nullptr, 0.0,
                      (T2 *)c->d_cgb_ph, c->th_full, c->th_half);
    };
    auto solve = [&]() -> int {
        int s = cgb_solve_t<T>(c, d_pf, X, n, cg_tol, cg_max_iter, it.data(), nullptr, c->d_cgb_ph, N2);
        for (int b = 0; b < n; ++b) total[b] += it[b];
        if (s == HQMC_ENOCONV) { noconv = true; return HQMC_OK; }
        return s;
    };
    auto kick = [&](double half_eps, int nkick) -> int {
        return with_cfg(c, [&](auto bpt, auto maxt) -> int {
            constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
            return launch(c, HQMC_K_FORCE, k_force<T, B, M, true>, dim3(c->g.Nt, n), dim3(c->cfg.threads), force_smem(c), c->g,
                          (const T2 *)c->d_cgb_ph, (const T2 *)X, (T)c->C, d_p, (const double *)d_theta, half_eps, c->prm.c_tau,
                          c->prm.K, c->prm.compact, nkick, c->th_full, c->th_half);
        });
    };
    auto energies = [&](int slot0) -> int {
        for (int b = 0; b < n; ++b)
            HQ_TRY(enqueue_energies_at(c, d_theta + b * N2, d_p + b * N2, (const char *)d_pf + b * N * c->esz,
                                       (const char *)X + b * N * c->esz, c->d_cgb_scal + 8 * b + slot0));
        return HQMC_OK;
    };
    CUDA_TRY(cudaMemsetAsync(c->d_cgb_scal, 0, sizeof(double) * 8 * n, c->stream));
    HQ_TRY(phase(false));
    HQ_TRY(solve());
    HQ_TRY(energies(0));                                                      // H0 parts
    for (int k = 0; k < nsteps; ++k) {
        if (k == 0) HQ_TRY(kick(0.5 * eps, 1));                               // p += F(theta_0) eps/2
        HQ_TRY(phase(true));                                                  // theta += 2 p eps
        HQ_TRY(solve());
        HQ_TRY(kick(0.5 * eps, (k == nsteps - 1) ? 1 : 2));                   // closing half kick (+ opening one of step k+1)
    }
    HQ_TRY(energies(3));                                                      // H1 parts
    CUDA_TRY(cudaMemcpyAsync(c->h_cgb_scal, c->d_cgb_scal, sizeof(double) * 8 * n, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    for (int b = 0; b < n; ++b) {
        const double *h = c->h_cgb_scal + 8 * b;
        if (H0_out) H0_out[b] = h[0] + h[1] + h[2];
        if (H1_out) H1_out[b] = h[3] + h[4] + h[5];
        if (cg_iters_out) cg_iters_out[b] = total[b];
    }
    return noconv ? HQMC_ENOCONV : HQMC_OK;
}

extern "C" int hqmc_leapfrog_trajectory_batched(hqmc_ctx *c, double *d_theta, double *d_p, const void *d_pf, int n_chain, int nsteps,
                                                double eps, double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out,
                                                long long *cg_iters_out) {
    if (!c || !aligned16(d_theta) || !aligned16(d_p) || !aligned16(d_pf) || n_chain < 1 || nsteps < 0 || cg_max_iter < 0) return HQMC_EINVAL;
    // the chains are independent: advance them in groups whose PCG live set stays L2-resident (the rule of hqmc_green_apply;
    // hqmc_set_green_batch overrides), which also bounds the workspace
    int bs = cgb_supported(c) ? green_batch_size(c, n_chain) : 1;
    if (bs <= 1) {
        // one vector's live set already fills the L2 (L = 48, Ntau = 480), or the slice needs more than one block per thread
        // (L > 48): the tuned one-chain kernels (TMA streaming / cluster M^+M, tiled preconditioner, PDL) beat a batch of one,
        // so the chains go through hqmc_leapfrog_trajectory one after the other.  The context's own theta is overwritten.
        int worst1 = HQMC_OK;
        for (int k = 0; k < n_chain; ++k) {
            const int st = hqmc_leapfrog_trajectory(c, d_theta + (size_t)k * 2 * c->N, d_p + (size_t)k * 2 * c->N,
                                                    (const char *)d_pf + (size_t)k * c->N * c->esz, nsteps, eps, cg_tol, cg_max_iter,
                                                    H0_out ? H0_out + k : nullptr, H1_out ? H1_out + k : nullptr,
                                                    cg_iters_out ? cg_iters_out + k : nullptr);
            if (st == HQMC_ENOCONV) worst1 = st; else if (st != HQMC_OK) return st;
        }
        c->theta_set = false;                      // the context's phase tables now belong to the last chain
        return worst1;
    }
    { const int groups = (n_chain + bs - 1) / bs; bs = (n_chain + groups - 1) / groups; }   // even groups: fewer distinct graphs
    int worst = HQMC_OK;
    for (int k = 0; k < n_chain; k += bs) {
        const int n = std::min(bs, n_chain - k);
        double *th = d_theta + (size_t)k * 2 * c->N, *p = d_p + (size_t)k * 2 * c->N;
        const void *pf = (const char *)d_pf + (size_t)k * c->N * c->esz;
        double *h0 = H0_out ? H0_out + k : nullptr, *h1 = H1_out ? H1_out + k : nullptr;
        long long *it = cg_iters_out ? cg_iters_out + k : nullptr;
        const int st = DISPATCH_T(c, traj_batched_t<double>(c, th, p, pf, n, nsteps, eps, cg_tol, cg_max_iter, h0, h1, it),
                                  traj_batched_t<float>(c, th, p, pf, n, nsteps, eps, cg_tol, cg_max_iter, h0, h1, it));
        if (st == HQMC_ENOCONV) worst = st; else if (st != HQMC_OK) return st;
    }
    return worst;
}

// phi_b = M^+(theta_b) eta_b for the chains (PAPER.md:185 step i): fills the per-chain phase tables from d_theta first
template <typename T> static int refresh_batched_t(hqmc_ctx *c, const double *d_theta, const void *d_eta, void *d_phi, int n) {
    typedef typename Cx<T>::type T2;
    HQ_TRY(cgb_reserve(c, n));
    Geo gb = c->g; gb.Nt = c->g.Nt * n;
    const int grid_ph = (int)std::min<long long>((long long)((2 * c->N * n + 255) / 256), (long long)c->n_sm * 8);
    HQ_TRY(launch(c, HQMC_K_PHASE, k_phase<T, false>, dim3(grid_ph), dim3(256), 0, gb, const_cast<double *>(d_theta), (const double *)nullptr,
                  0.0, (T2 *)c->d_cgb_ph, c->th_full, c->th_half));
    // the n chains are n * Ntau slices with n antiperiodic wraps: k_apply_M per chain through its grid's y index needs the
    // chain's own phase table, so the chains are launched one by one (once per trajectory)
    for (int b = 0; b < n; ++b)
        HQ_TRY(with_cfg(c, [&](auto bpt, auto maxt) -> int {
            constexpr int B = decltype(bpt)::value, M = decltype(maxt)::value;
            return launch(c, HQMC_K_M, k_apply_M<T, B, M>, dim3(c->g.Nt), dim3(c->cfg.threads), block_smem(c), c->g,
                          (const T2 *)c->d_cgb_ph + (size_t)b * 2 * c->N, (const T2 *)d_eta + (size_t)b * c->N,
                          (T2 *)d_phi + (size_t)b * c->N, 1, (T)c->C);
        }));
    return HQMC_OK;
}

extern "C" int hqmc_refresh_batched(hqmc_ctx *c, const double *d_theta, const void *d_eta, void *d_phi, int n_chain) {
    if (!c || !aligned16(d_theta) || !aligned16(d_eta) || !aligned16(d_phi) || d_eta == d_phi || n_chain < 1) return HQMC_EINVAL;
    if (!cgb_supported(c)) { g_last_error = "batched trajectories need L <= 48 (one thread per 2x2 block) and Ntau <= 4096"; return HQMC_EINVAL; }
    return DISPATCH_T(c, refresh_batched_t<double>(c, d_theta, d_eta, d_phi, n_chain), refresh_batched_t<float>(c, d_theta, d_eta, d_phi, n_chain));
}

// One HQMC update of every chain, steps (i)-(iv) of PAPER.md:185-201, as hqmc_hqmc_step does for one: the random numbers are
// inputs (d_eta, d_p on the device; u on the host, one uniform per chain).  Rejected chains get their theta back.
extern "C" int hqmc_hqmc_step_batched(hqmc_ctx *c, double *d_theta, double *d_p, const void *d_eta, const double *u, int n_chain,
                                      int nsteps, double eps, double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out,
                                      int *accepted_out, long long *cg_iters_out) {
    if (!c || !aligned16(d_theta) || !aligned16(d_p) || !aligned16(d_eta) || !u || n_chain < 1 || nsteps < 0 || cg_max_iter < 0) return HQMC_EINVAL;
    if (!cgb_supported(c) || green_batch_size(c, n_chain) <= 1) {           // see hqmc_leapfrog_trajectory_batched: one chain at a time
        int worst1 = HQMC_OK;
        for (int k = 0; k < n_chain; ++k) {
            const int st = hqmc_hqmc_step(c, d_theta + (size_t)k * 2 * c->N, d_p + (size_t)k * 2 * c->N,
                                          (const char *)d_eta + (size_t)k * c->N * c->esz, u[k], nsteps, eps, cg_tol, cg_max_iter,
                                          H0_out ? H0_out + k : nullptr, H1_out ? H1_out + k : nullptr,
                                          accepted_out ? accepted_out + k : nullptr, cg_iters_out ? cg_iters_out + k : nullptr);
            if (st == HQMC_ENOCONV) worst1 = st; else if (st != HQMC_OK) return st;
        }
        c->theta_set = false;
        return worst1;
    }
    const size_t tb = sizeof(double) * 2 * c->N;
    HQ_TRY(cgb_reserve(c, n_chain));
    // theta_0 of every chain (for the rejections) and the pseudofermions: library-owned, grown on demand
    if (c->cgb_theta0_cap < n_chain) {
        if (c->d_cgb_theta0) { CUDA_TRY(cudaStreamSynchronize(c->stream)); cudaFree(c->d_cgb_theta0); c->d_cgb_theta0 = nullptr; c->cgb_theta0_cap = 0; }
        CUDA_TRY(cudaMalloc((void **)&c->d_cgb_theta0, tb * n_chain));
        c->cgb_theta0_cap = n_chain;
    }
    if (c->d_cgb_pf_cap < n_chain) {
        if (c->d_cgb_pf) { CUDA_TRY(cudaStreamSynchronize(c->stream)); cudaFree(c->d_cgb_pf); c->d_cgb_pf = nullptr; c->d_cgb_pf_cap = 0; }
        CUDA_TRY(cudaMalloc(&c->d_cgb_pf, c->N * c->esz * n_chain));
        c->d_cgb_pf_cap = n_chain;
    }
    CUDA_TRY(cudaMemcpyAsync(c->d_cgb_theta0, d_theta, tb * n_chain, cudaMemcpyDeviceToDevice, c->stream));
    HQ_TRY(hqmc_refresh_batched(c, d_theta, d_eta, c->d_cgb_pf, n_chain));                        // (i)
    std::vector<double> H0((size_t)n_chain), H1((size_t)n_chain);
    int s = hqmc_leapfrog_trajectory_batched(c, d_theta, d_p, c->d_cgb_pf, n_chain, nsteps, eps, cg_tol, cg_max_iter, H0.data(),
                                             H1.data(), cg_iters_out);                                  // (ii)
    if (s != HQMC_OK && s != HQMC_ENOCONV) return s;
    bool any_rej = false;
    for (int b = 0; b < n_chain; ++b) {
        double r = std::exp(H0[b] - H1[b]);
        if (r > 1.0) r = 1.0;
        const int acc = (u[b] < r) ? 1 : 0;                                                             // (iii)
        if (!acc) {                                                                                     // (iv)
            CUDA_TRY(cudaMemcpyAsync(d_theta + (size_t)b * 2 * c->N, c->d_cgb_theta0 + (size_t)b * 2 * c->N, tb, cudaMemcpyDeviceToDevice, c->stream));
            any_rej = true;
        }
        if (H0_out) H0_out[b] = H0[b];
        if (H1_out) H1_out[b] = H1[b];
        if (accepted_out) accepted_out[b] = acc;
    }
    if (any_rej) CUDA_TRY(cudaStreamSynchronize(c->stream));
    return s;
}

// n_updates HQMC updates of n_chain independent chains with every random number drawn on the device: chain b
// is the chain hqmc_sweep would run from seed + b (same counters, key shifted by b), its updates advanced together with the other
// chains' by hqmc_hqmc_step_batched.
extern "C" int hqmc_sweep_batched(hqmc_ctx *c, double *d_theta, unsigned long long seed, unsigned first_update, int n_updates, int n_chain,
                                  int nsteps, double eps, double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out,
                                  int *accepted_out, long long *cg_iters_out) {
    if (!c || !aligned16(d_theta) || n_updates < 0 || n_chain < 1 || nsteps < 0 || cg_max_iter < 0) return HQMC_EINVAL;
    void *d_eta = nullptr; double *d_p = nullptr;
    CUDA_TRY(cudaMalloc(&d_eta, (size_t)n_chain * c->N * c->esz));
    if (cudaMalloc((void **)&d_p, (size_t)n_chain * 2 * c->N * sizeof(double)) != cudaSuccess) { cudaFree(d_eta); g_last_error = "cudaMalloc"; return HQMC_ENOMEM; }
    std::vector<double> u((size_t)n_chain);
    int worst = HQMC_OK, st = HQMC_OK;
    for (int k = 0; k < n_updates && st == HQMC_OK; ++k) {
        const uint32_t upd = (uint32_t)first_update + (uint32_t)k;
        for (int b = 0; b < n_chain && st == HQMC_OK; ++b) {
            const unsigned long long sb = seed + (unsigned long long)b;
            void *eb = (char *)d_eta + (size_t)b * c->N * c->esz;
            if (c->prm.prec == HQMC_C128) st = launch(c, HQMC_K_MISC, k_rng<double, 2>, dim3(rng_grid(c, c->N)), dim3(256), 0, sb, upd, 0u, c->N, eb);
            else st = launch(c, HQMC_K_MISC, k_rng<float, 2>, dim3(rng_grid(c, c->N)), dim3(256), 0, sb, upd, 0u, c->N, eb);
            if (st == HQMC_OK)
                st = launch(c, HQMC_K_MISC, k_rng<double, 1>, dim3(rng_grid(c, c->N)), dim3(256), 0, sb, upd, 1u, c->N, (void *)(d_p + (size_t)b * 2 * c->N));
            u[b] = hqmc_rng_uniform(sb, upd);
        }
        if (st != HQMC_OK) break;
        const size_t o = (size_t)k * n_chain;
        st = hqmc_hqmc_step_batched(c, d_theta, d_p, d_eta, u.data(), n_chain, nsteps, eps, cg_tol, cg_max_iter, H0_out ? H0_out + o : nullptr,
                                    H1_out ? H1_out + o : nullptr, accepted_out ? accepted_out + o : nullptr, cg_iters_out ? cg_iters_out + o : nullptr);
        if (st == HQMC_ENOCONV) { worst = st; st = HQMC_OK; }
    }
    cudaStreamSynchronize(c->stream);
    cudaFree(d_eta); cudaFree(d_p);
    return st != HQMC_OK ? st : worst;
}
