// hqmc_api_md.inl -- forces, energies, leapfrog trajectory (Eq.12, 207-214 Eq.16) and the
// host-buffer entry points.

extern "C" int hqmc_force(hqmc_ctx *c, const void *d_x, double *d_out) {
    if (!c || !aligned16(d_x) || !aligned16(d_out)) return HQMC_EINVAL;
    if (!c->theta_set) { g_last_error = "hqmc_set_theta has not been called"; return HQMC_EINVAL; }
    return DISPATCH_T(c, do_force<double>(c, d_x, d_out, false, 0.0, 0), do_force<float>(c, d_x, d_out, false, 0.0, 0));
}

extern "C" int hqmc_force_boson(hqmc_ctx *c, double *d_out) {
    if (!c || !aligned16(d_out)) return HQMC_EINVAL;
    if (!c->theta_set) { g_last_error = "hqmc_set_theta has not been called"; return HQMC_EINVAL; }
    return launch(c, HQMC_K_MISC, k_force_boson, dim3(c->grid_ew), dim3(256), 0, c->g, (const double *)c->d_theta, d_out,
                  c->prm.c_tau, c->prm.K, c->prm.compact);
}

// enqueue the reductions for the gauge field d_theta: d_out[0..2] = S_B, sum p^2, S_F = Re <phi, x>
static int enqueue_energies_at(hqmc_ctx *c, const double *d_theta, const double *d_p, const void *d_phi, const void *d_x, double *d_out) {
    HQ_TRY(launch(c, HQMC_K_MISC, k_action_boson, dim3(c->grid_ew), dim3(256), 0, c->g, d_theta, c->prm.c_tau,
                  c->prm.K, c->prm.compact, c->d_part_misc));
    HQ_TRY(launch(c, HQMC_K_MISC, k_final_sum, dim3(1), dim3(32), 0, (const double *)c->d_part_misc, c->grid_ew, d_out));
    if (d_p) {
        HQ_TRY(launch(c, HQMC_K_MISC, k_reduce<double>, dim3(c->grid_ew), dim3(256), 0, 0, (size_t)2 * c->N, (const void *)d_p,
                      (const void *)nullptr, c->d_part_misc));
        HQ_TRY(launch(c, HQMC_K_MISC, k_final_sum, dim3(1), dim3(32), 0, (const double *)c->d_part_misc, c->grid_ew, d_out + 1));
    }
    if (d_phi && d_x) {
        if (c->prm.prec == HQMC_C128)
            HQ_TRY(launch(c, HQMC_K_MISC, k_reduce<double>, dim3(c->grid_ew), dim3(256), 0, 1, c->N, d_phi, d_x, c->d_part_misc));
        else
            HQ_TRY(launch(c, HQMC_K_MISC, k_reduce<float>, dim3(c->grid_ew), dim3(256), 0, 1, c->N, d_phi, d_x, c->d_part_misc));
        HQ_TRY(launch(c, HQMC_K_MISC, k_final_sum, dim3(1), dim3(32), 0, (const double *)c->d_part_misc, c->grid_ew, d_out + 2));
    }
    return HQMC_OK;
}
// at the context's theta; results land in c->d_scal[slot0 .. slot0 + 2]
static int enqueue_energies(hqmc_ctx *c, const double *d_p, const void *d_phi, const void *d_x, int slot0) {
    return enqueue_energies_at(c, c->d_theta, d_p, d_phi, d_x, c->d_scal + slot0);
}

extern "C" int hqmc_energies(hqmc_ctx *c, const double *d_p, const void *d_phi, const void *d_x, double *SB, double *p2, double *SF) {
    if (!c) return HQMC_EINVAL;
    if (!c->theta_set) { g_last_error = "hqmc_set_theta has not been called"; return HQMC_EINVAL; }
    CUDA_TRY(cudaMemsetAsync(c->d_scal, 0, sizeof(double) * 8, c->stream));
    HQ_TRY(enqueue_energies(c, d_p, d_phi, d_x, 0));
    CUDA_TRY(cudaMemcpyAsync(c->h_scal, c->d_scal, sizeof(double) * 8, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    if (SB) *SB = c->h_scal[0];
    if (p2) *p2 = c->h_scal[1];
    if (SF) *SF = c->h_scal[2];
    return HQMC_OK;
}

static int kick(hqmc_ctx *c, double *d_p, double half_eps, int nkick) {
    return DISPATCH_T(c, do_force<double>(c, c->d_X, d_p, true, half_eps, nkick), do_force<float>(c, c->d_X, d_p, true, half_eps, nkick));
}

// Leapfrog step as ONE CUDA graph ("CUDA graph for the whole fermionic force computation"; north_star (b)):
// drift + link-phase rebuild, a whole fixed-count PCG solve (start-up kernels + the chunk graph as child graph
// nodes) and the fused force + kick.  which = 0: a middle step (closing half kick + opening one of the next step),
// which = 1: the last step.  Only for fixed-count solves: a tolerance stop needs the host to look at the flag.
template <typename T> static int md_step_enqueue(hqmc_ctx *c, double *d_p, const void *d_pf, double eps, long long iters, int nkick) {
    HQ_TRY(do_phase<T>(c, d_p, 2.0 * eps));                                  // theta += 2 p eps
    HQ_TRY(cg_enqueue_fixed<T>(c, d_pf, c->d_X, iters));
    return do_force<T>(c, c->d_X, d_p, true, 0.5 * eps, nkick);
}
static int md_graph_get(hqmc_ctx *c, int which, double *d_p, const void *d_pf, double eps, long long iters) {
    HQ_TRY(DISPATCH_T(c, cg_build_graph<double>(c, c->d_X), cg_build_graph<float>(c, c->d_X)));     // before the capture
    hqmc_ctx::MdGraph &m = c->md[which];
    if (m.exec && m.p == d_p && m.pf == d_pf && m.eps == eps && m.iters == iters && m.epoch == c->cfg_epoch) return HQMC_OK;
    if (m.exec) { cudaGraphExecDestroy(m.exec); m.exec = nullptr; }
    for (int i = 0; i < HQMC_K_COUNT; ++i) m.nodes[i] = 0;
    cudaGraph_t graph = nullptr;
    CUDA_TRY(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed));
    c->capturing_md = true; c->md_nodes_cur = m.nodes;
    const int nkick = which ? 1 : 2;
    int st = DISPATCH_T(c, md_step_enqueue<double>(c, d_p, d_pf, eps, iters, nkick), md_step_enqueue<float>(c, d_p, d_pf, eps, iters, nkick));
    c->capturing_md = false; c->md_nodes_cur = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    if (st != HQMC_OK || e != cudaSuccess) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return st != HQMC_OK ? st : HQMC_ECUDA; }
    e = cudaGraphInstantiate(&m.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { m.exec = nullptr; cudaGetLastError(); return HQMC_ECUDA; }
    m.p = d_p; m.pf = d_pf; m.eps = eps; m.iters = iters; m.epoch = c->cfg_epoch;
    return HQMC_OK;
}

extern "C" int hqmc_leapfrog_trajectory(hqmc_ctx *c, double *d_theta, double *d_p, const void *d_pf, int nsteps, double eps,
                                        double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out,
                                        long long *cg_iters_out) {
    if (!c || !aligned16(d_theta) || !aligned16(d_p) || !aligned16(d_pf) || nsteps < 0 || cg_max_iter < 0) return HQMC_EINVAL;
    long long total = 0, it = 0;
    bool noconv = false;
    auto solve = [&]() -> int {
        if (cg_tol <= 0.0 && cg_use_persistent(c)) {                        // fixed count on a small lattice: one launch, no host round trip
            total += cg_max_iter;
            return DISPATCH_T(c, cg_solve_persistent<double>(c, d_pf, c->d_X, 0.0, cg_max_iter), cg_solve_persistent<float>(c, d_pf, c->d_X, 0.0, cg_max_iter));
        }
        int s = cg_solve_any(c, d_pf, c->d_X, cg_tol, cg_max_iter, &it, nullptr);
        total += it;
        if (s == HQMC_ENOCONV) { noconv = true; return HQMC_OK; }
        return s;
    };
    HQ_TRY(hqmc_set_theta(c, d_theta));
    CUDA_TRY(cudaMemsetAsync(c->d_scal, 0, sizeof(double) * 8, c->stream));
    HQ_TRY(solve());
    HQ_TRY(enqueue_energies(c, d_p, d_pf, c->d_X, 0));                      // H0 parts -> d_scal[0..2]
    bool step_graph = c->md_graph && !c->md_graph_broken && !c->profiling && c->skip_mask == 0 && cg_tol <= 0.0 && cg_max_iter > 0 &&
                      !cg_use_persistent(c);        // (the persistent solve is already one launch)
    for (int n = 0; n < nsteps; ++n) {
        if (n == 0) HQ_TRY(kick(c, d_p, 0.5 * eps, 1));                     // p += F(theta_0) eps/2
        if (step_graph) {
            const int which = (n == nsteps - 1) ? 1 : 0;
            if (md_graph_get(c, which, d_p, d_pf, eps, cg_max_iter) == HQMC_OK) {
                CUDA_TRY(cudaGraphLaunch(c->md[which].exec, c->stream));
                for (int i = 0; i < HQMC_K_COUNT; ++i) c->launches[i] += c->md[which].nodes[i];
                total += cg_max_iter;
                continue;
            }
            c->md_graph_broken = true; step_graph = false;                  // e.g. child-graph capture refused: plain launches
        }
        HQ_TRY(DISPATCH_T(c, do_phase<double>(c, d_p, 2.0 * eps), do_phase<float>(c, d_p, 2.0 * eps)));   // theta += 2 p eps
        HQ_TRY(solve());
        HQ_TRY(kick(c, d_p, 0.5 * eps, (n == nsteps - 1) ? 1 : 2));         // closing half kick (+ opening one of step n+1)
    }
    HQ_TRY(enqueue_energies(c, d_p, d_pf, c->d_X, 3));                      // H1 parts -> d_scal[3..5]
    if (d_theta != c->d_theta)
        CUDA_TRY(cudaMemcpyAsync(d_theta, c->d_theta, sizeof(double) * 2 * c->N, cudaMemcpyDeviceToDevice, c->stream));
    CUDA_TRY(cudaMemcpyAsync(c->h_scal, c->d_scal, sizeof(double) * 8, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    if (H0_out) *H0_out = c->h_scal[0] + c->h_scal[1] + c->h_scal[2];
    if (H1_out) *H1_out = c->h_scal[3] + c->h_scal[4] + c->h_scal[5];
    if (cg_iters_out) *cg_iters_out = total;
    return noconv ? HQMC_ENOCONV : HQMC_OK;
}

extern "C" int hqmc_hqmc_step(hqmc_ctx *c, double *d_theta, double *d_p, const void *d_eta, double u, int nsteps, double eps,
                              double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out, int *accepted_out,
                              long long *cg_iters_out) {
    if (!c || !aligned16(d_theta) || !aligned16(d_p) || !aligned16(d_eta) || nsteps < 0 || cg_max_iter < 0) return HQMC_EINVAL;
    if (d_theta == c->d_force || d_theta == c->d_theta) return HQMC_EINVAL;      // d_force keeps theta_0 for the rejection
    const size_t tb = sizeof(double) * 2 * c->N;
    CUDA_TRY(cudaMemcpyAsync(c->d_force, d_theta, tb, cudaMemcpyDeviceToDevice, c->stream));
    HQ_TRY(hqmc_set_theta(c, d_theta));
    HQ_TRY(hqmc_apply_Mdag(c, d_eta, c->d_phi));                                 // (i) pseudofermion refresh
    double H0 = 0.0, H1 = 0.0;
    int s = hqmc_leapfrog_trajectory(c, d_theta, d_p, c->d_phi, nsteps, eps, cg_tol, cg_max_iter, &H0, &H1, cg_iters_out);   // (ii)
    if (s != HQMC_OK && s != HQMC_ENOCONV) return s;
    double r = std::exp(H0 - H1);
    if (r > 1.0) r = 1.0;
    const int acc = (u < r) ? 1 : 0;                                             // (iii)
    if (!acc) {                                                                  // (iv)
        CUDA_TRY(cudaMemcpyAsync(d_theta, c->d_force, tb, cudaMemcpyDeviceToDevice, c->stream));
        CUDA_TRY(cudaStreamSynchronize(c->stream));
        c->theta_set = false;                                                    // the context's phase tables belong to theta_t
    }
    if (H0_out) *H0_out = H0;
    if (H1_out) *H1_out = H1;
    if (accepted_out) *accepted_out = acc;
    return s;
}

// ---------------------------------------------------------------------------------------------------
// on-device random numbers and the sweep loop
// ---------------------------------------------------------------------------------------------------
static int rng_grid(const hqmc_ctx *c, size_t n) { return (int)std::max<size_t>(1, std::min<size_t>((n + 255) / 256, (size_t)c->n_sm * 8)); }

extern "C" int hqmc_rng_raw(hqmc_ctx *c, unsigned long long seed, unsigned update, unsigned stream, long long n, unsigned *d_out) {
    if (!c || n < 0 || !aligned16(d_out)) return HQMC_EINVAL;
    if (n == 0) return HQMC_OK;
    return launch(c, HQMC_K_MISC, k_rng<double, 0>, dim3(rng_grid(c, (size_t)n)), dim3(256), 0, seed, (uint32_t)update, (uint32_t)stream, (size_t)n, (void *)d_out);
}
extern "C" int hqmc_rng_gauss(hqmc_ctx *c, unsigned long long seed, unsigned update, unsigned stream, long long n, double *d_out) {
    if (!c || n < 0 || !aligned16(d_out)) return HQMC_EINVAL;
    if (n == 0) return HQMC_OK;
    return launch(c, HQMC_K_MISC, k_rng<double, 1>, dim3(rng_grid(c, (size_t)n)), dim3(256), 0, seed, (uint32_t)update, (uint32_t)stream, (size_t)n, (void *)d_out);
}
extern "C" double hqmc_rng_uniform(unsigned long long seed, unsigned update) {
    const Philox4 b = rng_block(seed, (uint32_t)update, 2u, 0ull);
    return rng_u53(b.x[0], b.x[1]);
}

extern "C" int hqmc_sweep(hqmc_ctx *c, double *d_theta, unsigned long long seed, unsigned first_update, int n_updates, int nsteps, double eps,
                          double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out, int *accepted_out, long long *cg_iters_out) {
    if (!c || !aligned16(d_theta) || n_updates < 0 || nsteps < 0 || cg_max_iter < 0) return HQMC_EINVAL;
    int worst = HQMC_OK;
    for (int k = 0; k < n_updates; ++k) {
        const uint32_t upd = (uint32_t)first_update + (uint32_t)k;
        // (i) R and p drawn on the device: R into the CG's z buffer (consumed by phi = M^+ R before the solver touches it),
        //     p into the context's momentum buffer
        if (c->prm.prec == HQMC_C128)
            HQ_TRY(launch(c, HQMC_K_MISC, k_rng<double, 2>, dim3(rng_grid(c, c->N)), dim3(256), 0, seed, upd, 0u, c->N, c->d_z));
        else
            HQ_TRY(launch(c, HQMC_K_MISC, k_rng<float, 2>, dim3(rng_grid(c, c->N)), dim3(256), 0, seed, upd, 0u, c->N, c->d_z));
        HQ_TRY(launch(c, HQMC_K_MISC, k_rng<double, 1>, dim3(rng_grid(c, c->N)), dim3(256), 0, seed, upd, 1u, c->N, (void *)c->d_p));
        const double u = hqmc_rng_uniform(seed, upd);
        // (ii)-(iv)
        const int st = hqmc_hqmc_step(c, d_theta, c->d_p, c->d_z, u, nsteps, eps, cg_tol, cg_max_iter, H0_out ? H0_out + k : nullptr,
                                      H1_out ? H1_out + k : nullptr, accepted_out ? accepted_out + k : nullptr,
                                      cg_iters_out ? cg_iters_out + k : nullptr);
        if (st == HQMC_ENOCONV) worst = st; else if (st != HQMC_OK) return st;
    }
    return worst;
}

// ---------------------------------------------------------------------------------------------------
// host-buffer variants: H2D copies, compute, D2H copies, all on the context's stream
// ---------------------------------------------------------------------------------------------------
extern "C" int hqmc_apply_MdagM_host(hqmc_ctx *c, const void *h_in, void *h_out) {
    if (!c || !h_in || !h_out) return HQMC_EINVAL;
    const size_t vb = c->N * c->esz;
    CUDA_TRY(cudaMemcpyAsync(c->d_d, h_in, vb, cudaMemcpyHostToDevice, c->stream));
    HQ_TRY(hqmc_apply_MdagM(c, c->d_d, c->d_Od));
    CUDA_TRY(cudaMemcpyAsync(h_out, c->d_Od, vb, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return HQMC_OK;
}

extern "C" int hqmc_refresh_host(hqmc_ctx *c, const double *h_theta, const void *h_eta, void *h_phi) {
    if (!c || !h_eta || !h_phi) return HQMC_EINVAL;
    const size_t vb = c->N * c->esz;
    if (h_theta) {
        CUDA_TRY(cudaMemcpyAsync(c->d_theta, h_theta, sizeof(double) * 2 * c->N, cudaMemcpyHostToDevice, c->stream));
        HQ_TRY(hqmc_set_theta(c, c->d_theta));
    }
    if (!c->theta_set) { g_last_error = "no theta"; return HQMC_EINVAL; }
    CUDA_TRY(cudaMemcpyAsync(c->d_d, h_eta, vb, cudaMemcpyHostToDevice, c->stream));
    HQ_TRY(hqmc_apply_Mdag(c, c->d_d, c->d_phi));
    CUDA_TRY(cudaMemcpyAsync(h_phi, c->d_phi, vb, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return HQMC_OK;
}

extern "C" int hqmc_cg_solve_host(hqmc_ctx *c, const double *h_theta, const void *h_rhs, void *h_x, double tol,
                                  long long max_iter, long long *iters_out, double *relres_out) {
    if (!c || !h_rhs || !h_x || max_iter < 0) return HQMC_EINVAL;
    const size_t vb = c->N * c->esz;
    if (h_theta) {
        CUDA_TRY(cudaMemcpyAsync(c->d_theta, h_theta, sizeof(double) * 2 * c->N, cudaMemcpyHostToDevice, c->stream));
        HQ_TRY(hqmc_set_theta(c, c->d_theta));
    }
    if (!c->theta_set) { g_last_error = "no theta"; return HQMC_EINVAL; }
    CUDA_TRY(cudaMemcpyAsync(c->d_phi, h_rhs, vb, cudaMemcpyHostToDevice, c->stream));
    int s = cg_solve_any(c, c->d_phi, c->d_X, tol, max_iter, iters_out, relres_out);
    if (s != HQMC_OK && s != HQMC_ENOCONV) return s;
    CUDA_TRY(cudaMemcpyAsync(h_x, c->d_X, vb, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return s;
}

extern "C" int hqmc_leapfrog_trajectory_host(hqmc_ctx *c, double *h_theta, double *h_p, const void *h_pf, int nsteps, double eps,
                                             double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out,
                                             long long *cg_iters_out) {
    if (!c || !h_theta || !h_p || !h_pf) return HQMC_EINVAL;
    const size_t vb = c->N * c->esz, tb = sizeof(double) * 2 * c->N;
    CUDA_TRY(cudaMemcpyAsync(c->d_theta, h_theta, tb, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaMemcpyAsync(c->d_p, h_p, tb, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaMemcpyAsync(c->d_phi, h_pf, vb, cudaMemcpyHostToDevice, c->stream));
    int s = hqmc_leapfrog_trajectory(c, c->d_theta, c->d_p, c->d_phi, nsteps, eps, cg_tol, cg_max_iter, H0_out, H1_out, cg_iters_out);
    if (s != HQMC_OK && s != HQMC_ENOCONV) return s;
    CUDA_TRY(cudaMemcpyAsync(h_theta, c->d_theta, tb, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaMemcpyAsync(h_p, c->d_p, tb, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return s;
}
