// hqmc_api_slab.inl -- vector steps of the tau-slab PCG: see slab_kernels.cuh and
// paper_2508_16298_b200/slab.py.  The operators of a slab are the ordinary entry points (hqmc_apply_MdagM, hqmc_precond,
// hqmc_force) of a context created for the slab's EXTENDED lattice (owned slices + halo slices).

static int slab_grid(const hqmc_ctx *c, long long n) {
    long long g = (n + 255) / 256, cap = (long long)c->n_sm * 8;
    if (cap > HQMC_MAX_PART) cap = HQMC_MAX_PART;
    return (int)(g < 1 ? 1 : (g < cap ? g : cap));
}

extern "C" int hqmc_slab_dot(hqmc_ctx *c, const void *d_a, const void *d_b, long long n, double *d_out) {
    if (!c || n < 0 || !aligned16(d_a) || !aligned16(d_b) || !d_out) return HQMC_EINVAL;
    const int G = slab_grid(c, n);
    HQ_TRY(DISPATCH_T(c, launch(c, HQMC_K_MISC, k_reduce<double>, dim3(G), dim3(256), 0, 1, (size_t)n, d_a, d_b, c->d_part_misc),
                      launch(c, HQMC_K_MISC, k_reduce<float>, dim3(G), dim3(256), 0, 1, (size_t)n, d_a, d_b, c->d_part_misc)));
    return launch(c, HQMC_K_MISC, k_final_sum, dim3(1), dim3(32), 0, (const double *)c->d_part_misc, G, d_out);
}

template <typename T> static int slab_axpy_t(hqmc_ctx *c, void *x, void *r, const void *d, const void *Od, long long n,
                                             const double *num, const double *den, double *rr_out) {
    typedef typename Cx<T>::type T2;
    const int G = slab_grid(c, n);
    HQ_TRY(launch(c, HQMC_K_AXPY, k_slab_axpy<T>, dim3(G), dim3(256), 0, (size_t)n, (T2 *)x, (T2 *)r, (const T2 *)d, (const T2 *)Od,
                  num, den, c->d_part_misc));
    return launch(c, HQMC_K_MISC, k_final_sum, dim3(1), dim3(32), 0, (const double *)c->d_part_misc, G, rr_out);
}

extern "C" int hqmc_slab_axpy(hqmc_ctx *c, void *d_x, void *d_r, const void *d_d, const void *d_Od, long long n,
                              const double *d_num, const double *d_den, double *d_rr_out) {
    if (!c || n < 0 || !aligned16(d_x) || !aligned16(d_r) || !aligned16(d_d) || !aligned16(d_Od) || !d_num || !d_den || !d_rr_out)
        return HQMC_EINVAL;
    return DISPATCH_T(c, slab_axpy_t<double>(c, d_x, d_r, d_d, d_Od, n, d_num, d_den, d_rr_out),
                      slab_axpy_t<float>(c, d_x, d_r, d_d, d_Od, n, d_num, d_den, d_rr_out));
}

template <typename T> static int slab_dupdate_t(hqmc_ctx *c, void *d, const void *z, long long n, const double *num, const double *den) {
    typedef typename Cx<T>::type T2;
    return launch(c, HQMC_K_DUPDATE, k_slab_dupdate<T>, dim3(slab_grid(c, n)), dim3(256), 0, (size_t)n, (T2 *)d, (const T2 *)z, num, den);
}

extern "C" int hqmc_slab_dupdate(hqmc_ctx *c, void *d_d, const void *d_z, long long n, const double *d_num, const double *d_den) {
    if (!c || n < 0 || !aligned16(d_d) || !aligned16(d_z) || !d_num || !d_den) return HQMC_EINVAL;
    return DISPATCH_T(c, slab_dupdate_t<double>(c, d_d, d_z, n, d_num, d_den), slab_dupdate_t<float>(c, d_d, d_z, n, d_num, d_den));
}

extern "C" int hqmc_slab_scale(hqmc_ctx *c, void *d_v, long long n, double s) {
    if (!c || n < 0 || !aligned16(d_v)) return HQMC_EINVAL;
    if (n == 0) return HQMC_OK;
    return DISPATCH_T(c, launch(c, HQMC_K_MISC, k_slab_scale<double>, dim3(slab_grid(c, n)), dim3(256), 0, (size_t)n, (double2 *)d_v, s),
                      launch(c, HQMC_K_MISC, k_slab_scale<float>, dim3(slab_grid(c, n)), dim3(256), 0, (size_t)n, (float2 *)d_v, (float)s));
}

extern "C" int hqmc_slab_sum_rows(hqmc_ctx *c, const double *d_in, int rows, int stride, int cols, double *d_out) {
    if (!c || !d_in || !d_out || rows < 1 || cols < 1 || stride < cols) return HQMC_EINVAL;
    return launch(c, HQMC_K_MISC, k_slab_sum_rows, dim3((cols + 63) / 64), dim3(64), 0, d_in, rows, stride, cols, d_out);
}

extern "C" int hqmc_slab_field_axpy(hqmc_ctx *c, double *d_y, const double *d_x, double a, long long n) {
    if (!c || n < 0 || !d_y || !d_x) return HQMC_EINVAL;
    if (n == 0) return HQMC_OK;
    return launch(c, HQMC_K_MISC, k_slab_field_axpy, dim3(slab_grid(c, n)), dim3(256), 0, (size_t)n, d_y, d_x, a);
}

extern "C" int hqmc_slab_action_boson(hqmc_ctx *c, int first_slice, int n_slices, double *d_out) {
    if (!c || !d_out || first_slice < 0 || n_slices < 1 || first_slice + n_slices >= c->g.Nt) return HQMC_EINVAL;
    if (!c->theta_set) { g_last_error = "hqmc_set_theta has not been called"; return HQMC_EINVAL; }
    const int G = slab_grid(c, (long long)2 * c->g.Vs * n_slices);
    HQ_TRY(launch(c, HQMC_K_MISC, k_slab_action_boson, dim3(G), dim3(256), 0, c->g, (const double *)c->d_theta, first_slice, n_slices,
                  c->prm.c_tau, c->prm.K, c->prm.compact, c->d_part_misc));
    return launch(c, HQMC_K_MISC, k_final_sum, dim3(1), dim3(32), 0, (const double *)c->d_part_misc, G, d_out);
}
