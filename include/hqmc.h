/*
 * hqmc.h -- C ABI of libhqmc.so: the pseudofermion hot path of the hybrid quantum Monte Carlo
 * method of arxiv/paper_2508_16298 ("Scalable hybrid quantum Monte Carlo simulation of U(1) gauge
 * field coupled to fermions on GPU"), hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * Citations are to /root/reference/PAPER.md (line numbers) and to the readings C1-C25 listed in
 * DESIGN.md (taken from SURVEY.md section 8c).
 *
 * Conventions (all entry points)
 *  - Lattice: L x L sites per time slice (L even, >= 4), Ntau >= 2 slices, N = Ntau*L*L sites.
 *    Site s = x + L*y.  Vector element (tau, s) lives at index tau*L*L + s, interleaved (re, im):
 *    complex128 for HQMC_C128, complex64 for HQMC_C64.
 *  - Gauge field theta (and momentum p, and dS/dtheta): always fp64, layout [Ntau][2][L][L]:
 *    bond (tau, mu, s) at (tau*2 + mu)*L*L + s; mu = 0: s -> s + x, mu = 1: s -> s + y, periodic in
 *    space (Eq.1, 46 Fig.1; reading C3: matrix element (i, j) of a bond i -> j is
 *    e^{+i theta}).  Temporal links are fixed to 0.
 *  - Pointers named d_* are DEVICE pointers, 16-byte aligned, owned by the caller; pointers named
 *    h_* / *_out are HOST pointers.  The library never frees or keeps caller memory beyond the call
 *    (hqmc_set_theta copies theta into the context).  `in` and `out` must not alias unless marked
 *    in/out.
 *  - All work is enqueued on the CUDA stream given to hqmc_create.  Calls with host out-parameters
 *    (hqmc_cg_solve, hqmc_leapfrog_trajectory, hqmc_energies, *_host) synchronise that stream
 *    before returning; the others return as soon as the work is enqueued.
 *  - Return value: 0 on success, negative hqmc_status otherwise.  No exceptions, no exit(), no CPU
 *    fallback: without a CUDA device every compute call returns HQMC_ECUDA.
 */
#ifndef HQMC_H
#define HQMC_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hqmc_ctx hqmc_ctx; /* opaque: phase table, theta copy, CG workspace, reduction scratch, graphs */

typedef enum { HQMC_C128 = 0, HQMC_C64 = 1 } hqmc_prec;

typedef enum {
    HQMC_OK = 0,
    HQMC_EINVAL = -1,  /* bad argument: odd L, L < 4, Ntau < 2, null or misaligned pointer, bad W   */
    HQMC_ECUDA = -2,   /* CUDA error (text via hqmc_last_error)                                    */
    HQMC_ENOCONV = -3, /* CG hit max_iter above tol; x, iters_out, relres_out are still valid      */
    HQMC_ENOMEM = -4   /* device allocation failed                                                 */
} hqmc_status;

typedef struct {
    int L, Ntau;       /* L even >= 4; Ntau >= 2.  Paper: Ntau = 10 L                 */
    double dtau, t;    /* Trotter step 0.1 and hopping 1                         */
    double c_tau, K;   /* S_B couplings: c_tau = 1/(J dtau^2), K (reading C12)     */
    int compact;       /* 1: compact L_B^c; 0: non-compact L_B^nc (Eq.2) */
    int precond_W;     /* preconditioner half bandwidth in tau, 0..32; 0 = identity (reading C10);  */
                       /* 1..12 run the TMA-tiled kernel, wider ones the generic kernel              */
    hqmc_prec prec;    /* arithmetic of the fermion vectors                                        */
} hqmc_params;

/* Create a context for one lattice.  cuda_stream is a cudaStream_t; NULL = the library creates (and owns) a blocking
 * stream of its own, which is ordered with the legacy default stream.
 * Allocates the workspace (phase table, theta copy, 5 CG vectors, scratch) and, if precond_W > 0,
 * builds the default preconditioner taps on the device from the library's own B at pi-flux
 * (reading C10: c_k = [B_pi^k]_00, p_m = sum_k c_k c_{k+m}). */
int hqmc_create(const hqmc_params *params, void *cuda_stream, hqmc_ctx **out);
int hqmc_destroy(hqmc_ctx *ctx);

/* Override the preconditioner: z_{tau,i} = sum_{m=-W..W} taps[|m|] s(tau,m) r_{tau+m,i}, s = -1 when
 * tau+m wraps (antiperiodic fermions).  taps_host has W+1 entries (host memory). */
int hqmc_set_precond(hqmc_ctx *ctx, int W, const double *taps_host);
/* Read back the taps in use (host array of at least 33 doubles); *W_out receives W. */
int hqmc_get_precond(hqmc_ctx *ctx, int *W_out, double *taps_host);

/* Copy theta [Ntau][2][L][L] (device, fp64) into the context and rebuild the link-phase table
 * e^{i theta} (scaled per bond family, Eq.22-26).  Must precede apply/solve/force. */
int hqmc_set_theta(hqmc_ctx *ctx, const double *d_theta);

/* Matrix-free fermion matrix (Eq.8; reading C1; 0-based slices), with
 * B_tau = e^{V4/2} e^{V3/2} e^{V2/2} e^{V1} e^{V2/2} e^{V3/2} e^{V4/2} (Eq.22, reading C5):
 *   (M v)_t    = v_t - B_{t-1} v_{t-1} (t >= 1),   (M v)_0       = v_0 + B_{Nt-1} v_{Nt-1}
 *   (M^+ w)_t  = w_t - B_t w_{t+1}   (t < Nt-1),  (M^+ w)_{Nt-1} = w_{Nt-1} + B_{Nt-1} w_0
 * hqmc_apply_MdagM is the fused O = M^+ M of PAPER.md:248, 284-314. */
int hqmc_apply_M(hqmc_ctx *ctx, const void *d_in, void *d_out);
int hqmc_apply_Mdag(hqmc_ctx *ctx, const void *d_in, void *d_out);
int hqmc_apply_MdagM(hqmc_ctx *ctx, const void *d_in, void *d_out);

/* Banded preconditioner O~^{-1} r (reading C10). */
int hqmc_precond(hqmc_ctx *ctx, const void *d_in, void *d_out);

/* Preconditioned CG on M^+M x = rhs (Eq.20; readings C8, C9): x_0 = 0, d_0 = P r_0,
 * stop when ||r_n|| / ||rhs|| <= tol (recurrence residual, tested after the r update).
 * tol <= 0: run exactly max_iter iterations (the paper's fixed-count CUDA-graph mode).
 * iters_out / relres_out (host, may be NULL): iterations done and ||r|| / ||rhs|| at exit. */
int hqmc_cg_solve(hqmc_ctx *ctx, const void *d_rhs, void *d_x, double tol, long long max_iter,
                  long long *iters_out, double *relres_out);

/* Fermionic force dS_F/dtheta for S_F = phi^+ (M^+M)^{-1} phi, given x = (M^+M)^{-1} phi
 * (PAPER.md:455-477 SI; reading C11): dS_F/dtheta_{b,t} = 2 sigma_t Re[ Y_{t+1}^+ (dB_t/dtheta_b) x_t ],
 * Y = M x.  Output fp64 [Ntau][2][L][L]. */
int hqmc_force(hqmc_ctx *ctx, const void *d_x, double *d_dSF_dtheta);

/* Bosonic force dS_B/dtheta at the context's theta.  Output as above. */
int hqmc_force_boson(hqmc_ctx *ctx, double *d_dSB_dtheta);

/* Energies at the context's theta: S_B(theta); sum p^2 (if d_p != NULL); S_F = Re <phi, x>
 * (if d_phi and d_x != NULL) (Eq.12).  Host outputs, any may be NULL. */
int hqmc_energies(hqmc_ctx *ctx, const double *d_p, const void *d_phi, const void *d_x, double *SB_out,
                  double *p2_out, double *SF_out);

/* One molecular-dynamics trajectory of nsteps leapfrog steps (Eq.16; reading C7):
 *   p += F eps/2;  theta += 2 p eps;  p += F eps/2,   F = -dS_B/dtheta - dS_F/dtheta,
 * with H = S_B + sum p^2 + phi^+ (M^+M)^{-1} phi (Eq.12): nsteps + 1 CG solves.
 * d_theta, d_p: in/out (fp64 [Ntau][2][L][L]); d_pf: the pseudofermion phi.  H0_out / H1_out: H at
 * the start / end; cg_iters_out: total CG iterations (host, may be NULL).
 * Returns HQMC_ENOCONV if any solve hit cg_max_iter with cg_tol > 0 (results still written). */
int hqmc_leapfrog_trajectory(hqmc_ctx *ctx, double *d_theta, double *d_p, const void *d_pf, int nsteps,
                             double eps, double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out,
                             long long *cg_iters_out);

/* n_chain independent trajectories advanced together (independent Markov chains on one lattice shape):
 * d_theta, d_p: [n_chain][Ntau][2][L][L] fp64 in/out, d_pf: [n_chain][Ntau][L][L] complex, all device, caller-owned, 16-byte
 * aligned.  Chain b evolves exactly as hqmc_leapfrog_trajectory would evolve (theta_b, p_b, phi_b); the launches carry the
 * chain index (one phase-table, one multi-right-hand-side PCG and one force/kick launch sequence per leapfrog step for all
 * chains), the per-chain link-phase tables and solutions live in library-owned workspace.  H0_out, H1_out, cg_iters_out:
 * HOST arrays of n_chain entries (may be NULL).  The context's own theta (hqmc_set_theta) is not used; call hqmc_set_theta
 * again before the one-field entry points (where a batch of one would not pay -- one vector's PCG live set fills the L2,
 * e.g. L = 48, Ntau = 480, or L > 48 -- the chains run one after the other on the one-chain kernels and overwrite it).
 * HQMC_ENOCONV if any solve of any chain missed cg_tol. */
int hqmc_leapfrog_trajectory_batched(hqmc_ctx *ctx, double *d_theta, double *d_p, const void *d_pf, int n_chain, int nsteps,
                                     double eps, double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out,
                                     long long *cg_iters_out);
/* Pseudofermion refresh of the chains (PAPER.md:185 step i): phi_b = M^+(theta_b) eta_b.  d_eta and d_phi must not overlap. */
int hqmc_refresh_batched(hqmc_ctx *ctx, const double *d_theta, const void *d_eta, void *d_phi, int n_chain);

/* One HQMC update of every chain, steps (i)-(iv) of PAPER.md:185-201, chain by chain what hqmc_hqmc_step does: d_eta
 * [n_chain][Ntau][L][L] complex Gaussian, d_p [n_chain][...] Gaussian (device); u: HOST array of n_chain uniforms in [0,1).
 * Chain b is accepted iff u[b] < min(1, exp(H0_b - H1_b)); rejected chains get their theta back; d_p holds the final momenta.
 * H0_out, H1_out, accepted_out, cg_iters_out: HOST arrays of n_chain entries (may be NULL). */
int hqmc_hqmc_step_batched(hqmc_ctx *ctx, double *d_theta, double *d_p, const void *d_eta, const double *u, int n_chain,
                           int nsteps, double eps, double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out,
                           int *accepted_out, long long *cg_iters_out);

/* One HQMC update, steps (i)-(iv) of PAPER.md:185-201.  The random numbers are inputs (d_eta complex Gaussian with
 * <|eta|^2> = 1, d_p Gaussian with variance 1/2, u uniform in [0,1); reading C6), so the caller owns the generator:
 *   phi = M^+(theta) eta;  leapfrog trajectory of nsteps steps (as hqmc_leapfrog_trajectory);
 *   accepted iff u < min(1, exp(H0 - H1)) (Eq.15); on rejection d_theta is restored.
 * d_theta: in/out; d_p: in/out (holds the final momenta whatever the decision).  *accepted_out: 1 or 0. */
int hqmc_hqmc_step(hqmc_ctx *ctx, double *d_theta, double *d_p, const void *d_eta, double u, int nsteps, double eps,
                   double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out, int *accepted_out,
                   long long *cg_iters_out);

/* Random numbers of the update, drawn on the device (PAPER.md:185 step (i), :199 step (iii); readings C6, C25).  Counter
 * based: element i of stream s of update k is the Philox4x32-10 block at counter (i lo, i hi, s, k) under key (seed lo,
 * seed hi); streams 0 = R, 1 = p, 2 = u; two 53-bit uniforms per block, Box-Muller pair sqrt(-ln(1 - u1)) (cos, sin)(2 pi u2):
 * two independent N(0, 1/2).  hqmc_rng_raw: the four words of elements 0..n-1 (d_out[4 n], uint32); hqmc_rng_gauss: the
 * Gaussian pairs (d_out[2 n], fp64); hqmc_rng_uniform: the Metropolis uniform of update k (first uniform of element 0 of
 * stream 2), computed on the host. */
int hqmc_rng_raw(hqmc_ctx *ctx, unsigned long long seed, unsigned update, unsigned stream, long long n, unsigned *d_out);
int hqmc_rng_gauss(hqmc_ctx *ctx, unsigned long long seed, unsigned update, unsigned stream, long long n, double *d_out);
double hqmc_rng_uniform(unsigned long long seed, unsigned update);

/* n_updates HQMC updates (the sweep loop of PAPER.md:183-201) on d_theta (in/out): update k = first_update + 0, 1, ...
 * draws R (stream 0) and p (stream 1) on the device and u (stream 2), then runs steps (i)-(iv) as hqmc_hqmc_step does.
 * H0_out, H1_out, accepted_out, cg_iters_out: HOST arrays of n_updates entries (may be NULL).  HQMC_ENOCONV if any solve
 * missed cg_tol (the sweep still completes). */
int hqmc_sweep(hqmc_ctx *ctx, double *d_theta, unsigned long long seed, unsigned first_update, int n_updates, int nsteps,
               double eps, double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out, int *accepted_out,
               long long *cg_iters_out);

/* The same sweep for n_chain independent chains advanced together (hqmc_hqmc_step_batched per update): d_theta
 * [n_chain][Ntau][2][L][L] in/out; chain b draws exactly what hqmc_sweep would draw from seed + b (same counters and streams,
 * update index first_update + k), so a batched sweep is reproducible chain by chain.  H0_out, H1_out, accepted_out,
 * cg_iters_out: HOST arrays of n_updates * n_chain entries, update-major ([k][b]); any may be NULL.  The eta and p workspace is
 * allocated for the call and freed before it returns (synchronises the stream). */
int hqmc_sweep_batched(hqmc_ctx *ctx, double *d_theta, unsigned long long seed, unsigned first_update, int n_updates, int n_chain,
                       int nsteps, double eps, double cg_tol, long long cg_max_iter, double *H0_out, double *H1_out,
                       int *accepted_out, long long *cg_iters_out);

/* ---- Stochastic estimation of fermionic observables ----
 * All pointers are DEVICE pointers to lattice vectors [Ntau][L][L] of the context's complex type (n_rv of them back to
 * back where a count is given), 16-byte aligned, caller-owned.  The calls enqueue on the context's stream; cuFFT provides
 * the transforms of Eq.19 (plan created on first use and owned by the context). */

/* g_k = G xi_k = (M^+ M)^{-1} R_k,  R_k := M^+ xi_k, k = 0..n_rv-1, each by the PCG of Eq.20 to the
 * relative residual `tol` (at most max_iter iterations per vector).  *iters_total (host, may be NULL): iterations summed
 * over the vectors.  Needs hqmc_set_theta.  d_xi and d_g must not overlap.  Returns HQMC_ENOCONV if any solve did not
 * reach tol (all results are still written). */
int hqmc_green_apply(hqmc_ctx *ctx, const void *d_xi, void *d_g, int n_rv, double tol, long long max_iter,
                     long long *iters_total);

/* The same PCG for n_vec right-hand sides at once (the N_rv noise vectors share one theta): d_rhs and d_x
 * hold n_vec lattice vectors back to back (device, 16-byte aligned, caller-owned, must not overlap); vector b is solved
 * exactly as hqmc_cg_solve would (x_0 = 0, Eq.20, readings C8-C9), with its own alpha, beta and stopping test; one kernel
 * launch carries all vectors (vector index in the grid), the workspace (4 n_vec vectors) is library-owned and grown on
 * demand.  iters_out / relres_out: HOST arrays of n_vec entries (may be NULL).  Supported where one thread holds a 2x2
 * block (L <= 48) and Ntau <= 4096, else HQMC_EINVAL.  Synchronises the stream.  HQMC_ENOCONV if any vector missed tol. */
int hqmc_cg_solve_batched(hqmc_ctx *ctx, const void *d_rhs, void *d_x, int n_vec, double tol, long long max_iter,
                          long long *iters_out, double *relres_out);

/* Eq.17-19: C(Delta) = (1/N) sum_i a_i b_{i+Delta} = (1/N) F^{-1}[F[a]_{-k} F[b]_k](Delta), i + Delta periodic in tau, y and
 * x (reading C23), N = L*L*Ntau.  d_C may alias d_a or d_b. */
int hqmc_translation_average(hqmc_ctx *ctx, const void *d_a, const void *d_b, void *d_C);

/* Translation average of the two-point estimate G^_ij = [G xi]_i xi_j^* (PAPER.md:240): a = g_k, b = conj(xi_k), mean over
 * the n_rv vectors (accumulated in Fourier space, one inverse transform). */
int hqmc_green_2pt(hqmc_ctx *ctx, const void *d_g, const void *d_xi, int n_rv, void *d_C);

/* The paper's example C(i,j) = G_ij G_ij: a_i = (G xi)_i (G xi')_i, b_j = xi_j^* xi'_j^*, Eq.19 for
 * every unordered pair of the n_rv >= 2 vectors, mean over the binom(n_rv, 2) pairs. */
int hqmc_pair_correlator(hqmc_ctx *ctx, const void *d_g, const void *d_xi, int n_rv, void *d_C);

/* ---- tau-slab sharding (the paper is single-GPU) ----
 * M and M^+ couple slice t only to t -+ 1 and the preconditioner to t +- W (PAPER.md:155 Eq.8, :316-326), so the lattice shards
 * into contiguous runs of time slices.  A rank (or each of the slabs one process owns) creates an ordinary context for its
 * EXTENDED lattice -- its nt_loc owned slices with H = max(1, W) halo slices on either side, Ntau = nt_loc + 2 H -- and sets the
 * extended theta (the neighbours' slices in the halo).  With the halo slices of a vector filled from the neighbours, multiplied
 * by -1 where they crossed the antiperiodic boundary (tau = Ntau_global - 1 -> 0), hqmc_apply_M / _Mdag / _MdagM, hqmc_precond
 * and hqmc_force of that context return on the OWNED slices exactly what the global operators return (the extended lattice's
 * own wrap only reaches its outermost halo slices, which are discarded).  What is left of a PCG iteration (Eq.20) are the
 * vector updates and the inner products over the owned range, which is one contiguous run of n elements: the calls below,
 * whose coefficients are quotients of DEVICE scalars (sums the ranks have all-reduced), so an iteration is enqueued without the
 * host reading a number.  All pointers are device pointers, vectors 16-byte aligned; everything is enqueued on the context's
 * stream, nothing synchronises.  The exchange itself (NCCL send/recv and all-reduce through torch.distributed) and the loop
 * are paper_2508_16298_b200/slab.py. */
/* d_out[0] = Re <a, b> over n elements (two-stage, fixed order). */
int hqmc_slab_dot(hqmc_ctx *ctx, const void *d_a, const void *d_b, long long n, double *d_out);
/* alpha = *d_num / *d_den;  x += alpha d;  r -= alpha Od;  d_rr_out[0] = ||r||^2 over the n elements. */
int hqmc_slab_axpy(hqmc_ctx *ctx, void *d_x, void *d_r, const void *d_d, const void *d_Od, long long n,
                   const double *d_num, const double *d_den, double *d_rr_out);
/* beta = *d_num / *d_den;  d = z + beta d. */
int hqmc_slab_dupdate(hqmc_ctx *ctx, void *d_d, const void *d_z, long long n, const double *d_num, const double *d_den);
/* v *= s over n elements (s = -1: a halo that crossed the antiperiodic boundary; reading C1). */
int hqmc_slab_scale(hqmc_ctx *ctx, void *d_v, long long n, double s);
/* d_out[j] = sum_i d_in[i * stride + j], i < rows in order, j < cols: the partial sums of the slabs one process owns. */
int hqmc_slab_sum_rows(hqmc_ctx *ctx, const double *d_in, int rows, int stride, int cols, double *d_out);
/* y += a x over n doubles: the drift theta += 2 eps p and the kicks p -= (eps/2) dS/dtheta on a slab's owned slices
 * (Eq.16; dS_F/dtheta from hqmc_force, dS_B/dtheta from hqmc_force_boson of the extended context). */
int hqmc_slab_field_axpy(hqmc_ctx *ctx, double *d_y, const double *d_x, double a, long long n);
/* d_out[0] = the part of S_B that belongs to the slices [first_slice, first_slice + n_slices) of the context's
 * (extended) theta: their plaquette terms and the temporal terms between slice t and t + 1, no wrap -- slice
 * first_slice + n_slices must exist (the upper halo), else HQMC_EINVAL.  Summed over the slabs it is the global S_B. */
int hqmc_slab_action_boson(hqmc_ctx *ctx, int first_slice, int n_slices, double *d_out);

/* HOST-buffer variants (pageable or pinned host memory; the copies run inside the call on the
 * context's stream and the call returns after the result has landed in h_out / h_x). */
int hqmc_apply_MdagM_host(hqmc_ctx *ctx, const void *h_in, void *h_out);
/* Pseudofermion refresh from host buffers (PAPER.md:185 step i): copies h_theta (may be NULL: keep the
 * context's theta) and h_eta to the device, phi = M^+(theta) eta, copies phi to h_phi. */
int hqmc_refresh_host(hqmc_ctx *ctx, const double *h_theta, const void *h_eta, void *h_phi);
int hqmc_cg_solve_host(hqmc_ctx *ctx, const double *h_theta, const void *h_rhs, void *h_x, double tol,
                       long long max_iter, long long *iters_out, double *relres_out);
int hqmc_leapfrog_trajectory_host(hqmc_ctx *ctx, double *h_theta, double *h_p, const void *h_pf, int nsteps,
                                  double eps, double cg_tol, long long cg_max_iter, double *H0_out,
                                  double *H1_out, long long *cg_iters_out);

/* ALLOCATION-FREE S_B (for callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it).  S_B(theta) of PAPER.md:52-54 (the same sum hqmc_energies returns as SB_out) written to the
 * DEVICE double d_SB_out[0], with no context: the call allocates nothing -- no cudaMalloc, cudaFree or allocating library
 * routine -- and enqueues two kernels on cuda_stream (a cudaStream_t of the CURRENT device; NULL = the default stream)
 * without synchronising.  d_theta: device, fp64 [Ntau][2][L][L], read only; c_tau, K, compact as in hqmc_params; any
 * L >= 2 (odd allowed), Ntau >= 1.  The per-CTA partial sums live in a static device array inside the library (64 KB, held
 * by every GPU that loads the library until exit) with room for HQMC_NOALLOC_MAX_LINKS = 2^25 links: a lattice with
 * 2 L^2 Ntau beyond that is rejected with HQMC_EINVAL and a message in hqmc_last_error (config 5, L = 64, Ntau = 640, has
 * 5.2 M links).  Every call shares the array: calls whose kernels OVERLAP on the GPU (different streams without an event
 * between them, or two host threads) race on it and may both return wrong sums; calls on one stream are safe.  Nothing in
 * the array needs clearing between calls (each call writes every partial it reads).  The sum order differs from
 * hqmc_energies (fixed 4096-link CTAs): results agree to rounding (~1e-14 relative), not bit for bit. */
#define HQMC_NOALLOC_MAX_LINKS (1 << 25)
int hqmc_action_boson_noalloc(const double *d_theta, int L, int Ntau, double c_tau, double K, int compact,
                              double *d_SB_out, void *cuda_stream);

/* Instrumentation and tuning knobs (launch statistics, kernel selection, timing experiments) are declared in
 * hqmc_tuning.h; nothing in this header depends on them. */

const char *hqmc_strerror(int status);
const char *hqmc_last_error(void); /* text of the last CUDA error seen by this thread, or "" */
int hqmc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HQMC_H */
