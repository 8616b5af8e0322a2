/*
 * hqmc_tuning.h -- instrumentation and tuning knobs of libhqmc.so.  NOT part of the operations of the method
 * (those are in hqmc.h, which does not depend on this header): launch statistics for the benchmarks, kernel
 * selection for parity tests of every code path, and timing experiments.  Every setter returns 0 or a negative
 * hqmc_status; results of the hot path are the same in every setting unless stated otherwise.
 */
#ifndef HQMC_TUNING_H
#define HQMC_TUNING_H

#include "hqmc.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Instrumentation.  hqmc_set_profiling(ctx, 1) makes the library bracket each launch of its kernels
 * with CUDA events on the context's stream (CG then runs without graph replay); hqmc_get_kernel_stats
 * returns, for kernel class `which` (HQMC_K_*), the number of launches and the summed device time in
 * ms since the last hqmc_reset_stats.  Launch counts are kept even when profiling is off. */
enum { HQMC_K_MDAGM = 0, HQMC_K_AXPY = 1, HQMC_K_PRECOND = 2, HQMC_K_DUPDATE = 3, HQMC_K_M = 4,
       HQMC_K_FORCE = 5, HQMC_K_PHASE = 6, HQMC_K_MISC = 7, HQMC_K_COUNT = 8 };
int hqmc_set_profiling(hqmc_ctx *ctx, int on);
int hqmc_reset_stats(hqmc_ctx *ctx);
int hqmc_get_kernel_stats(hqmc_ctx *ctx, int which, long long *launches_out, double *ms_out);

/* Fused M^+M kernel.  AUTO: the streaming kernel (TMA bulk copies, packed link phases, time run
 * swept backwards) where its staging buffers fit one SM (L <= 48 in complex128), the cluster kernel (the slice split
 * over 2/4/8 SMs with distributed shared memory) where they do not (e.g. L = 64), else the register-only kernel.
 * A kernel that does not exist for the lattice gives HQMC_EINVAL. */
enum { HQMC_MDAGM_AUTO = 0, HQMC_MDAGM_REGISTER = 1, HQMC_MDAGM_CLUSTER = 2, HQMC_MDAGM_STREAM = 3 };
int hqmc_set_mdagm_kernel(hqmc_ctx *ctx, int which);
/* Slices per CTA of the fused M^+M kernel (0 = library default: one CTA, or cluster, per SM with the slices dealt
 * out evenly). */
int hqmc_set_time_tile(hqmc_ctx *ctx, int slices_per_cta);

/* Preconditioner kernel for W = 1..6: n > 0: TMA-tiled kernel, runs of n slices per CTA; n < 0: register-ring
 * kernel with runs of -n slices; 0 = library default (TMA-tiled, shortest run that fits one wave). */
int hqmc_set_precond_tile(hqmc_ctx *ctx, int slices_per_run);

/* PCG vector kernels (Eq.20).  AUTO = by footprint: TEXTBOOK (M^+M | x += alpha d, r -= alpha Od |
 * z = P r | d = z + beta d) while the loop's live set (r, d, Od|z, packed phases) fits the L2, DEFERRED_X
 * (M^+M | r -= alpha Od | z = P r | x += alpha d, d = z + beta d: 16 B/site less traffic) otherwise.  Same iterates. */
enum { HQMC_CG_AUTO = 0, HQMC_CG_TEXTBOOK = 1, HQMC_CG_DEFERRED_X = 2 };
int hqmc_set_cg_variant(hqmc_ctx *ctx, int which);

/* Whole PCG solve as ONE persistent cooperative kernel (pcg_persist.cuh; small lattices are launch-bound):
 * one CTA per time slice, x, r, d, z and the decoded links in registers for the whole solve; per iteration the two global sums
 * of Eq.20 as all-to-all exchanges of tagged words and two point-to-point halo hand-overs, no kernel boundary, no atomic.
 * Usable where one thread holds a 2x2 block and all Ntau CTAs are resident at once (L <= 22 at Ntau = 10 L on a B200).  AUTO
 * (default) = taken by hqmc_cg_solve and every entry point that solves to a tolerance through it (trajectories, sweeps, the
 * one-vector path of hqmc_green_apply) where usable and the lattice has at most HQMC_PERSIST_AUTO_SITES sites (measured: 10.8 us
 * per iteration against 15.5-17.3 for the four-kernel graph at L = 8...16, 15.5 against 18.9 at L = 20); OFF = never; ON = wherever
 * usable (HQMC_EINVAL where it is not).  Same iterates as the four-kernel loop up to the order of the sums. */
enum { HQMC_PERSIST_AUTO = 0, HQMC_PERSIST_OFF = 1, HQMC_PERSIST_ON = 2 };
#define HQMC_PERSIST_AUTO_SITES 100000
int hqmc_set_cg_persistent(hqmc_ctx *ctx, int mode);

/* Vectors hqmc_green_apply solves per launch: 0 (default) = as many as keep the batch's live set L2-resident, 1 = one
 * at a time on the one-vector kernels, n > 1 = n at a time. */
int hqmc_set_green_batch(hqmc_ctx *ctx, int n);

/* Leapfrog steps captured in a CUDA graph: 1 (default) = phase/drift, the PCG chunks, force + kick of one
 * step are replayed as one graph when the solves run a fixed iteration count; 0 = plain launches.  Bit-identical. */
int hqmc_set_md_graph(hqmc_ctx *ctx, int on);

/* Programmatic dependent launch inside the PCG iteration (kernel k+1 is dispatched under kernel k's tail and waits
 * on-device for its completion before reading its output). 1 (default) = every launch of the iteration up to L = 44, and at
 * L >= 48 the preconditioner and the d update only, the two launches that follow a kernel filling every SM evenly; 0 = off; 16 + mask = per-kernel-class mask (bit = HQMC_K_* class),
 * for timing experiments. Results are bit-identical in every setting. */
int hqmc_set_pdl(hqmc_ctx *ctx, int on);

/* TIMING ONLY: bit k of mask set = kernels of class HQMC_K_<k> are not launched (leave-one-out timing of a kernel
 * inside the graph-replayed PCG iteration; the numerical results are then MEANINGLESS).  0 restores normal operation. */
int hqmc_set_debug_skip(hqmc_ctx *ctx, unsigned mask);

#ifdef __cplusplus
}
#endif
#endif /* HQMC_TUNING_H */
