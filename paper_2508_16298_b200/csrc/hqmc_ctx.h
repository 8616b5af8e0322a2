// hqmc_ctx.h -- private context of libhqmc.so and launch helpers (host code).
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/hqmc.h"
#include "../../include/hqmc_tuning.h"
#include "cg_kernels.cuh"
#include "force_kernels.cuh"
#include "force_stream.cuh"
#include "kernels.cuh"
#include "mdagm_stream.cuh"
#include "mdagm_cluster.cuh"
#include "mdagm_back.cuh"
#include "precond_tma.cuh"
#include "measure_kernels.cuh"
#include "cg_batched.cuh"
#include "rng_kernels.cuh"
#include "slab_kernels.cuh"
#include "pcg_persist.cuh"

namespace hqmc {

extern thread_local std::string g_last_error;

#define CUDA_TRY(expr)                                                                                     \
    do {                                                                                                   \
        cudaError_t _e = (expr);                                                                           \
        if (_e != cudaSuccess) {                                                                           \
            g_last_error = std::string(#expr) + ": " + cudaGetErrorString(_e);                             \
            return (_e == cudaErrorMemoryAllocation) ? HQMC_ENOMEM : HQMC_ECUDA;                           \
        }                                                                                                  \
    } while (0)
#define HQ_TRY(expr)                                                                                       \
    do {                                                                                                   \
        int _s = (expr);                                                                                   \
        if (_s != HQMC_OK) return _s;                                                                      \
    } while (0)

struct KernelCfg { int bpt; int maxt; int threads; };

struct EventPair { cudaEvent_t a, b; int kclass; };

}  // namespace hqmc

// Kernel classes launched programmatically (griddepcontrol) by default: the preconditioner after the residual update and the
// d update after the preconditioner. Both predecessors fill every SM evenly, so the early-dispatched CTAs spread evenly too
// (-0.8 us per iteration at L=48). Not after M^+M: its grid leaves SMs idle, the next kernel's CTAs pile onto those and its
// grid-stride loop then runs unbalanced (+4.7 us, measured; profiles/r01_summary.md).
#define HQMC_PDL_DEFAULT ((1 << HQMC_K_PRECOND) | (1 << HQMC_K_DUPDATE))

struct hqmc_ctx {
    hqmc_params prm;
    hqmc::Geo g;
    size_t N;            // sites
    size_t esz;          // bytes per complex element
    cudaStream_t stream;
    bool own_stream;
    int n_sm;
    hqmc::KernelCfg cfg;
    int time_tile;       // slices per CTA of k_mdagm (0 = auto)
    double C;            // cosh(a/2)^6 cosh(a)
    double th_full, th_half;
    hqmc::Taps taps;
    // device memory owned by the context
    double *d_theta;     // copy of the gauge field
    void *d_ph;          // phase table [Nt][2][L][L] complex
    void *d_packed;      // packed link phases [Nt][4][nb][2] (8 B each) for the streaming M^+M kernel
    double2 *d_tab;      // [2][1024] tanh(a) e^{i k delta} (half step, full step)
    bool stream_on;      // runtime switch (hqmc_set_mdagm_kernel): the streaming kernel k_mdagm_back is selected
    bool use_cluster, cluster_on;   // cluster kernel (slice split over R SMs) usable / selected
    int cl_R, cl_threads; size_t cl_smem;
    bool use_stream;     // streaming kernel usable (one block per thread and its staging buffers fit one SM)
    size_t stream_smem;
    size_t force_stream_smem = 0;   // k_force_stream (follows stream_on)
    void *d_r, *d_z, *d_d, *d_Od, *d_X, *d_phi;   // CG vectors, trajectory solution / pseudofermion
    double *d_p, *d_force;                        // host-variant staging
    double *d_part_dOd, *d_part_rr, *d_part_rz[2], *d_part_misc;
    hqmc::CgState *d_state;
    hqmc::CgState *h_state;  // pinned
    double *d_scal;          // 8 doubles
    double *h_scal;          // pinned
    bool theta_set;
    // grids
    int grid_ew, grid_mdagm;
    int pc_tile;         // slices per run of the sliding-window preconditioner kernel (0 = generic kernel)
    int pc_gx, pc_gy, n_part_rz;
    int pc_kind;         // 0: generic k_precond, 1: register-ring k_precond_win, 2: TMA-tiled k_precond_tma
    size_t pc_smem;
    // CG chunk graph
    cudaGraphExec_t cg_graph;
    void *cg_graph_x;        // x pointer baked into the graph
    int cg_graph_tile;
    bool cg_graph_defer;
    size_t l2_bytes;     // device L2 size
    // stochastic estimator (hqmc_api_measure.inl): workspace and 3-D FFT plan, created on first use
    bool ms_ready = false, ms_plan_ok = false;
    cufftHandle ms_plan = 0;
    void *d_ms_a = nullptr, *d_ms_b = nullptr, *d_ms_acc = nullptr;
    // multi-right-hand-side PCG (hqmc_api_cgb.inl): workspace for cgb_cap vectors, created on first use
    int cgb_cap = 0, cgb_pstride = 0;
    void *d_cgb_r = nullptr, *d_cgb_d = nullptr, *d_cgb_Od = nullptr, *d_cgb_phi = nullptr;
    void *d_cgb_ph = nullptr; double *d_cgb_scal = nullptr, *h_cgb_scal = nullptr; const void *cgb_graph_ph = nullptr; size_t cgb_graph_phs = 0;
    double *d_cgb_theta0 = nullptr; int cgb_theta0_cap = 0; void *d_cgb_pf = nullptr; int d_cgb_pf_cap = 0;   // hqmc_hqmc_step_batched
    double *d_cgb_part = nullptr;          // [5][cgb_cap][cgb_pstride]: dOd, rr, rz[0], rz[1], spare
    hqmc::CgState *d_cgb_state = nullptr, *h_cgb_state = nullptr;
    cudaGraphExec_t cgb_graph = nullptr;
    void *cgb_graph_x = nullptr; int cgb_graph_n = 0, cgb_graph_tt = 0, cgb_graph_W = -1;
    long long cgb_nodes[HQMC_K_COUNT] = {};
    int green_batch = 0;                   // hqmc_set_green_batch: 0 = by footprint, 1 = one vector at a time, n = n at a time
    // whole-solve persistent kernel (pcg_persist.cuh): usable (one block per thread, all Ntau CTAs co-resident) / mode
    bool persist_ok = false; int persist_mode = 0;        // 0 = auto (small lattices), 1 = never, 2 = whenever usable
    size_t persist_smem = 0; unsigned long long *d_ctr = nullptr;
    bool cg_defer_x;     // deferred-x PCG vector kernels (k_cg_raxpy + k_cg_xdupdate)
    int cg_chunk;            // iterations per graph launch
    bool md_graph = true;    // leapfrog steps with fixed-count solves replayed as one CUDA graph (hqmc_set_md_graph)
    bool md_graph_broken = false;            // capturing a step failed once on this context: plain launches from then on
    bool capturing_md = false;               // a leapfrog step is being captured (launch() counts into md_nodes_cur)
    long long cfg_epoch = 0;                 // bumped whenever the PCG chunk graph is rebuilt (kernel selection, taps, tiles, ...)
    struct MdGraph {                         // [0]: a middle step (closing + opening half kick), [1]: the last step of a trajectory
        cudaGraphExec_t exec = nullptr;
        const double *p = nullptr; const void *pf = nullptr; double eps = 0.0; long long iters = -1, epoch = -1;
        long long nodes[HQMC_K_COUNT] = {};
    } md[2];
    long long *md_nodes_cur = nullptr;
    // instrumentation
    bool pdl_next;        // set by a call site whose kernel calls griddepcontrol.wait; consumed by launch()
    int pdl;              // bit per kernel class: programmatic dependent launch of the PCG kernels (hqmc_set_pdl)
    unsigned skip_mask;   // timing-only: kernel classes NOT launched inside the PCG iteration (hqmc_set_debug_skip)
    bool profiling;
    bool capturing;
    long long launches[HQMC_K_COUNT];
    long long graph_nodes[HQMC_K_COUNT];   // kernels of each class inside one cg_graph replay
    double ms[HQMC_K_COUNT];
    std::vector<hqmc::EventPair> pending;
    std::vector<hqmc::EventPair> pool;
};

// Default programmatic-launch mask: every edge of the iteration where the streaming M^+M CTA leaves room on its SM (up to 512 threads,
// L <= 44: 2 % at L = 32...44, neutral below; measured, profiles/r02_summary.md), the two safe edges where it fills the SM (L = 48:
// the early axpy CTAs pile up behind it, +6 us) and for the cluster / register kernels.
static int pdl_default(const hqmc_ctx *c) {
    return (c->use_stream && c->stream_on && c->cfg.threads <= 512) ? 15 : HQMC_PDL_DEFAULT;
}

// The PCG loop's live set is r, d, Od|z and the packed phases (4 x N x esz; x is streamed). While it fits the L2 the textbook
// kernels win (their traffic is L2 traffic); beyond it the deferred-x pair, which moves 16 B/site less, does
// (L=64, Ntau=640, 168 MB: 128.9 vs 131.5 us per iteration; L=48, Ntau=480, 71 MB: 53.2 vs 52.4; profiles/r01_summary.md).
static bool cg_defer_default(const hqmc_ctx *c) { return 4 * c->N * c->esz > c->l2_bytes; }

