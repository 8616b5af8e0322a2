// hqmc_noalloc.cu -- hqmc_action_boson_noalloc: S_B(theta) without any allocation.  See include/hqmc.h.
//
// For callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): no
// context, no cudaMalloc / cudaFree / allocating library routine anywhere on this path.  The per-CTA partial sums of the
// reduction live in the file-scope array g_noalloc_part below; every GPU that loads libhqmc.so holds its 64 KB until the
// process exits.  All calls share that array: two calls whose kernels overlap on the GPU (different streams, or one device
// used from two threads without ordering) race on it.  Nothing in it has to start at zero: every call writes each partial
// it later reads, whatever an earlier call left there.
//
// This file is self-contained on purpose (its own kernels, no header of the hot path) so that adding it changes no existing
// code path; it shares only the status codes and the last-error text with hqmc.cu.
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>
#include <string>

#include "../../include/hqmc.h"

namespace hqmc {
extern thread_local std::string g_last_error;
}

namespace {

constexpr int NA_THREADS = 256;                       // threads per CTA
constexpr int NA_PER_THREAD = 16;                     // links per thread
constexpr int NA_LINKS_PER_CTA = NA_THREADS * NA_PER_THREAD;          // 4096 links = one partial
constexpr int NA_MAX_PART = HQMC_NOALLOC_MAX_LINKS / NA_LINKS_PER_CTA;  // 8192 partials = 64 KB
constexpr int NA_MAX_DEV = 64;

static_assert((long long)NA_MAX_PART * NA_LINKS_PER_CTA == HQMC_NOALLOC_MAX_LINKS, "limit must be a whole number of CTAs");

// The scratch.  In HOST code this name is a host-side stand-in, not a device address: the address the kernels get comes
// from cudaGetSymbolAddress (scratch_of_current_device below).
static __device__ __align__(256) double g_noalloc_part[NA_MAX_PART];

__device__ __forceinline__ double na_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// Variant of k_action_boson (force_kernels.cuh) with a FIXED partition: CTA b sums the terms of links
// [4096 b, 4096 (b + 1)) -- one temporal term per link, one plaquette term per site (the mu = 0 links) -- into part[b].
// theta is [Ntau][2][L][L]; curl theta(s) = th_x(s) + th_y(s + x) - th_x(s + y) - th_y(s).
__global__ void __launch_bounds__(NA_THREADS) k_action_boson_noalloc(int L, int Nt, const double *__restrict__ theta,
                                                                     double c_tau, double K, int compact,
                                                                     double *__restrict__ part) {
    __shared__ double red[NA_THREADS / 32];
    const int Vs = L * L;
    const size_t per_slice = (size_t)2 * Vs, n = per_slice * Nt;
    const size_t base = (size_t)blockIdx.x * NA_LINKS_PER_CTA;
    double acc = 0.0;
#pragma unroll 4
    for (int k = 0; k < NA_PER_THREAD; ++k) {
        const size_t i = base + (size_t)k * NA_THREADS + threadIdx.x;
        if (i >= n) break;
        const int t = (int)(i / per_slice), r = (int)(i - (size_t)t * per_slice);
        const int tn = (t + 1 == Nt) ? 0 : t + 1;
        const double d = theta[(size_t)tn * per_slice + r] - theta[i];
        acc += c_tau * (compact ? (1.0 - cos(d)) : d * d);
        if (r < Vs) {
            const double *th = theta + (size_t)t * per_slice;
            const int y = r / L, x = r - y * L;
            const int xp = (x + 1 == L) ? 0 : x + 1, yp = (y + 1 == L) ? 0 : y + 1;
            acc += K * cos(th[y * L + x] + th[Vs + y * L + xp] - th[yp * L + x] - th[Vs + y * L + x]);
        }
    }
    acc = na_warp_sum(acc);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double r = (threadIdx.x < NA_THREADS / 32) ? red[threadIdx.x] : 0.0;
        r = na_warp_sum(r);
        if (threadIdx.x == 0) part[blockIdx.x] = r;
    }
}

// out[0] = sum of part[0 .. n_part) in a fixed order (one CTA; thread j takes j, j + 256, ...).
__global__ void __launch_bounds__(NA_THREADS) k_noalloc_final_sum(const double *__restrict__ part, int n_part,
                                                                  double *__restrict__ out) {
    __shared__ double red[NA_THREADS / 32];
    double acc = 0.0;
    for (int j = threadIdx.x; j < n_part; j += NA_THREADS) acc += part[j];
    acc = na_warp_sum(acc);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double r = (threadIdx.x < NA_THREADS / 32) ? red[threadIdx.x] : 0.0;
        r = na_warp_sum(r);
        if (threadIdx.x == 0) out[0] = r;
    }
}

// Device address of g_noalloc_part on the CURRENT device, looked up once per device with that device current.
std::mutex g_na_mutex;
double *g_na_ptr[NA_MAX_DEV] = {};

int scratch_of_current_device(double **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { hqmc::g_last_error = std::string("cudaGetDevice: ") + cudaGetErrorString(e); return HQMC_ECUDA; }
    if (dev < 0 || dev >= NA_MAX_DEV) { hqmc::g_last_error = "hqmc_action_boson_noalloc: device ordinal beyond 63"; return HQMC_EINVAL; }
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (g_na_ptr[dev] == nullptr) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_noalloc_part);
        if (e != cudaSuccess || p == nullptr) {
            hqmc::g_last_error = std::string("cudaGetSymbolAddress(g_noalloc_part): ") + cudaGetErrorString(e);
            return HQMC_ECUDA;
        }
        g_na_ptr[dev] = p;
    }
    *out = g_na_ptr[dev];
    return HQMC_OK;
}

}  // namespace

extern "C" int hqmc_action_boson_noalloc(const double *d_theta, int L, int Ntau, double c_tau, double K, int compact,
                                         double *d_SB_out, void *cuda_stream) {
    if (d_theta == nullptr || d_SB_out == nullptr || (reinterpret_cast<uintptr_t>(d_theta) & 7u) ||
        (reinterpret_cast<uintptr_t>(d_SB_out) & 7u)) {
        hqmc::g_last_error = "hqmc_action_boson_noalloc: null or misaligned pointer";
        return HQMC_EINVAL;
    }
    if (L < 2 || Ntau < 1 || L > 16384) { hqmc::g_last_error = "hqmc_action_boson_noalloc: need L >= 2, Ntau >= 1"; return HQMC_EINVAL; }
    const long long n_links = 2LL * L * L * Ntau;
    if (n_links > (long long)HQMC_NOALLOC_MAX_LINKS) {
        hqmc::g_last_error = "hqmc_action_boson_noalloc: 2 L^2 Ntau = " + std::to_string(n_links) +
                             " links exceed HQMC_NOALLOC_MAX_LINKS = " + std::to_string((long long)HQMC_NOALLOC_MAX_LINKS) +
                             " (the static scratch holds one partial per 4096 links); use hqmc_energies";
        return HQMC_EINVAL;
    }
    double *d_part = nullptr;
    const int s = scratch_of_current_device(&d_part);
    if (s != HQMC_OK) return s;
    const int n_part = (int)((n_links + NA_LINKS_PER_CTA - 1) / NA_LINKS_PER_CTA);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    k_action_boson_noalloc<<<n_part, NA_THREADS, 0, st>>>(L, Ntau, d_theta, c_tau, K, compact, d_part);
    k_noalloc_final_sum<<<1, NA_THREADS, 0, st>>>(d_part, n_part, d_SB_out);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { hqmc::g_last_error = std::string("hqmc_action_boson_noalloc launch: ") + cudaGetErrorString(e); return HQMC_ECUDA; }
    return HQMC_OK;
}
