// slab_kernels.cuh -- vector kernels of the tau-slab PCG (Eq.20).
//
// A rank owns a run of time slices; its vectors are stored with `halo` extra slices on either side, so the slices the rank
// OWNS are one contiguous range of elements.  These kernels work on such a range (pointer + element count) and take their
// coefficients as quotients of DEVICE scalars (sums every rank has already all-reduced), so that a PCG iteration is enqueued
// without the host ever reading a number:
//     alpha = <r,z> / <d,Od>;   x += alpha d;   r -= alpha Od;   partial ||r||^2
//     beta  = <r,z>_new / <r,z>_old;   d = z + beta d
// Sums are two-stage and run in a fixed order (one partial per CTA, then k_final_sum): deterministic run to run.
#pragma once
#include "cg_kernels.cuh"
#include "force_kernels.cuh"

namespace hqmc {

template <typename T>
__global__ void k_slab_axpy(size_t n, typename Cx<T>::type *__restrict__ x, typename Cx<T>::type *__restrict__ r,
                            const typename Cx<T>::type *__restrict__ d, const typename Cx<T>::type *__restrict__ Od,
                            const double *__restrict__ num, const double *__restrict__ den, double *__restrict__ part_rr) {
    typedef typename Cx<T>::type T2;
    __shared__ double red[32];
    const T alpha = (T)(*num / *den);
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const T2 di = d[i], oi = Od[i];
        T2 xi = x[i], ri = r[i];
        xi.x = fma(alpha, di.x, xi.x); xi.y = fma(alpha, di.y, xi.y);
        ri.x = fma(-alpha, oi.x, ri.x); ri.y = fma(-alpha, oi.y, ri.y);
        x[i] = xi; r[i] = ri;
        acc += (double)ri.x * (double)ri.x + (double)ri.y * (double)ri.y;
    }
    const double s = block_sum(acc, red);
    if (threadIdx.x == 0) part_rr[blockIdx.x] = s;
}

template <typename T>
__global__ void k_slab_dupdate(size_t n, typename Cx<T>::type *__restrict__ d, const typename Cx<T>::type *__restrict__ z,
                               const double *__restrict__ num, const double *__restrict__ den) {
    typedef typename Cx<T>::type T2;
    const T beta = (T)(*num / *den);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const T2 zi = z[i];
        T2 di = d[i];
        di.x = fma(beta, di.x, zi.x); di.y = fma(beta, di.y, zi.y);
        d[i] = di;
    }
}

// v *= s (s = -1: a halo that crossed the antiperiodic boundary, Eq.8 / reading C1)
template <typename T>
__global__ void k_slab_scale(size_t n, typename Cx<T>::type *__restrict__ v, T s) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        typename Cx<T>::type a = v[i];
        a.x *= s; a.y *= s;
        v[i] = a;
    }
}

// y += a x over n doubles: the drift theta += 2 eps p and the kicks p -= (eps/2) dS/dtheta of a slab's owned slices (Eq.16)
__global__ void k_slab_field_axpy(size_t n, double *__restrict__ y, const double *__restrict__ x, double a) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) y[i] = fma(a, x[i], y[i]);
}

// S_B restricted to the slices [first, first + count) of an extended lattice: the temporal term of slice t couples
// it to slice t + 1, which must exist in the buffer (the upper halo); no wrap.  One partial per CTA.
__global__ void k_slab_action_boson(Geo g, const double *__restrict__ theta, int first, int count, double c_tau, double K, int compact,
                                    double *__restrict__ part) {
    __shared__ double red[32];
    const size_t per = (size_t)2 * g.Vs, n = per * (size_t)count;
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int t = first + (int)(i / per);
        const int r = (int)(i % per);
        const double d = theta[(size_t)(t + 1) * per + r] - theta[(size_t)t * per + r];
        acc += c_tau * (compact ? (1.0 - cos(d)) : d * d);
        if (r < g.Vs) {
            const int y = r / g.L, x = r - y * g.L;
            acc += K * cos(curl_at(theta + (size_t)t * per, g.L, g.Vs, x, y));
        }
    }
    const double s = block_sum(acc, red);
    if (threadIdx.x == 0) part[blockIdx.x] = s;
}

// out[j] = sum_{i < rows} in[i * stride + j], j < cols, rows added in index order (the slabs one process owns)
__global__ void k_slab_sum_rows(const double *__restrict__ in, int rows, int stride, int cols, double *__restrict__ out) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= cols) return;
    double s = 0.0;
    for (int i = 0; i < rows; ++i) s += in[(size_t)i * stride + j];
    out[j] = s;
}

}  // namespace hqmc
