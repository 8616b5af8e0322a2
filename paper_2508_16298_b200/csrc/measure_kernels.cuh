// measure_kernels.cuh -- stochastic estimation of fermionic observables (widening row NEXT-2).
//
//   G xi = (M^+ M)^{-1} M^+ xi                       (the PCG of cg_kernels.cuh)
//   C^(i,j) = a_i b_j                                (Eq.18)
//   C^(Delta) = (1/N) sum_i a_i b_{i+Delta} = (1/N) F^{-1}[ F[a]_{-k} F[b]_k ](Delta)      (Eq.17, 19)
//
// The FFTs are cuFFT's (a library primitive, as in the paper); the kernels here build a and b, form the spectral product
// with the index reflection k -> -k, and accumulate over vectors or pairs IN FOURIER SPACE (the inverse transform is linear,
// so one inverse FFT serves any number of pairs).
#pragma once
#include "kernels.cuh"

namespace hqmc {

// a = g (copy), b = conj(xi)                                                     two-point estimate
template <typename T>
__global__ void k_ms_2pt_ab(size_t N, const typename Cx<T>::type *__restrict__ g, const typename Cx<T>::type *__restrict__ xi,
                            typename Cx<T>::type *__restrict__ a, typename Cx<T>::type *__restrict__ b) {
    typedef typename Cx<T>::type T2;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        const T2 x = xi[i];
        a[i] = g[i];
        T2 o; o.x = x.x; o.y = -x.y;
        b[i] = o;
    }
}

// a = g .* g',  b = conj(xi) .* conj(xi')                                          PAPER.md:240 (C(i,j) = G_ij G_ij)
template <typename T>
__global__ void k_ms_pair_ab(size_t N, const typename Cx<T>::type *__restrict__ g1, const typename Cx<T>::type *__restrict__ g2,
                             const typename Cx<T>::type *__restrict__ x1, const typename Cx<T>::type *__restrict__ x2,
                             typename Cx<T>::type *__restrict__ a, typename Cx<T>::type *__restrict__ b) {
    typedef typename Cx<T>::type T2;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        const T2 p = g1[i], q = g2[i], u = x1[i], v = x2[i];
        T2 o;
        o.x = p.x * q.x - p.y * q.y; o.y = p.x * q.y + p.y * q.x;
        a[i] = o;
        o.x = u.x * v.x - u.y * v.y; o.y = -(u.x * v.y + u.y * v.x);      // conj(u v)
        b[i] = o;
    }
}

// D[k] (+)= scale * Fa[-k] * Fb[k]        k = (kt, ky, kx) on the Nt x L x L lattice, -k taken modulo the extent (Eq.19)
template <typename T, bool ACC>
__global__ void k_ms_spectral(int Nt, int L, const typename Cx<T>::type *__restrict__ Fa, const typename Cx<T>::type *__restrict__ Fb,
                              typename Cx<T>::type *__restrict__ D, T scale) {
    typedef typename Cx<T>::type T2;
    const size_t Vs = (size_t)L * L, N = Vs * Nt;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        const int kt = (int)(i / Vs), r = (int)(i - (size_t)kt * Vs), ky = r / L, kx = r - ky * L;
        const int mt = kt ? Nt - kt : 0, my = ky ? L - ky : 0, mx = kx ? L - kx : 0;
        const T2 a = Fa[((size_t)mt * L + my) * L + mx], b = Fb[i];
        T2 o;
        o.x = scale * (a.x * b.x - a.y * b.y); o.y = scale * (a.x * b.y + a.y * b.x);
        if (ACC) { const T2 d = D[i]; o.x += d.x; o.y += d.y; }
        D[i] = o;
    }
}

}  // namespace hqmc
