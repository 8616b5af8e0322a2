// rng_kernels.cuh -- random numbers of the HQMC update on the device (PAPER.md:185 step (i): Gaussian p and R
// step (iii): uniform u; readings C6, C25).
//
// Counter-based, so a sweep is reproducible from (seed, update index) and needs no generator state in memory: element i of
// stream s of update k is the Philox4x32-10 block (Salmon et al., SC'11) at counter (i lo, i hi, s, k) under key
// (seed lo, seed hi); streams: 0 = R, 1 = p (pairs), 2 = u.  The four words give two 53-bit uniforms
//     u1 = ((x0 >> 5) 2^26 + (x1 >> 6)) / 2^53,  u2 = ((x2 >> 5) 2^26 + (x3 >> 6)) / 2^53,
// and Box-Muller the pair sqrt(-ln(1 - u1)) (cos 2 pi u2, sin 2 pi u2): two independent N(0, 1/2), i.e. one complex R with
// E|R|^2 = 1 or two momenta with variance 1/2.  The integer stream is bit-identical to the CPU twin used by the tests; the
// Gaussians agree to the last bits of log / sincos.
#pragma once
#include <cstdint>

#include "block_engine.cuh"

namespace hqmc {

struct Philox4 { uint32_t x[4]; };

__host__ __device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    Philox4 o; o.x[0] = c0; o.x[1] = c1; o.x[2] = c2; o.x[3] = c3;
    return o;
}
__host__ __device__ __forceinline__ Philox4 rng_block(unsigned long long seed, uint32_t update, uint32_t stream, unsigned long long i) {
    return philox4x32_10((uint32_t)i, (uint32_t)(i >> 32), stream, update, (uint32_t)seed, (uint32_t)(seed >> 32));
}
__host__ __device__ __forceinline__ double rng_u53(uint32_t a, uint32_t b) {
    return ((double)(a >> 5) * 67108864.0 + (double)(b >> 6)) * (1.0 / 9007199254740992.0);
}

// MODE 0: the four raw words (uint32 out[4 n]); 1: the Gaussian pair as doubles (out[2 n]); 2: as one complex number of
// the vector type T (out[n])
template <typename T, int MODE>
__global__ void k_rng(unsigned long long seed, uint32_t update, uint32_t stream, size_t n, void *__restrict__ out) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const Philox4 b = rng_block(seed, update, stream, i);
        if (MODE == 0) {
            reinterpret_cast<uint4 *>(out)[i] = make_uint4(b.x[0], b.x[1], b.x[2], b.x[3]);
        } else {
            const double u1 = rng_u53(b.x[0], b.x[1]), u2 = rng_u53(b.x[2], b.x[3]);
            const double r = sqrt(-log(1.0 - u1));
            double s, c;
            sincos(6.283185307179586476925286766559 * u2, &s, &c);
            if (MODE == 1) reinterpret_cast<double2 *>(out)[i] = make_double2(r * c, r * s);
            else { typename Cx<T>::type z; z.x = (T)(r * c); z.y = (T)(r * s); reinterpret_cast<typename Cx<T>::type *>(out)[i] = z; }
        }
    }
}

}  // namespace hqmc
