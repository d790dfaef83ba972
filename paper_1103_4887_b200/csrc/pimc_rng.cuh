// Counter-based random numbers for the PIMC kernels (row A1 of SURVEY.md §8(a)).
// Philox4x32-10 as published by Salmon, Moraes, Dror and Shaw (SC'11); stateless, so the draw for
// (seed, sweep, chain, site-or-parameter, stream) is the same whatever thread computes it.
// Replaces the per-thread "Hybrid Tausworthe" generator of PAPER.md:234.
#pragma once
#include <cstdint>

#include "pimc_math.cuh"

namespace pimc {

enum : uint32_t { kStreamStateProposal = 0, kStreamStateAccept = 1, kStreamParam = 2 };

struct Words4 { uint32_t w[4]; };

__device__ __forceinline__ Words4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                 uint32_t k0, uint32_t k1) {
    constexpr uint32_t kMulA = 0xD2511F53u, kMulB = 0xCD9E8D57u;
    constexpr uint32_t kWeylA = 0x9E3779B9u, kWeylB = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hiA = __umulhi(kMulA, c0), loA = kMulA * c0;
        const uint32_t hiB = __umulhi(kMulB, c2), loB = kMulB * c2;
        c0 = hiB ^ c1 ^ k0;
        c1 = loB;
        c2 = hiA ^ c3 ^ k1;
        c3 = loA;
        k0 += kWeylA;
        k1 += kWeylB;
    }
    Words4 o;
    o.w[0] = c0; o.w[1] = c1; o.w[2] = c2; o.w[3] = c3;
    return o;
}

// counter = (index, sweep low word, chain, stream | block << 8 | (sweep high bits) << 16); key = seed.
__device__ __forceinline__ Words4 draw(uint64_t seed, uint64_t sweep, uint32_t chain, uint32_t index,
                                        uint32_t stream, uint32_t block) {
    return philox4x32_10(index, (uint32_t)sweep, chain, stream | (block << 8) | ((uint32_t)(sweep >> 32) << 16),
                         (uint32_t)seed, (uint32_t)(seed >> 32));
}

// Uniforms strictly inside (0,1), exactly representable in the target type.
__device__ __forceinline__ double unit_open(uint32_t w) { return (__uint2double_rn(w) + 0.5) * 0x1p-32; }
__device__ __forceinline__ double unit_open52(uint32_t w0, uint32_t w1) {
    const unsigned long long v = (((unsigned long long)w1 << 32) | (unsigned long long)w0) >> 12;
    return (__ull2double_rn(v) + 0.5) * 0x1p-52;
}
__device__ __forceinline__ float unit_openf(uint32_t w) { return (__uint2float_rn(w >> 9) + 0.5f) * 0x1p-23f; }

// Box-Muller pair from two uniforms: radius sqrt(-2 ln u1), angle 2 pi u2.
__device__ __forceinline__ void normal_pair(double u1, double u2, double& z0, double& z1) {
    const double radius = sqrt_fast(-2.0 * log_fast(u1));
    double s, c;
    sincos_fast(6.283185307179586476925286766559 * u2, s, c);
    z0 = radius * c;
    z1 = radius * s;
}
__device__ __forceinline__ void normal_pair(float u1, float u2, float& z0, float& z1) {
    const float radius = sqrtf(-2.0f * logf(u1));
    float s, c;
    sincosf(6.283185307179586476925286766559f * u2, &s, &c);
    z0 = radius * c;
    z1 = radius * s;
}

}  // namespace pimc
