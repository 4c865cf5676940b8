// voila_device.cuh -- device-side helpers shared by libvoila's kernels (noise, rounding, ordering).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace voila {

// Noise streams (reading R3): which Philox stream feeds which random input.
constexpr uint32_t kStreamRolloutT = 1u;
constexpr uint32_t kStreamRolloutZ = 2u;
constexpr uint32_t kStreamBeliefT = 3u;
constexpr uint32_t kStreamResample = 4u;
constexpr uint32_t kStreamPwObs = 5u;     // progressive widening: noise of the sampled observation
constexpr uint32_t kStreamPwAttach = 6u;  // progressive widening: word that picks an existing branch
constexpr uint32_t kStreamDiffusion = 7u;  // diffusion teacher: the initial noise x_1 = omega

// Philox4x32-10 (Salmon et al., SC'11): counter-based generator, one 128-bit block per call.
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

// Counter layout (R3): key = seed, counter = (p, q, t, stream << 16 | blk).
__device__ __forceinline__ uint4 noise_words(uint64_t seed, uint32_t p, uint32_t q, uint32_t t,
                                             uint32_t stream, uint32_t blk) {
    return philox4x32_10(make_uint4(p, q, t, (stream << 16) | blk),
                         make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)));
}

// 32-bit word -> uniform in (0, 1] (R4): u = x * 2^-32 + 2^-33, x converted round-to-nearest.
__device__ __forceinline__ float u01(uint32_t x) {
    return fmaf(__uint2float_rn(x), 2.3283064365386963e-10f, 1.1641532182693481e-10f);
}

// Box-Muller on a word pair (R4).  FAST = approximate intrinsics (bf16 tensor-core mode only;
// their error is far below bf16 resolution).
template <bool FAST>
__device__ __forceinline__ void box_muller(uint32_t xa, uint32_t xb, float &z0, float &z1) {
    const float ua = u01(xa), ub = u01(xb);
    if (FAST) {
        const float r = sqrtf(-2.0f * __logf(ua));
        float s, c;
        __sincosf(6.283185307179586f * ub, &s, &c);
        z0 = r * c;
        z1 = r * s;
    } else {
        const float r = sqrtf(-2.0f * logf(ua));
        const float ang = 6.283185307179586f * ub;
        z0 = r * cosf(ang);
        z1 = r * sinf(ang);
    }
}

template <bool FAST>
__device__ __forceinline__ void normals4(uint64_t seed, uint32_t p, uint32_t q, uint32_t t,
                                         uint32_t stream, uint32_t blk, float z[4]) {
    const uint4 x = noise_words(seed, p, q, t, stream, blk);
    box_muller<FAST>(x.x, x.y, z[0], z[1]);
    box_muller<FAST>(x.z, x.w, z[2], z[3]);
}

// fp32 -> nearest bf16 (ties to even), returned as fp32 / as 16-bit pattern.
__device__ __forceinline__ uint16_t bf16_bits(float x) {
    uint32_t u = __float_as_uint(x);
    if ((u & 0x7f800000u) == 0x7f800000u) return (uint16_t)(u >> 16);
    u += 0x7fffu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}
__device__ __forceinline__ float bf16_round(float x) {
    return __uint_as_float(((uint32_t)bf16_bits(x)) << 16);
}
__device__ __forceinline__ float bf16_to_float(uint16_t b) {
    return __uint_as_float(((uint32_t)b) << 16);
}

// Order-preserving map float -> int32 so that atomicMax on ints is a float max.  Any NaN maps to INT_MAX
// (above +inf) so that a NaN score poisons the maximum and is flagged downstream.
__device__ __forceinline__ int float_to_ordered(float f) {
    if (f != f) return 0x7fffffff;
    const int i = __float_as_int(f);
    return i >= 0 ? i : i ^ 0x7fffffff;
}
__device__ __forceinline__ float ordered_to_float(int i) {
    return __int_as_float(i >= 0 ? i : i ^ 0x7fffffff);
}

// An action index as the kernels use it: clamped into [0, A), so that an out-of-range entry of
// action_seqs can never index past the per-action tables (voila.h: such entries are clamped).
__device__ __forceinline__ int clamp_action(int a, int A) { return a < 0 ? 0 : (a >= A ? A - 1 : a); }

__device__ __forceinline__ float act_apply(float x, int act) {
    if (act == 1) return x > 0.0f ? x : 0.0f;
    if (act == 2) return x / (1.0f + expf(-x));
    return x;
}

}  // namespace voila
