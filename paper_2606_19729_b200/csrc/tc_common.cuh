// tc_common.cuh -- device helpers shared by the tcgen05 kernels (rollout_tc.cu, rollout_tc2.cu):
// operand-buffer addressing, fused activation epilogue of a hidden chunk, Philox noise packing,
// non-quadratic rewards from the packed bf16 state.
#pragma once
#include "sm100_ptx.cuh"
#include "tc_program.h"
#include "voila_device.cuh"
#include "voila_internal.h"

namespace voila {
namespace tcc {

using namespace ptx;

__device__ __forceinline__ float bf16lo(uint32_t v) { return __uint_as_float(v << 16); }
__device__ __forceinline__ float bf16hi(uint32_t v) { return __uint_as_float(v & 0xffff0000u); }

__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d)
                 : "memory");
}

// Address of the 16-byte unit holding operand columns [8*unit8, 8*unit8+8) of `row` (unit8 counts
// 8-column units across the whole operand; chunk = unit8 / 8).
__device__ __forceinline__ uint32_t a_unit_addr(uint32_t a_base, int row, int unit8) {
    const int chunk = unit8 >> 3, u = unit8 & 7;
    return a_base + chunk * kTcChunkBytes + row * 128 + ((u ^ (row & 7)) << 4);
}

template <int ACT>
__device__ __forceinline__ float act_fast(float x) {
    if (ACT == VOILA_ACT_RELU) return fmaxf(x, 0.0f);
    if (ACT == VOILA_ACT_SILU) {
        const float h = 0.5f * x;  // x * sigmoid(x) = h + h * tanh(h)
        return fmaf(h, tanh_approx(h), h);
    }
    return x;
}

// One 64-column chunk of a hidden layer for this warp's 32 rows x 32 columns.
template <int ACT>
__device__ __forceinline__ void hidden_chunk(uint32_t taddr, const float *__restrict__ bias, uint32_t row_addr,
                                             int row, int half) {
    uint32_t v[32];
    tmem_ld32(taddr, v);
    float4 b[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) b[i] = __ldg(reinterpret_cast<const float4 *>(bias) + i);
    tmem_ld_wait();
    uint32_t o[16];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float y0 = act_fast<ACT>(__uint_as_float(v[4 * i + 0]) + b[i].x);
        const float y1 = act_fast<ACT>(__uint_as_float(v[4 * i + 1]) + b[i].y);
        const float y2 = act_fast<ACT>(__uint_as_float(v[4 * i + 2]) + b[i].z);
        const float y3 = act_fast<ACT>(__uint_as_float(v[4 * i + 3]) + b[i].w);
        o[2 * i] = pack_bf16x2(y0, y1);
        o[2 * i + 1] = pack_bf16x2(y2, y3);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int unit = half * 4 + u;
        st_shared_v4(row_addr + ((unit ^ (row & 7)) << 4), o[4 * u], o[4 * u + 1], o[4 * u + 2], o[4 * u + 3]);
    }
}

// Nz (<= 32, multiple of 8) standard normals of (seed; p, q, t, stream) packed as bf16 pairs.
__device__ __forceinline__ void gen_noise(uint32_t (&nz)[16], uint64_t seed, uint32_t p, uint32_t q,
                                          uint32_t t, uint32_t stream, int Nz) {
#pragma unroll
    for (int b = 0; b < 8; ++b) {
        if (4 * b < Nz) {
            float z[4];
            normals4<true>(seed, p, q, t, stream, (uint32_t)b, z);
            nz[2 * b] = pack_bf16x2(z[0], z[1]);
            nz[2 * b + 1] = pack_bf16x2(z[2], z[3]);
        }
    }
}

// Eight normals (Philox blocks 2u and 2u+1) packed as one 16-byte operand unit.  Deliberately NOT
// inlined: the Philox rounds + Box-Muller of a block are ~160 instructions, and the pair kernel
// draws noise at several places of its epilogue; one copy keeps the kernel inside the instruction
// cache (the inlined form was 3/4 of the kernel's SASS).
static __device__ __noinline__ uint4 noise_unit8(uint64_t seed, uint32_t p, uint32_t q, uint32_t t, uint32_t stream,
                                          uint32_t u) {
    float z[8];
    normals4<true>(seed, p, q, t, stream, 2u * u, z);
    normals4<true>(seed, p, q, t, stream, 2u * u + 1u, z + 4);
    return make_uint4(pack_bf16x2(z[0], z[1]), pack_bf16x2(z[2], z[3]), pack_bf16x2(z[4], z[5]),
                      pack_bf16x2(z[6], z[7]));
}
// Four fp32 normals of one Philox block (same fast intrinsics as noise_unit8); not inlined either.
static __device__ __noinline__ float4 normals_f4(uint64_t seed, uint32_t p, uint32_t q, uint32_t t, uint32_t stream,
                                                 uint32_t blk) {
    float z[4];
    normals4<true>(seed, p, q, t, stream, blk, z);
    return make_float4(z[0], z[1], z[2], z[3]);
}
__device__ __forceinline__ void gen_noise_call(uint32_t (&nz)[16], uint64_t seed, uint32_t p, uint32_t q,
                                               uint32_t t, uint32_t stream, int Nz) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        if (8 * u < Nz) {
            const uint4 v = noise_unit8(seed, p, q, t, stream, (uint32_t)u);
            nz[4 * u] = v.x; nz[4 * u + 1] = v.y; nz[4 * u + 2] = v.z; nz[4 * u + 3] = v.w;
        }
    }
}

// One 8-column unit (16 bytes) of a public bf16 row of S_io columns: rows whose length is a multiple
// of 8 are 16-byte aligned and move as one vector; other lengths (paper-shaped states, S = 39 / 45) go
// element by element with the tail zero-filled / masked.
__device__ __forceinline__ uint4 load_row_unit(const uint16_t *__restrict__ row, int S_io, int u) {
    if ((S_io & 7) == 0) return __ldg(reinterpret_cast<const uint4 *>(row) + u);
    uint32_t w[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const int c = 8 * u + 2 * e;
        const uint32_t lo = c < S_io ? (uint32_t)__ldg(row + c) : 0u;
        const uint32_t hi = c + 1 < S_io ? (uint32_t)__ldg(row + c + 1) : 0u;
        w[e] = lo | (hi << 16);
    }
    return make_uint4(w[0], w[1], w[2], w[3]);
}
__device__ __forceinline__ void store_row_unit(uint16_t *row, int S_io, int u, uint4 v) {
    if ((S_io & 7) == 0) {
        *(reinterpret_cast<uint4 *>(row) + u) = v;
        return;
    }
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const int c = 8 * u + 2 * e;
        if (c < S_io) row[c] = (uint16_t)(w[e] & 0xffffu);
        if (c + 1 < S_io) row[c + 1] = (uint16_t)(w[e] >> 16);
    }
}

// R(s, a) from the bf16 state for the non-quadratic reward kinds (R14).
__device__ __forceinline__ float reward_from_state(const uint32_t *st, int S, int kind,
                                                   const float *__restrict__ param) {
    float acc = 0.0f;
#pragma unroll
    for (int c2 = 0; c2 < 32; ++c2) {
        if (2 * c2 < S) {  // S: the PUBLIC state width (an odd S leaves the last pair half used)
            const bool two = 2 * c2 + 1 < S;
            const float s0 = bf16lo(st[c2]), s1 = bf16hi(st[c2]);
            const float p0 = __ldg(param + 2 * c2), p1 = two ? __ldg(param + 2 * c2 + 1) : 0.0f;
            if (kind == VOILA_R_NEG_L2_GOAL) {
                acc = fmaf(s0 - p0, s0 - p0, acc);
                if (two) acc = fmaf(s1 - p1, s1 - p1, acc);
            } else {
                acc = fmaf(p0, s0, acc);
                if (two) acc = fmaf(p1, s1, acc);
            }
        }
    }
    return kind == VOILA_R_NEG_L2_GOAL ? -sqrtf(acc) : acc + __ldg(param + S);
}

}  // namespace tcc
}  // namespace voila
