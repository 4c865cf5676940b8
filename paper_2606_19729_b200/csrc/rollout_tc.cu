// rollout_tc.cu -- tcgen05 / TMEM / bulk-copy path of libvoila (bf16 mode): the persistent fused-MLP
// rollout kernel.  See tc_program.h for the execution model.  Per CTA (one per SM, persistent over
// (sequence, 128-particle block) work units):
//   warp 0   producer: streams pre-swizzled weight tiles L2 -> shared-memory ring (cp.async.bulk)
//   warp 1   MMA issuer: one thread issues tcgen05.mma (M=128, N=bn, K=16, bf16 -> fp32 in TMEM)
//   warp 2   TMEM allocation
//   warps 4-11 epilogue: tcgen05.ld accumulator -> bias + activation -> bf16 -> operand buffer
//            (in place), Philox noise, reward / return accumulation, observation witness.
// The horizon loop never leaves the SM: HBM sees the particle tile once per work unit and the
// per-unit partial sums; weights come from L2.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <string>
#include <vector>

#include "tc_common.cuh"
#include "voila_kernels.h"

namespace voila {

namespace {

using namespace ptx;

#ifdef VOILA_TC_TRACE
__device__ unsigned long long g_tc_trace[32];
#define TRACE_T0() const long long _t0 = clock64()
#define TRACE_ADD(var) var += clock64() - _t0
#else
#define TRACE_T0()
#define TRACE_ADD(var)
#endif

struct TcRolloutParams {
    const uint8_t *wstream;
    const float *bias;
    const TcLayer *layers;
    const TcTile *tiles;
    TcProgramHeader hdr;
    const uint16_t *particles;  // [P][S] bf16
    const int32_t *seqs;        // [Q][H]
    const float *weights;       // [P] or nullptr
    int P, Q, H;
    uint64_t seed;
    double *part_value;    // [Q][tiles_per_q]
    double *part_witness;  // [Q][tiles_per_q][O] or nullptr
    float *returns_out;
    float *final_states_out;
    int tiles_per_q, n_units;
    int S, O, A, Nz;
    float gamma;
    int reward_kind;
    const float *reward_param;
    const float *action_cost;
};

// Shared-memory carve-up (offsets from the 1024-aligned base).
struct SmemMap {
    uint32_t a, ring, layers, tiles, bars, misc, total;
};
__host__ __device__ inline SmemMap smem_map(const TcProgramHeader &h) {
    SmemMap m;
    m.a = 0;
    m.ring = m.a + (uint32_t)h.a_chunks * kTcChunkBytes;
    m.layers = m.ring + (uint32_t)h.n_stages * kTcStageBytes;
    m.tiles = m.layers + kTcMaxLayers * (uint32_t)sizeof(TcLayer);
    m.bars = m.tiles + (((uint32_t)h.n_tiles * (uint32_t)sizeof(TcTile) + 15u) & ~15u);
    m.misc = m.bars + (8 + 8 + kTcEvtRing + 1) * 8;
    m.total = m.misc + 16 + 4 * 8 + 4 * 64 * 4;
    return m;
}

using namespace tcc;

__global__ void __launch_bounds__(kTcThreads, 1) rollout_tc_kernel(const TcRolloutParams p) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw_u32 = smem_u32(smem_raw);
    uint8_t *smem = smem_raw + (((raw_u32 + 1023u) & ~1023u) - raw_u32);
    const SmemMap map = smem_map(p.hdr);
    TcLayer *L = reinterpret_cast<TcLayer *>(smem + map.layers);
    TcTile *T = reinterpret_cast<TcTile *>(smem + map.tiles);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + map.bars);
    uint64_t *empty = full + 8;
    uint64_t *evt = empty + 8;
    uint64_t *layer_done = evt + kTcEvtRing;
    uint32_t *tmem_ptr = reinterpret_cast<uint32_t *>(smem + map.misc);
    double *red_g = reinterpret_cast<double *>(smem + map.misc + 16);
    float *red_w = reinterpret_cast<float *>(smem + map.misc + 16 + 4 * 8);
    const uint32_t a_u32 = smem_u32(smem + map.a), ring_u32 = smem_u32(smem + map.ring);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_layers = p.hdr.n_layers, n_tiles = p.hdr.n_tiles, n_stages = p.hdr.n_stages;

    // ---- one-time setup: program -> smem, zero the operand buffer, barriers, TMEM ----
    {
        const uint32_t *src = reinterpret_cast<const uint32_t *>(p.layers);
        uint32_t *dst = reinterpret_cast<uint32_t *>(L);
        for (int i = threadIdx.x; i < n_layers * (int)(sizeof(TcLayer) / 4); i += kTcThreads) dst[i] = src[i];
        src = reinterpret_cast<const uint32_t *>(p.tiles);
        dst = reinterpret_cast<uint32_t *>(T);
        for (int i = threadIdx.x; i < n_tiles * (int)(sizeof(TcTile) / 4); i += kTcThreads) dst[i] = src[i];
        uint4 *az = reinterpret_cast<uint4 *>(smem + map.a);
        for (int i = threadIdx.x; i < p.hdr.a_chunks * kTcChunkBytes / 16; i += kTcThreads)
            az[i] = make_uint4(0u, 0u, 0u, 0u);
        fence_proxy_async_smem();
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < 8; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 1);
        }
        for (int i = 0; i < kTcEvtRing; ++i) mbar_init(&evt[i], 8);
        mbar_init(layer_done, 1);
        fence_barrier_init();
    }
    if (warp == 2) {
        tmem_alloc(tmem_ptr, (uint32_t)p.hdr.tmem_cols);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    const int n_my_units = (p.n_units - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int total_steps = n_my_units * p.H;

    if (warp == 0) {
        // ===== producer: weight tiles, in the program's issue order, once per step =====
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            long long tr_empty = 0;
            const long long tr_start = clock64();
            for (int step = 0; step < total_steps; ++step) {
                for (int i = 0; i < n_tiles; ++i) {
                    {
                        TRACE_T0();
                        mbar_wait(&empty[stage], phase ^ 1u);
                        TRACE_ADD(tr_empty);
                    }
                    const uint32_t bytes = T[i].bytes;
                    mbar_arrive_expect_tx(&full[stage], bytes);
                    bulk_g2s(smem + map.ring + stage * kTcStageBytes, p.wstream + T[i].src_off, bytes,
                             &full[stage]);
                    if (++stage == (uint32_t)n_stages) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
            }
#ifdef VOILA_TC_TRACE
            if (blockIdx.x == 0) {
                g_tc_trace[0] = tr_empty;
                g_tc_trace[1] = clock64() - tr_start;
            }
#endif
            (void)tr_empty; (void)tr_start;
        }
    } else if (warp == 1) {
        // ===== MMA issuer: the warp walks the tile program converged (waits are warp-uniform); one
        // elected lane issues, so each tcgen05.mma / commit is ONE instruction (no ELECT loop) =====
        {
            uint32_t stage = 0, phase = 0;
            int waited = -1, base = 1;
            long long tr_evt = 0, tr_full = 0;
            const long long tr_start = clock64();
            for (int step = 0; step < total_steps; ++step) {
                for (int i = 0; i < n_tiles; ++i) {
                    const TcTile t = T[i];
                    const TcLayer &l = L[t.layer];
                    const int need = base + (int)t.need;
                    if (need > waited) {
                        TRACE_T0();
                        mbar_wait(&evt[need & (kTcEvtRing - 1)], (uint32_t)(need / kTcEvtRing) & 1u);
                        TRACE_ADD(tr_evt);
                        waited = need;
                    }
                    {
                        TRACE_T0();
                        mbar_wait(&full[stage], phase);
                        TRACE_ADD(tr_full);
                    }
                    tc_fence_after();
                    if (elect_one_sync()) {
                    const uint64_t ad = umma_desc_sw128(a_u32 + (uint32_t)t.kc * kTcChunkBytes);
                    const uint64_t bd = umma_desc_sw128(ring_u32 + stage * kTcStageBytes);
                    const uint32_t d = tmem_base + (uint32_t)t.n * l.bn;
#pragma unroll
                    for (int k = 0; k < 4; ++k)  // 64-wide chunk = 4 x (K = 16); +32 bytes per K step
                        umma_ss(d, ad + 2u * k, bd + 2u * k, l.idesc, (t.first && k == 0) ? 0u : 1u);
                    umma_commit(&empty[stage]);
                    if (t.last) umma_commit(layer_done);
                    }
                    __syncwarp();
                    if (++stage == (uint32_t)n_stages) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
                base += p.hdr.evt_per_step;
            }
#ifdef VOILA_TC_TRACE
            if (blockIdx.x == 0 && lane == 0) {
                g_tc_trace[2] = tr_evt;
                g_tc_trace[3] = tr_full;
                g_tc_trace[4] = clock64() - tr_start;
            }
#endif
            (void)tr_evt; (void)tr_full; (void)tr_start;
        }
    } else if (warp >= 4) {
        // ===== epilogue warps =====
        const int ew = warp - 4, qd = warp & 3, half = ew >> 2;
        const int row = qd * 32 + lane;
        const uint32_t lane_taddr = tmem_base + ((uint32_t)(qd * 32) << 16);
        const int S = p.S, O = p.O, Nz = p.Nz;
        const int in_units = p.hdr.in_chunks * 8;  // 8-column units of the step's input operand
        uint32_t persist[64];  // half 0: packed bf16 state (32 words); half 1: fp32 witness (64 words)
        uint32_t nz[16];
        float G = 0.0f, disc = 1.0f, w_row = 0.0f;
        int ev = 0, t = 0, unit_i = 0, q = 0, blk = 0, p_idx = 0;
        bool valid = false;
        uint32_t ld_phase = 0;

        auto arrive_event = [&]() {
            __syncwarp();
            if (lane == 0) mbar_arrive(&evt[ev & (kTcEvtRing - 1)]);
            ++ev;
        };
        long long tr_layer = 0;
        const long long tr_start = clock64();
        auto wait_layer = [&]() {
            TRACE_T0();
            mbar_wait(layer_done, ld_phase);
            TRACE_ADD(tr_layer);
            ld_phase ^= 1u;
            tc_fence_after();
        };
        auto load_unit = [&]() {
            const int unit = (int)blockIdx.x + unit_i * (int)gridDim.x;
            q = unit / p.tiles_per_q;
            blk = unit - q * p.tiles_per_q;
            p_idx = blk * kTcRows + row;
            valid = p_idx < p.P;
            w_row = valid ? (p.weights ? __ldg(p.weights + p_idx) : 1.0f) : 0.0f;
            G = 0.0f;
            disc = 1.0f;
            t = 0;
            if (half == 0) {
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    uint4 v = make_uint4(0u, 0u, 0u, 0u);
                    if (8 * u < S && valid)
                        v = __ldg(reinterpret_cast<const uint4 *>(p.particles + (size_t)p_idx * S) + u);
                    persist[4 * u] = v.x; persist[4 * u + 1] = v.y;
                    persist[4 * u + 2] = v.z; persist[4 * u + 3] = v.w;
                }
            } else {
#pragma unroll
                for (int c = 0; c < 64; ++c) persist[c] = 0u;
            }
        };
        // Writes the generator input [s ; w ; 0] of the next layer-1 into the operand buffer: the
        // `state_half` warps write the state units, the other half the noise and padding units.
        auto write_input = [&](int state_half, int noise_half) {
            if (half == state_half) {
#pragma unroll
                for (int u = 0; u < 8; ++u)
                    if (8 * u < S)
                        st_shared_v4(a_unit_addr(a_u32, row, u), persist[4 * u], persist[4 * u + 1],
                                     persist[4 * u + 2], persist[4 * u + 3]);
            }
            if (half == noise_half) {
                const int u0 = S >> 3;
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (8 * u < Nz)
                        st_shared_v4(a_unit_addr(a_u32, row, u0 + u), nz[4 * u], nz[4 * u + 1], nz[4 * u + 2],
                                     nz[4 * u + 3]);
                for (int u = u0 + (Nz >> 3); u < in_units; ++u)
                    st_shared_v4(a_unit_addr(a_u32, row, u), 0u, 0u, 0u, 0u);
            }
        };
        auto step_reward = [&]() {  // non-quadratic reward kinds: R(s_t, a_t) from the state words
            if (half == 0 && p.reward_kind != VOILA_R_NEG_QUADRATIC) {
                float r = reward_from_state(persist, S, p.reward_kind, p.reward_param);
                if (p.action_cost) r += __ldg(p.action_cost + clamp_action(__ldg(p.seqs + (size_t)q * p.H + t), p.A));
                G = fmaf(disc, r, G);
            }
        };

        if (n_my_units > 0) {
            load_unit();
            if (half == 0) gen_noise(nz, p.seed, (uint32_t)p_idx, (uint32_t)q, 0u, kStreamRolloutT, Nz);
            write_input(0, 0);
            step_reward();
            fence_proxy_async_smem();
            arrive_event();
        }
        for (int step = 0; step < total_steps; ++step) {
            const int a_t = clamp_action(__ldg(p.seqs + (size_t)q * p.H + t), p.A);
            for (int li = 0; li < n_layers; ++li) {
                const TcLayer l = L[li];
                const float *bias = p.bias + l.bias_off + (l.bias_per_action ? (size_t)a_t * l.n_pad : 0);
                if (l.epi == TC_EPI_HIDDEN) {
                    wait_layer();
                    const int chunks = l.n_pad >> 6;
                    for (int j = 0; j < chunks; ++j) {
                        const uint32_t taddr = lane_taddr + (uint32_t)(64 * j + 32 * half);
                        const uint32_t row_addr = a_u32 + j * kTcChunkBytes + row * 128;
                        const float *bj = bias + 64 * j + 32 * half;
                        if (l.act == VOILA_ACT_SILU) hidden_chunk<VOILA_ACT_SILU>(taddr, bj, row_addr, row, half);
                        else if (l.act == VOILA_ACT_RELU) hidden_chunk<VOILA_ACT_RELU>(taddr, bj, row_addr, row, half);
                        else hidden_chunk<VOILA_ACT_NONE>(taddr, bj, row_addr, row, half);
                        fence_proxy_async_smem();
                        tc_fence_before();
                        arrive_event();
                    }
                } else if (l.epi == TC_EPI_REWARD) {
                    wait_layer();
                    if (half == 0) {
                        float r = 0.0f;
#pragma unroll
                        for (int g = 0; g < 4; ++g) {
                            if (16 * g < (int)l.n_pad) {
                                uint32_t v[16];
                                tmem_ld16(lane_taddr + 16 * g, v);
                                tmem_ld_wait();
#pragma unroll
                                for (int c = 0; c < 16; c += 2) {
                                    const uint32_t sw = persist[(16 * g + c) >> 1];
                                    r = fmaf(bf16lo(sw), __uint_as_float(v[c]), r);
                                    r = fmaf(bf16hi(sw), __uint_as_float(v[c + 1]), r);
                                }
                            }
                        }
                        r = -r;
                        if (p.action_cost) r += __ldg(p.action_cost + a_t);
                        G = fmaf(disc, r, G);
                    }
                    tc_fence_before();
                    arrive_event();
                } else if (l.epi == TC_EPI_STATE) {
                    // w_Z(t) is independent of the state: draw it while the output layer's MMAs run
                    if (half == 1) gen_noise(nz, p.seed, (uint32_t)p_idx, (uint32_t)q, (uint32_t)t, kStreamRolloutZ, Nz);
                    wait_layer();
                    if (half == 0) {
#pragma unroll
                        for (int g = 0; g < 4; ++g) {
                            if (16 * g < (int)l.n_pad) {
                                uint32_t v[16];
                                tmem_ld16(lane_taddr + 16 * g, v);
                                float4 b[4];
#pragma unroll
                                for (int i = 0; i < 4; ++i) b[i] = __ldg(reinterpret_cast<const float4 *>(bias + 16 * g) + i);
                                tmem_ld_wait();
#pragma unroll
                                for (int i = 0; i < 4; ++i) {
                                    persist[8 * g + 2 * i] = pack_bf16x2(__uint_as_float(v[4 * i]) + b[i].x,
                                                                        __uint_as_float(v[4 * i + 1]) + b[i].y);
                                    persist[8 * g + 2 * i + 1] = pack_bf16x2(__uint_as_float(v[4 * i + 2]) + b[i].z,
                                                                            __uint_as_float(v[4 * i + 3]) + b[i].w);
                                }
                            }
                        }
                    }
                    write_input(0, 1);
                    fence_proxy_async_smem();
                    tc_fence_before();
                    arrive_event();
                } else {  // TC_EPI_OBS: last layer of the step
                    const bool last_step = (t == p.H - 1);
                    if (half == 0 && !last_step)
                        gen_noise(nz, p.seed, (uint32_t)p_idx, (uint32_t)q, (uint32_t)(t + 1), kStreamRolloutT, Nz);
                    wait_layer();
                    if (half == 1) {
#pragma unroll
                        for (int g = 0; g < 4; ++g) {
                            if (16 * g < (int)l.n_pad) {
                                uint32_t v[16];
                                tmem_ld16(lane_taddr + 16 * g, v);
                                float4 b[4];
#pragma unroll
                                for (int i = 0; i < 4; ++i) b[i] = __ldg(reinterpret_cast<const float4 *>(bias + 16 * g) + i);
                                tmem_ld_wait();
#pragma unroll
                                for (int i = 0; i < 4; ++i) {
                                    const float o0 = __uint_as_float(v[4 * i]) + b[i].x, o1 = __uint_as_float(v[4 * i + 1]) + b[i].y;
                                    const float o2 = __uint_as_float(v[4 * i + 2]) + b[i].z, o3 = __uint_as_float(v[4 * i + 3]) + b[i].w;
                                    const int c0 = 16 * g + 4 * i;
                                    persist[c0] = __float_as_uint(fmaf(disc, o0, __uint_as_float(persist[c0])));
                                    persist[c0 + 1] = __float_as_uint(fmaf(disc, o1, __uint_as_float(persist[c0 + 1])));
                                    persist[c0 + 2] = __float_as_uint(fmaf(disc, o2, __uint_as_float(persist[c0 + 2])));
                                    persist[c0 + 3] = __float_as_uint(fmaf(disc, o3, __uint_as_float(persist[c0 + 3])));
                                }
                            }
                        }
                    }
                    ++t;
                    disc *= p.gamma;
                    if (last_step) {
                        // ---- work unit finished: per-(q, tile) weighted partial sums, fixed order ----
                        if (half == 0) {
                            double v = valid ? (double)w_row * (double)G : 0.0;
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                            if (lane == 0) red_g[qd] = v;
                            if (valid && p.returns_out) p.returns_out[(size_t)q * p.P + p_idx] = G;
                            if (valid && p.final_states_out) {
                                float *fs = p.final_states_out + ((size_t)q * p.P + p_idx) * S;
#pragma unroll
                                for (int c2 = 0; c2 < 32; ++c2)
                                    if (2 * c2 < S) {
                                        fs[2 * c2] = bf16lo(persist[c2]);
                                        fs[2 * c2 + 1] = bf16hi(persist[c2]);
                                    }
                            }
                        } else if (p.part_witness) {
#pragma unroll
                            for (int c = 0; c < 64; ++c) {
                                if (c < O) {
                                    float x = w_row * __uint_as_float(persist[c]);
#pragma unroll
                                    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
                                    if (lane == 0) red_w[qd * 64 + c] = x;
                                }
                            }
                        }
                        named_bar_sync(1, 256);
                        if (ew == 0 && lane == 0)
                            p.part_value[(size_t)q * p.tiles_per_q + blk] = (red_g[0] + red_g[1]) + (red_g[2] + red_g[3]);
                        if (ew == 4 && p.part_witness) {
                            for (int c = lane; c < O; c += 32)
                                p.part_witness[((size_t)q * p.tiles_per_q + blk) * O + c] =
                                    ((double)red_w[c] + (double)red_w[64 + c]) +
                                    ((double)red_w[128 + c] + (double)red_w[192 + c]);
                        }
                        named_bar_sync(1, 256);
                        ++unit_i;
                        if (unit_i < n_my_units) {
                            load_unit();
                            if (half == 0) gen_noise(nz, p.seed, (uint32_t)p_idx, (uint32_t)q, 0u, kStreamRolloutT, Nz);
                        }
                    }
                    if (unit_i < n_my_units) {
                        write_input(0, 0);
                        step_reward();
                    }
                    fence_proxy_async_smem();
                    tc_fence_before();
                    arrive_event();
                }
            }
        }
#ifdef VOILA_TC_TRACE
        if (blockIdx.x == 0 && lane == 0) {
            g_tc_trace[8 + 2 * ew] = tr_layer;
            g_tc_trace[9 + 2 * ew] = clock64() - tr_start;
        }
#endif
        (void)tr_layer; (void)tr_start;
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc(tmem_base, (uint32_t)p.hdr.tmem_cols);
}

}  // namespace

// =====================================================================================
// Host side: program construction (weight packing, issue order), context, launchers
// =====================================================================================
namespace {

constexpr size_t kMaxDynSmem = 232448;  // 227 KB per CTA on sm_100

uint16_t host_bf16_bits(float x) {
    uint32_t u;
    std::memcpy(&u, &x, 4);
    if ((u & 0x7f800000u) != 0x7f800000u) u += 0x7fffu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}
float host_bf16_round(float x) {
    const uint32_t u = (uint32_t)host_bf16_bits(x) << 16;
    float y;
    std::memcpy(&y, &u, 4);
    return y;
}
int round_up(int x, int m) { return (x + m - 1) / m * m; }

struct ProgramBuilder {
    std::vector<TcLayer> layers;
    std::vector<TcTile> tiles;
    std::vector<uint8_t> wstream;
    std::vector<float> bias;
    int evt = 0;                       // next event index, relative to the step's first event
    int col_free[512];                 // event after which accumulator column c may be overwritten
    int a_ready[8];                    // event after which operand chunk k holds the next layer's input
    int a_chunks = 1;

    ProgramBuilder() {
        for (int &c : col_free) c = -1;
        for (int &a : a_ready) a = -1;
    }

    // W: [n0][k0] row-major fp32 (already in "algorithmic" column order); bias_rows x n0 biases.
    void add_layer(const float *W, int n0, int k0, const float *b, int bias_rows, int epi, int act) {
        TcLayer l{};
        const bool hidden = epi == TC_EPI_HIDDEN;
        const int k_pad = round_up(k0, 64);
        const int n_pad = hidden ? n0 : round_up(n0, 16);
        const int bn = (n_pad % 128 == 0) ? 128 : (n_pad <= 128 ? n_pad : 64);
        l.idesc = umma_idesc_bf16_m128((uint32_t)bn);
        l.bias_off = (uint32_t)bias.size();
        l.n_pad = (uint16_t)n_pad;
        l.bn = (uint16_t)bn;
        l.kc = (uint16_t)(k_pad / 64);
        l.epi = (uint8_t)epi;
        l.act = (uint8_t)act;
        l.bias_per_action = bias_rows > 1;
        for (int r = 0; r < bias_rows; ++r)
            for (int j = 0; j < n_pad; ++j) bias.push_back((b && j < n0) ? b[(size_t)r * n0 + j] : 0.0f);
        a_chunks = std::max(a_chunks, std::max((int)l.kc, hidden ? n_pad / 64 : 1));
        const int li = (int)layers.size();
        std::vector<TcTile> lt;
        for (int n = 0; n < n_pad / bn; ++n)
            for (int kc = 0; kc < l.kc; ++kc) {
                TcTile t{};
                t.src_off = (uint32_t)wstream.size();
                t.bytes = (uint32_t)bn * 128u;
                t.layer = (uint8_t)li;
                t.n = (uint8_t)n;
                t.kc = (uint8_t)kc;
                int need = a_ready[kc];
                for (int c = n * bn; c < (n + 1) * bn; ++c) need = std::max(need, col_free[c]);
                t.need = (int16_t)need;
                // pack the tile: bn rows x 64 columns, 128-byte rows, 16-byte units XOR (row & 7)
                wstream.resize(wstream.size() + t.bytes, 0);
                uint8_t *dst = wstream.data() + t.src_off;
                for (int i = 0; i < bn; ++i)
                    for (int u = 0; u < 8; ++u)
                        for (int e = 0; e < 8; ++e) {
                            const int row = n * bn + i, k = kc * 64 + u * 8 + e;
                            const float v = (row < n0 && k < k0) ? W[(size_t)row * k0 + k] : 0.0f;
                            const uint16_t h = host_bf16_bits(v);
                            std::memcpy(dst + i * 128 + ((u ^ (i & 7)) * 16) + e * 2, &h, 2);
                        }
                lt.push_back(t);
            }
        std::stable_sort(lt.begin(), lt.end(), [](const TcTile &x, const TcTile &y) { return x.need < y.need; });
        bool seen[8] = {false, false, false, false, false, false, false, false};
        for (TcTile &t : lt) {
            t.first = seen[t.n] ? 0 : 1;
            seen[t.n] = true;
        }
        lt.back().last = 1;
        tiles.insert(tiles.end(), lt.begin(), lt.end());
        layers.push_back(l);
        // events this layer's epilogue publishes
        if (hidden) {
            for (int j = 0; j < n_pad / 64; ++j) {
                for (int c = 64 * j; c < 64 * j + 64; ++c) col_free[c] = evt;
                a_ready[j] = evt;
                ++evt;
            }
        } else {
            for (int c = 0; c < n_pad; ++c) col_free[c] = evt;
            if (epi != TC_EPI_REWARD && epi != TC_EPI_SCORE)
                for (int &a : a_ready) a = evt;  // the next layer-1 input is written with this event
            ++evt;
        }
    }
};

struct TcHandle {
    TcProgramHeader hdr{};
    void *d_wstream = nullptr, *d_bias = nullptr, *d_layers = nullptr, *d_tiles = nullptr;
    size_t smem_bytes = 0;
    int sm_count = 0;
    size_t wstream_bytes = 0;
};

bool mlp_fits_tc(const voila_mlp &f, std::string *why) {
    if (f.n_layers < 2) {
        if (why) *why = "generator needs at least one hidden layer";
        return false;
    }
    for (int l = 1; l < f.n_layers; ++l)
        if (f.dims[l] % 64 != 0 || f.dims[l] > 512) {
            if (why) *why = "hidden widths must be multiples of 64, at most 512";
            return false;
        }
    return true;
}

// Generator layers -> program layers.  Layer 1 sees the "algorithmic" input [s ; w] (K = S + Nz):
// the one-hot block is folded into a per-action bias row b1 + W1[:, S + a].
void add_generator(ProgramBuilder &pb, const voila_mlp &f, int S, int A, int Nz, int last_epi) {
    for (int l = 0; l < f.n_layers; ++l) {
        const int K = f.dims[l], N = f.dims[l + 1];
        const bool last = l == f.n_layers - 1;
        if (l == 0) {
            const int k0 = S + Nz;
            std::vector<float> W((size_t)N * k0), b((size_t)A * N);
            for (int j = 0; j < N; ++j) {
                for (int k = 0; k < S; ++k) W[(size_t)j * k0 + k] = f.W[0][(size_t)j * K + k];
                for (int k = 0; k < Nz; ++k) W[(size_t)j * k0 + S + k] = f.W[0][(size_t)j * K + S + A + k];
                for (int a = 0; a < A; ++a)
                    b[(size_t)a * N + j] = f.b[0][j] + host_bf16_round(f.W[0][(size_t)j * K + S + a]);
            }
            pb.add_layer(W.data(), N, k0, b.data(), A, last ? last_epi : TC_EPI_HIDDEN, f.act);
        } else {
            pb.add_layer(f.W[l], N, K, f.b[l], 1, last ? last_epi : TC_EPI_HIDDEN, f.act);
        }
    }
}

}  // namespace

bool tc_supported(const voila_model_desc *d, std::string *why) {
    const int S = d->state_dim, O = d->obs_dim, Nz = d->noise_dim;
    auto fail = [&](const char *m) {
        if (why) *why = m;
        return false;
    };
    if (d->prec != VOILA_PREC_BF16) return fail("tcgen05 path is the bf16 mode");
    if (S % 8 != 0 || S > 64) return fail("state_dim must be a multiple of 8, at most 64");
    if (O > 64) return fail("obs_dim must be at most 64");
    if (Nz % 8 != 0 || Nz > 32 || Nz < 8) return fail("noise_dim must be 8, 16, 24 or 32");
    if (!mlp_fits_tc(d->f_T, why) || !mlp_fits_tc(d->f_Z, why)) return false;
    return true;
}

void *tc_create(const voila_model_desc *d, int sm_count, std::vector<void *> *allocs, std::string *err) {
    const int S = d->state_dim, A = d->n_actions, Nz = d->noise_dim;
    ProgramBuilder pb;
    if (d->reward.kind == VOILA_R_NEG_QUADRATIC)  // u = M s on the tensor pipe, r = -s^T u in the epilogue
        pb.add_layer(d->reward.param, S, S, nullptr, 1, TC_EPI_REWARD, VOILA_ACT_NONE);
    add_generator(pb, d->f_T, S, A, Nz, TC_EPI_STATE);
    add_generator(pb, d->f_Z, S, A, Nz, TC_EPI_OBS);
    if ((int)pb.layers.size() > kTcMaxLayers || (int)pb.tiles.size() > kTcMaxTiles) {
        if (err) *err = "model too deep for the tcgen05 program tables";
        return nullptr;
    }
    TcHandle *h = new TcHandle();
    h->sm_count = sm_count;
    h->hdr.n_layers = (int)pb.layers.size();
    h->hdr.n_tiles = (int)pb.tiles.size();
    h->hdr.evt_per_step = pb.evt;
    h->hdr.a_chunks = pb.a_chunks;
    h->hdr.in_chunks = round_up(S + Nz, 64) / 64;
    int max_n = 32;
    for (const TcLayer &l : pb.layers) max_n = std::max(max_n, (int)l.n_pad);
    int cols = 32;
    while (cols < max_n) cols *= 2;
    h->hdr.tmem_cols = cols;
    h->hdr.n_stages = 8;
#ifdef VOILA_TC_TRACE
    if (const char *e = getenv("VOILA_TC_STAGES")) h->hdr.n_stages = atoi(e);
#endif
    while (h->hdr.n_stages > 2 && smem_map(h->hdr).total + 1024 > kMaxDynSmem) --h->hdr.n_stages;
    h->smem_bytes = smem_map(h->hdr).total + 1024;
    if (h->smem_bytes > kMaxDynSmem) {
        if (err) *err = "model does not fit the shared-memory budget of the tcgen05 kernel";
        delete h;
        return nullptr;
    }
    auto upload = [&](const void *src, size_t bytes, void **dst) -> bool {
        if (cudaMalloc(dst, bytes) != cudaSuccess) return false;
        allocs->push_back(*dst);
        return cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess;
    };
    h->wstream_bytes = pb.wstream.size();
    if (!upload(pb.wstream.data(), pb.wstream.size(), &h->d_wstream) ||
        !upload(pb.bias.data(), pb.bias.size() * sizeof(float), &h->d_bias) ||
        !upload(pb.layers.data(), pb.layers.size() * sizeof(TcLayer), &h->d_layers) ||
        !upload(pb.tiles.data(), pb.tiles.size() * sizeof(TcTile), &h->d_tiles) ||
        cudaFuncSetAttribute(rollout_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)h->smem_bytes) != cudaSuccess) {
        if (err) *err = cudaGetErrorString(cudaGetLastError());
        delete h;
        return nullptr;
    }
    return h;
}

void tc_destroy(void *tc) { delete reinterpret_cast<TcHandle *>(tc); }
bool tc_has_belief(const void *) { return false; }

cudaError_t launch_rollout_tc(void *tc, const ModelDev &m, const RolloutArgs &a, cudaStream_t st,
                              std::string *kernel_name, int *n_launches) {
    const TcHandle *h = reinterpret_cast<const TcHandle *>(tc);
    TcRolloutParams p{};
    p.wstream = reinterpret_cast<const uint8_t *>(h->d_wstream);
    p.bias = reinterpret_cast<const float *>(h->d_bias);
    p.layers = reinterpret_cast<const TcLayer *>(h->d_layers);
    p.tiles = reinterpret_cast<const TcTile *>(h->d_tiles);
    p.hdr = h->hdr;
    p.particles = reinterpret_cast<const uint16_t *>(a.particles);
    p.seqs = a.action_seqs;
    p.weights = a.weights;
    p.P = a.P; p.Q = a.Q; p.H = a.H;
    p.seed = a.seed;
    p.part_value = a.part_value;
    p.part_witness = a.part_witness;
    p.returns_out = a.returns_out;
    p.final_states_out = a.final_states_out;
    p.tiles_per_q = a.tiles;
    p.n_units = a.tiles * a.Q;
    p.S = m.S; p.O = m.O; p.A = m.A; p.Nz = m.Nz;
    p.gamma = m.gamma;
    p.reward_kind = m.reward.kind;
    p.reward_param = m.reward.param;
    p.action_cost = m.reward.action_cost;
    const int grid = std::min(h->sm_count, p.n_units);
    rollout_tc_kernel<<<grid, kTcThreads, h->smem_bytes, st>>>(p);
    if (kernel_name) *kernel_name = "rollout_tc_kernel<tcgen05 bf16>";
    if (n_launches) *n_launches = 1;
    return cudaGetLastError();
}

cudaError_t launch_bu_propose_score_tc(void *, const ModelDev &, const BeliefArgs &, cudaStream_t, int *) {
    return cudaErrorNotSupported;
}

}  // namespace voila

#ifdef VOILA_TC_TRACE
extern "C" __attribute__((visibility("default"))) int voila_debug_tc_trace(unsigned long long *out32) {
    return (int)cudaMemcpyFromSymbol(out32, voila::g_tc_trace, sizeof(unsigned long long) * 32);
}
#endif
