// rollout_tc2.cu -- CTA-pair (cta_group::2) tcgen05 path of libvoila (bf16 mode): the persistent
// fused-MLP rollout kernel.  See tc2_program.h for the execution model.  A cluster of two CTAs
// (two SMs) is persistent over (sequence, 256-particle block) work units; per CTA:
//   warp 0    producer: TMA (cp.async.bulk.tensor, cta_group::2) streams this CTA's half of every
//             weight tile L2 -> shared-memory ring, completing bytes on the LEADER's mbarrier
//   warp 1    MMA issuer (leader CTA only): one thread issues tcgen05.mma.cta_group::2
//             (M = 256, N = bn, K = 16, bf16 -> fp32 in both CTAs' TMEM), multicast commits
//   warp 2    TMEM allocation
//   warps 4-11 epilogue: tcgen05.ld accumulator block -> bias + activation -> bf16 -> operand
//             buffer (in place), Philox noise, reward / return accumulation, observation witness
//   warps 12-19 (640-thread kernels: rollout_tc2x_kernel, belief_tc2_dual_kernel) a second set of
//             epilogue warps: the odd chunks of every hidden layer / the second unit in flight.
// The same machinery runs the belief update's propose+score program (belief_tc2*_kernel).
// The horizon loop never leaves the SMs: HBM sees the particle rows once per work unit and the
// per-unit partial sums; weights come from L2, half a tile per CTA.
#include <cuda.h>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <string>
#include <vector>

#include "tc2_program.h"
#include "tc_common.cuh"
#include "voila_kernels.h"

namespace voila {

namespace {

using namespace tcc;

// Optional wait-cycle trace (build with -DVOILA_T2_TRACE): where the producer, the MMA issuer and
// the epilogue warps of cluster 0 spend their time waiting.  Read with voila_debug_t2_trace().
#ifdef VOILA_T2_TRACE
__device__ unsigned long long g_t2_trace[64];
#define T2_TRACE_T0() const long long _t0 = clock64()
#define T2_TRACE_ADD(var) var += clock64() - _t0
// Timeline of the leader CTA of cluster 0 (one SM, so clock64 is one clock): (tag, cycle) pairs.
// tag = kind << 24 | layer-or-step << 8 | chunk-or-tile; kinds: 1 tile ready, 2 tile issued,
// 3 / 5 epilogue set 0 / 1 starts a chunk or layer (waits done), 4 / 6 it publishes the event.
constexpr unsigned kT2TlCap = 16384;
__device__ unsigned long long g_t2_tl[2 * kT2TlCap];
__device__ unsigned int g_t2_tl_n;
__device__ int g_t2_tl_win[2] = {40, 44};  // steps [win0, win1) are recorded
// every recording thread owns a region of the buffer and a private cursor: plain stores only
// (an atomic's round trip would stall the recorded thread for ~700 cycles per event)
__device__ __forceinline__ void t2_tl(bool on, uint32_t tag, uint32_t region, uint32_t &cursor) {
    if (on && cursor < kT2TlCap / 4) {
        const unsigned i = region * (kT2TlCap / 4) + cursor++;
        g_t2_tl[2 * i] = tag;
        g_t2_tl[2 * i + 1] = (unsigned long long)clock64();
    }
}
#define T2_TL(on, tag) t2_tl(on, tag, (es.tl_kind - 1u) >> 1, es.tl_n)
#define T2_TL_ISSUER(on, tag) t2_tl(on, tag, 0u, tl_n)
#else
#define T2_TRACE_T0()
#define T2_TRACE_ADD(var)
#define T2_TL(on, tag)
#define T2_TL_ISSUER(on, tag)
#endif

struct T2Params {
    const float *bias;        // global: all bias rows (SiLU hidden layers pre-halved)
    const float *sbias_init;  // image of the shared-memory bias table (action rows left empty)
    const T2Layer *layers;
    const T2TileDev *tiles;
    T2Header hdr;
    const uint16_t *particles;  // [P][S] bf16
    const int32_t *seqs;        // [Q][H]
    const float *weights;       // [P] or nullptr
    int P, Q, H;
    uint64_t seed;
    double *part_value;    // [Q][tiles_per_q]
    double *part_witness;  // [Q][tiles_per_q][O] or nullptr
    float *returns_out;
    float *final_states_out;
    int tiles_per_q, blocks_per_q, n_units;
    int S, O, A, Nz;  // S, Nz: as the operand sees them (padded to multiples of 8); O, A: public
    int S_io;         // public state width: rows of particles / proposals / final states
    float gamma;
    int reward_kind;
    const float *reward_param;
    const float *action_cost;
    TerminalDev term;  // terminal regions of the rollout (voila_terminal)
    // belief-update program (propose + score): one unit = 256 particles, one step per unit
    int bu_action;
    const float *bu_e;        // f(o), [d]
    uint16_t *bu_proposals;   // [N][S] bf16
    float *bu_logits;         // [N]
    int *bu_max_ordered;      // [1]
    double *bu_part_wsum;     // [(N + 31) / 32]: prior-weight sums per 32 particles
    float inv_lambda;
    int d;
    // progressive widening (voila_pw_update): every row has its own action (one-hot block in the
    // operand), its own tower embedding e and the running maximum of its own child belief
    const int32_t *pw_sim_action;  // [N] or nullptr (plain belief update)
    const int32_t *pw_sim_seg;     // [N] child index g * M_max + b
    const float *pw_E;             // [children][d]
    int *pw_seg_max;               // [children] ordered-int maxima
    // diffusion teacher (voila_diffusion_sample): one DDIM-ODE step per launch; the operand is
    // [c ; x ; onehot(a)], the time embedding sits in the step's bias row (bu_action = step index)
    float *diff_x;                 // [N][D] fp32 state, updated in place, or nullptr
    int diff_D, diff_first;        // first: x = omega (Philox stream 7) instead of the stored state
    float al, si, al_n, si_n;      // alpha, sigma at tau_k and tau_{k+1}
    // progressive widening, the small passes over the (action node, branch) slots (row = slot g * M_max + m):
    // MODE 3: slots opened in this call: s' = f_T(s_src, a_g, w_T(src)), o = f_Z(s', a_g, w_Z(src)) -> branch_obs
    // MODE 4: every stored branch (m < branch_count[g]): e = f(obs) -> embedding table
    const int32_t *slot_src;       // [slots] simulation that opened the slot, or -1
    const int32_t *slot_action;    // [G] action of the node
    const int32_t *slot_count;     // [G] branches stored per node (MODE 4)
    float *slot_obs;               // [slots][O] fp32
    float *slot_emb;               // [slots][d] fp32
    int slot_M;                    // M_max
};

struct Smem2 {
    uint32_t a, ring, layers, tiles, bars, misc, sbias, total;
};
constexpr uint32_t kT2SlotMisc = 4 * 8 + 4 * 64 * 4 + 256;  // red_g[4] doubles, red_w[4][64] floats, alive[2][128] bytes
__host__ __device__ inline Smem2 smem2_map(const T2Header &h) {
    Smem2 m;
    m.a = 0;
    m.ring = m.a + (uint32_t)h.a_chunks * kT2ChunkBytes;
    m.layers = m.ring + (uint32_t)h.n_stages * (uint32_t)h.stage_rows * 128u;
    m.tiles = m.layers + kT2MaxLayers * (uint32_t)sizeof(T2Layer);
    m.bars = m.tiles + (((uint32_t)h.n_tiles * (uint32_t)sizeof(T2TileDev) + 15u) & ~15u);
    m.misc = m.bars + (8 + 8 + kT2EvtRing + kT2AccRing + kT2FreeRing) * 8;
    m.sbias = m.misc + 16 + 2 * kT2SlotMisc;  // per slot: reduction scratch + per-row alive flags (two step parities)
    m.total = m.sbias + (((uint32_t)h.sbias_floats * 4u + 15u) & ~15u);
    return m;
}

// act(v + b) of a hidden layer.  SiLU layers carry PRE-HALVED biases: with h = (v + b) / 2,
// x * sigmoid(x) = h + h * tanh(h): one FFMA, one MUFU.TANH, one FFMA per element.
template <int ACT>
__device__ __forceinline__ float act_biased(uint32_t v, float b) {
    if (ACT == VOILA_ACT_SILU) {
        const float h = fmaf(__uint_as_float(v), 0.5f, b);
        return fmaf(h, tanh_approx(h), h);
    }
    const float x = __uint_as_float(v) + b;
    return ACT == VOILA_ACT_RELU ? fmaxf(x, 0.0f) : x;
}

// Per-thread constants of the hidden-layer epilogue, computed once and pinned in registers (the
// asm barrier keeps the compiler from re-deriving them from %tid / cvta in every chunk, which was
// ~40 % of the chunk's instructions).
struct EpiConst {
    uint32_t st_base;   // shared address of this row in operand chunk 0
    uint32_t sw[4];     // swizzled byte offsets of this warp's four 16-byte units inside a row
    uint32_t taddr0;    // TMEM address of this warp's lane quadrant + column half
    uint32_t sbias_u32; // shared address of the bias table + this warp's column half
};
__device__ __forceinline__ uint32_t pin_reg(uint32_t v) {
    asm volatile("mov.b32 %0, %0;" : "+r"(v));
    return v;
}
__device__ __forceinline__ EpiConst make_epi_const(uint32_t a_u32, uint32_t lane_taddr, const float *sbias, int row,
                                                   int half) {
    EpiConst c;
    c.st_base = pin_reg(a_u32 + (uint32_t)row * 128u);
#pragma unroll
    for (int u = 0; u < 4; ++u) c.sw[u] = (uint32_t)(((half * 4 + u) ^ (row & 7)) << 4);
    c.taddr0 = pin_reg(lane_taddr + (uint32_t)(32 * half));
    c.sbias_u32 = pin_reg(smem_u32(sbias) + (uint32_t)(32 * half) * 4u);
    return c;
}
__device__ __forceinline__ float4 ld_shared_f4(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// 16 accumulator columns of this thread's row (already in registers) -> bias (shared memory,
// broadcast reads) -> activation -> bf16 -> two 16-byte units of the 64-column operand chunk.
template <int ACT>
__device__ __forceinline__ void hidden_store16(const uint32_t (&v)[16], uint32_t bias_u32, uint32_t row_addr,
                                               uint32_t sw0, uint32_t sw1) {
    // (loading the 16 biases ahead of the TMEM wait was tried: more live registers, spills in the
    // 16-warp rollout kernel, CFG5 1140 -> 1073 TFLOP/s)
    uint32_t o[8];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float4 b = ld_shared_f4(bias_u32 + 16u * i);
        o[2 * i] = pack_bf16x2(act_biased<ACT>(v[4 * i], b.x), act_biased<ACT>(v[4 * i + 1], b.y));
        o[2 * i + 1] = pack_bf16x2(act_biased<ACT>(v[4 * i + 2], b.z), act_biased<ACT>(v[4 * i + 3], b.w));
    }
    st_shared_v4(row_addr + sw0, o[0], o[1], o[2], o[3]);
    st_shared_v4(row_addr + sw1, o[4], o[5], o[6], o[7]);
}

// Synchronisation state of one epilogue warp: the numbered events it publishes on the leader's
// mbarriers, and its positions in the accumulator hand-off and operand-chunk-free rings.
struct EpiSync {
    uint32_t evt_cl;       // cluster address of the leader's event ring
    uint64_t *layer_done;  // accumulator hand-off ring (this CTA's copy; multicast commits)
    uint64_t *cfree;       // operand-chunk-free ring
    int ev = 0;
    uint32_t ld_seq = 0, free_seq = 0;
    int lane;
    long long tr_layer = 0, tr_free = 0, tr_bar = 0;  // wait-cycle trace (VOILA_T2_TRACE)
    bool tl_on = false;     // timeline trace: this warp records the current step
    uint32_t tl_kind = 3u;  // 3: first epilogue set, 5: second set
    uint32_t tl_layer = 0, tl_n = 0;

    __device__ __forceinline__ void arrive_event() {
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(evt_cl + 8u * (uint32_t)(ev & (kT2EvtRing - 1)));
        ++ev;
    }
    __device__ __forceinline__ void wait_layer() {
        T2_TRACE_T0();
        mbar_wait(&layer_done[ld_seq & (kT2AccRing - 1)], (ld_seq >> 3) & 1u);
        T2_TRACE_ADD(tr_layer);
        ++ld_seq;
        tc_fence_after();
    }
    __device__ __forceinline__ void wait_chunk_free() {
        T2_TRACE_T0();
        mbar_wait(&cfree[free_seq & (kT2FreeRing - 1)], (free_seq >> 3) & 1u);
        T2_TRACE_ADD(tr_free);
        ++free_seq;
    }
};

// Epilogue of a hidden layer for this warp's 32 rows x one 32-column half of every 64-column chunk:
// software-pipelined over the chunks (the TMEM load of chunk j+1 is in flight while chunk j goes
// through bias / activation / pack / store / event).  One instantiation per activation, so the
// chunk loop carries no dispatch.
template <int ACT>
__device__ __forceinline__ void epi_hidden_loop(EpiSync &es, const T2Layer &l, uint32_t bias_u32, const EpiConst &ec) {
    // 16-column pieces, double-buffered: the TMEM load of piece k+1 is in flight while piece k goes
    // through bias / activation / pack / store (32 live accumulator registers instead of 64)
    uint32_t va[16], vb[16];
    const int chunks = l.n_pad >> 6;
    const int wait_chunks = l.wait_chunks;
    const int free_sh = 31 - __clz((int)l.free_nk);  // free_nk is 1, 2 or 4: a shift, not a division, per chunk
    const uint32_t blk_mask = l.blk_mask;
    const bool one_event = l.one_event != 0;  // one event for the whole layer (T2Layer::one_event)
    int free_have = 0;
    // accumulator blocks are handed over one by one: a chunk may be loaded once the block it
    // belongs to has been committed (blk_mask: chunks that start a block)
    if (blk_mask & 1u) es.wait_layer();
    tmem_ld16(ec.taddr0, va);
    for (int j = 0; j < chunks; ++j) {
        const uint32_t row_addr = ec.st_base + (uint32_t)j * kT2ChunkBytes;
        const uint32_t bj = bias_u32 + 256u * (uint32_t)j;
        tmem_ld_wait();
        tmem_ld16(ec.taddr0 + (uint32_t)(64 * j + 16), vb);
        if (j < wait_chunks) {  // in-place store: the last block must have read chunk j
            const int need_free = (j >> free_sh) + 1;
            while (free_have < need_free) {
                es.wait_chunk_free();
                ++free_have;
            }
            tc_fence_after();
        }
        T2_TL(es.tl_on, (es.tl_kind << 24) | (es.tl_layer << 8) | (uint32_t)j);
        hidden_store16<ACT>(va, bj, row_addr, ec.sw[0], ec.sw[1]);
        tmem_ld_wait();
        // the next chunk may belong to a block that is still being accumulated: then publish this
        // chunk first and wait afterwards (one un-overlapped TMEM load per block, not per chunk)
        const bool next_blk = (j + 1 < chunks) && ((blk_mask >> (j + 1)) & 1u);
        if (j + 1 < chunks && !next_blk) tmem_ld16(ec.taddr0 + (uint32_t)(64 * (j + 1)), va);
        hidden_store16<ACT>(vb, bj + 64u, row_addr, ec.sw[2], ec.sw[3]);
        if (!one_event || j + 1 == chunks) {
            fence_proxy_async_smem();
            tc_fence_before();
            es.arrive_event();
        }
        T2_TL(es.tl_on, ((es.tl_kind + 1u) << 24) | (es.tl_layer << 8) | (uint32_t)j);
        if (next_blk) {
            es.wait_layer();
            tmem_ld16(ec.taddr0 + (uint32_t)(64 * (j + 1)), va);
        }
    }
}
// The same for a layer that is ONE accumulator block (every hidden layer of a two-slot program, narrow
// layers elsewhere): no block hand-offs inside the layer and no in-place chunk-free waits, so the chunk
// loop carries no bookkeeping at all (the general loop spends more instructions on control than on math).
template <int ACT>
__device__ __forceinline__ void epi_hidden_loop_1blk(EpiSync &es, const T2Layer &l, uint32_t bias_u32, const EpiConst &ec) {
    uint32_t va[16], vb[16];
    const int chunks = l.n_pad >> 6;
    const bool one_event = l.one_event != 0;
    es.wait_layer();
    tmem_ld16(ec.taddr0, va);
    uint32_t row_addr = ec.st_base, bj = bias_u32, ta = ec.taddr0;
#pragma unroll 1
    for (int j = chunks; j > 0; --j) {
        tmem_ld_wait();
        tmem_ld16(ta + 16u, vb);
        T2_TL(es.tl_on, (es.tl_kind << 24) | (es.tl_layer << 8) | (uint32_t)(chunks - j));
        hidden_store16<ACT>(va, bj, row_addr, ec.sw[0], ec.sw[1]);
        tmem_ld_wait();
        ta += 64u;
        if (j > 1) tmem_ld16(ta, va);
        hidden_store16<ACT>(vb, bj + 64u, row_addr, ec.sw[2], ec.sw[3]);
        if (!one_event || j == 1) {
            fence_proxy_async_smem();
            tc_fence_before();
            es.arrive_event();
        }
        T2_TL(es.tl_on, ((es.tl_kind + 1u) << 24) | (es.tl_layer << 8) | (uint32_t)(chunks - j));
        row_addr += kT2ChunkBytes;
        bj += 256u;
    }
}
__device__ __forceinline__ void epi_hidden_layer(EpiSync &es, const T2Layer &l, int bias_float_off, const EpiConst &ec) {
    const uint32_t bias_u32 = ec.sbias_u32 + 4u * (uint32_t)bias_float_off;
    if (l.blk_mask == 1u && l.wait_chunks == 0) {
        if (l.act == VOILA_ACT_SILU) epi_hidden_loop_1blk<VOILA_ACT_SILU>(es, l, bias_u32, ec);
        else if (l.act == VOILA_ACT_RELU) epi_hidden_loop_1blk<VOILA_ACT_RELU>(es, l, bias_u32, ec);
        else epi_hidden_loop_1blk<VOILA_ACT_NONE>(es, l, bias_u32, ec);
        return;
    }
    if (l.act == VOILA_ACT_SILU) epi_hidden_loop<VOILA_ACT_SILU>(es, l, bias_u32, ec);
    else if (l.act == VOILA_ACT_RELU) epi_hidden_loop<VOILA_ACT_RELU>(es, l, bias_u32, ec);
    else epi_hidden_loop<VOILA_ACT_NONE>(es, l, bias_u32, ec);
}

// The same layer shared by TWO sets of epilogue warps (640-thread rollout kernel): a set handles the
// chunks j with (j & 1) == parity and keeps the books for the others (event numbers advance without
// an arrive; accumulator-block and chunk-free sequence numbers are brought up to date at the end).
// Every chunk's event still collects 16 arrivals: 8 warps of ONE set in each CTA.
template <int ACT>
__device__ __forceinline__ void epi_hidden_loop_par(EpiSync &es, const T2Layer &l, uint32_t bias_u32, const EpiConst &ec,
                                                    int parity) {
    uint32_t va[16], vb[16];
    const int chunks = l.n_pad >> 6;
    const int wait_chunks = l.wait_chunks;
    const int free_sh = 31 - __clz((int)l.free_nk);  // free_nk is 1, 2 or 4 (K chunks per ring stage)
    const uint32_t blk_mask = l.blk_mask;
    const int n_blocks = __popc(blk_mask);
    const int n_sig = wait_chunks > 0 ? ((wait_chunks - 1) >> free_sh) + 1 : 0;
    int free_have = 0, blocks_waited = 0;
    // this set's chunks: parity, parity + 2, ... (prefetching the next chunk's first columns across the
    // event was tried: spills in the 56-register helper warps)
    es.ev += parity;
    for (int j = parity; j < chunks; j += 2) {
        // blocks that start at a chunk <= j must have been handed over
        const int need_blocks = __popc(blk_mask & ((2u << j) - 1u));
        while (blocks_waited < need_blocks) {
            es.wait_layer();
            ++blocks_waited;
        }
        const uint32_t row_addr = ec.st_base + (uint32_t)j * kT2ChunkBytes;
        const uint32_t bj = bias_u32 + 256u * (uint32_t)j;
        tmem_ld16(ec.taddr0 + (uint32_t)(64 * j), va);
        tmem_ld_wait();
        tmem_ld16(ec.taddr0 + (uint32_t)(64 * j + 16), vb);
        if (j < wait_chunks) {  // in-place store: the last block must have read chunk j
            const int need_free = (j >> free_sh) + 1;
            while (free_have < need_free) {
                es.wait_chunk_free();
                ++free_have;
            }
            tc_fence_after();
        }
        T2_TL(es.tl_on, (es.tl_kind << 24) | (es.tl_layer << 8) | (uint32_t)j);
        hidden_store16<ACT>(va, bj, row_addr, ec.sw[0], ec.sw[1]);
        tmem_ld_wait();
        hidden_store16<ACT>(vb, bj + 64u, row_addr, ec.sw[2], ec.sw[3]);
        fence_proxy_async_smem();
        tc_fence_before();
        es.arrive_event();
        T2_TL(es.tl_on, ((es.tl_kind + 1u) << 24) | (es.tl_layer << 8) | (uint32_t)j);
        ++es.ev;  // the other set's chunk j + 1 (or j - 1: the count per layer is what matters)
    }
    // (an odd number of chunks: the set without the last chunk has counted one event too many / too few)
    es.ev += chunks - ((chunks - parity + 1) >> 1) * 2 - parity;
    es.ld_seq += (uint32_t)(n_blocks - blocks_waited);
    es.free_seq += (uint32_t)(n_sig - free_have);
}
__device__ __forceinline__ void epi_hidden_layer_par(EpiSync &es, const T2Layer &l, int bias_float_off,
                                                     const EpiConst &ec, int parity) {
    const uint32_t bias_u32 = ec.sbias_u32 + 4u * (uint32_t)bias_float_off;
    if (l.act == VOILA_ACT_SILU) epi_hidden_loop_par<VOILA_ACT_SILU>(es, l, bias_u32, ec, parity);
    else if (l.act == VOILA_ACT_RELU) epi_hidden_loop_par<VOILA_ACT_RELU>(es, l, bias_u32, ec, parity);
    else epi_hidden_loop_par<VOILA_ACT_NONE>(es, l, bias_u32, ec, parity);
}

// Second set of epilogue warps of the 640-thread rollout kernel (warps 12-19): the odd chunks of
// every hidden layer, nothing else (no per-row state: 72 registers).
__device__ __forceinline__ void t2_helper_epilogue(const T2Params &p, const T2Layer *L, uint32_t a_u32, uint32_t tmem_base,
                                                   uint64_t *evt, uint64_t *layer_done, float *sbias, int warp, int lane,
                                                   int total_steps) {
    const int n_layers = p.hdr.n_layers;
    const int ew = (warp - 4) & 7, qd = warp & 3, half = ew >> 2;
    const int row = qd * 32 + lane;
    const uint32_t lane_taddr = tmem_base + ((uint32_t)(qd * 32) << 16);
    EpiSync es;
    es.evt_cl = mapa_u32(smem_u32(evt), 0u);
    es.layer_done = layer_done;
    es.cfree = layer_done + kT2AccRing;
    es.lane = lane;
    const EpiConst ec = make_epi_const(a_u32, lane_taddr, sbias, row, half);
    es.ev = 1;  // the first set publishes the initial-input event
    es.tl_kind = 5u;
    for (int step = 0; step < total_steps; ++step) {
#ifdef VOILA_T2_TRACE
        es.tl_on = blockIdx.x == 0 && warp == 12 && lane == 0 && step >= g_t2_tl_win[0] && step < g_t2_tl_win[1];
#endif
        for (int li = 0; li < n_layers; ++li) {
            const T2Layer l = L[li];
            es.tl_layer = (uint32_t)li;
            if (l.epi == T2_EPI_HIDDEN) {
                EpiConst ecs = ec;
                ecs.taddr0 += (uint32_t)l.col_off;  // accumulators ping-pong between the TMEM halves (narrow models)
                epi_hidden_layer_par(es, l, (int)l.sbias_off + (l.bias_per_action ? (step & 1) * (int)l.n_pad : 0), ecs, 1);
            } else {
                ++es.ev;
                ++es.ld_seq;
            }
        }
    }
}

// Epilogue role (warps 4-11 of BOTH CTAs): each warp owns 32 rows (TMEM lane quadrant warp % 4) and,
// in hidden layers, one 32-column half of every 64-column chunk.  Events are published on the
// LEADER's mbarriers (remote arrive from the peer CTA).
// MODE: 1 = the model has terminal regions (voila_terminal); 0 compiles the alive-flag logic out (it cost
// the plain rollout 2.4 % when it was a runtime test).
template <int MODE>
__device__ __forceinline__ void t2_epilogue(const T2Params &p, const T2Layer *L, uint32_t a_u32, uint32_t tmem_base,
                                            uint64_t *evt, uint64_t *layer_done, double *red_g, float *red_w,
                                            uint8_t *alive_s, float *sbias, int warp, int lane, uint32_t rank,
                                            int cluster_id, int n_clusters, int n_my_units, int total_steps,
                                            bool shared_hidden, int my_slot) {
    // shared_hidden: a second set of epilogue warps takes the odd chunks of the hidden layers
    // my_slot < 0: one unit in flight.  my_slot = 0 | 1: TWO-SLOT program (hdr.n_slots == 2, models
    // whose layers are all <= 256 wide): this set of eight warps owns the rows of one slot (own operand
    // chunks, TMEM columns, reduction scratch, named barrier) and only keeps the books (event,
    // accumulator-block and chunk-free sequence numbers) for the other slot's layer records, so one
    // unit's epilogue overlaps the other unit's MMAs.  Both slots of a work unit belong to the same
    // sequence q (two adjacent 256-particle blocks): they share the action-dependent bias rows.
    const int n_layers = p.hdr.n_layers;
    const uint32_t evt_cl = mapa_u32(smem_u32(evt), 0u);
    const int n_slots = my_slot < 0 ? 1 : 2, slot_i = my_slot > 0 ? 1 : 0;
    const uint32_t bar_id = 1u + (uint32_t)slot_i;
    a_u32 += (uint32_t)(slot_i * p.hdr.slot_chunks) * kT2ChunkBytes;
    red_g += 4 * slot_i;
    red_w += 4 * 64 * slot_i;
    alive_s += 2 * kT2Rows * slot_i;
    {
        // ===== epilogue warps =====
        const int ew = (warp - 4) & 7, qd = warp & 3, half = ew >> 2;
        const int row = qd * 32 + lane;
        const uint32_t lane_taddr = tmem_base + ((uint32_t)(qd * 32) << 16);
        const int S = p.S, O = p.O, Nz = p.Nz;
        const int in_units = p.hdr.in_chunks * 8;  // 8-column units of the step's input operand
        uint32_t persist[64];  // half 0: packed bf16 state (32 words); half 1: fp32 witness (64 words)
        uint32_t nz[16];
        float G = 0.0f, disc = 1.0f, w_row = 0.0f;
        int t = 0, unit_i = 0, q = 0, blk = 0, p_idx = 0;
        bool valid = false;
        bool alive = true;  // the row's episode still runs (terminal regions, reading R25)
        const long long tr_start = clock64();
        EpiSync es;
        es.tl_kind = my_slot > 0 ? 5u : 3u;
        es.evt_cl = evt_cl;
        es.layer_done = layer_done;
        es.cfree = layer_done + kT2AccRing;
        es.lane = lane;
        auto arrive_event = [&]() { es.arrive_event(); };
        auto wait_layer = [&]() { es.wait_layer(); };
        const EpiConst ec = make_epi_const(a_u32, lane_taddr, sbias, row, half);
        auto load_unit = [&]() {
            const int unit = cluster_id + unit_i * n_clusters;
            q = unit / p.blocks_per_q;
            blk = ((unit - q * p.blocks_per_q) * n_slots + slot_i) * 2 + (int)rank;  // 128-row tile index within the sequence
            p_idx = blk * kT2Rows + row;
            valid = p_idx < p.P;
            w_row = valid ? (p.weights ? __ldg(p.weights + p_idx) : 1.0f) : 0.0f;
            G = 0.0f;
            disc = 1.0f;
            t = 0;
            alive = true;
            if (half == 0) {
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    uint4 v = make_uint4(0u, 0u, 0u, 0u);
                    if (8 * u < S && valid) v = load_row_unit(p.particles + (size_t)p_idx * p.S_io, p.S_io, u);
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
        // Pays step t's reward r_step = R(s_t, a_t) (half 0 warps, which hold the state).  Terminal
        // regions (voila_terminal, reading R25): every region holding s_t pays its reward; a stopping
        // one ends the episode here (r_step is not paid, the state freezes, nothing accrues later).
        // The row's alive flag of step t goes to shared memory for the warp that holds its witness.
        auto pay = [&](float r_step) {
            if (MODE == 0) {
                G = fmaf(disc, r_step, G);
                return;
            }
            float bonus = 0.0f;
            bool stop = false;
            for (int k = 0; k < p.term.n; ++k) {
                const float *c = p.term.centers + p.term.off[k];
                const int dim = p.term.dim[k];
                float d2 = 0.0f;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    if (j < dim) {
                        const float sj = (j & 1) ? bf16hi(persist[j >> 1]) : bf16lo(persist[j >> 1]);
                        const float d = sj - __ldg(c + j);
                        d2 = fmaf(d, d, d2);
                    }
                }
                if (d2 <= p.term.r2[k]) {
                    bonus += p.term.reward[k];
                    stop |= p.term.stop[k] != 0;
                }
            }
            if (alive) {
                G = fmaf(disc, stop ? bonus : bonus + r_step, G);
                if (stop) alive = false;
            }
            alive_s[(t & 1) * kT2Rows + row] = alive ? 1 : 0;
        };
        auto step_reward = [&]() {  // non-quadratic reward kinds: R(s_t, a_t) from the state words
            if (half == 0 && p.reward_kind != VOILA_R_NEG_QUADRATIC) {
                float r = reward_from_state(persist, p.S_io, p.reward_kind, p.reward_param);
                if (p.action_cost) r += __ldg(p.action_cost + clamp_action(__ldg(p.seqs + (size_t)q * p.H + t), p.A));
                pay(r);
            }
        };

        // Bias rows that depend on the action (one-hot block folded into the bias, R21):
        // the rows of the NEXT step are fetched mid-step into registers and parked in the other
        // half of a two-row slot of the shared-memory bias table at the end of the step.
        const int tid_e = ((int)threadIdx.x - 128) & 255;  // (two-slot: both sets park the same rows)
        float4 pa_reg[2] = {make_float4(0.f, 0.f, 0.f, 0.f), make_float4(0.f, 0.f, 0.f, 0.f)};
        auto refresh_issue = [&](int q_next, int t_next) {
            const int a_next = clamp_action(__ldg(p.seqs + (size_t)q_next * p.H + t_next), p.A);
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int li = p.hdr.pa_layer[i];
                if (li >= 0 && 4 * tid_e < (int)L[li].n_pad)
                    pa_reg[i] = __ldg(reinterpret_cast<const float4 *>(p.bias + L[li].bias_off +
                                                                         (size_t)a_next * L[li].n_pad) + tid_e);
            }
        };
        auto refresh_store = [&](int parity) {
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int li = p.hdr.pa_layer[i];
                if (li >= 0 && 4 * tid_e < (int)L[li].n_pad)
                    *reinterpret_cast<float4 *>(sbias + L[li].sbias_off + parity * (int)L[li].n_pad + 4 * tid_e) =
                        pa_reg[i];
            }
        };

        if (n_my_units > 0) {
            if (slot_i == 1) ++es.ev;  // slot 0's initial event (hdr.init_events = one per slot)
            load_unit();
            refresh_issue(q, 0);
            if (half == 0) gen_noise_call(nz, p.seed, (uint32_t)p_idx, (uint32_t)q, 0u, kStreamRolloutT, Nz);
            write_input(0, 0);
            step_reward();
            refresh_store(0);
            named_bar_sync(bar_id, 256);
            fence_proxy_async_smem();
            arrive_event();
            if (my_slot == 0) ++es.ev;  // slot 1's initial event
        }
        for (int step = 0; step < total_steps; ++step) {
            const int a_t = clamp_action(__ldg(p.seqs + (size_t)q * p.H + t), p.A);
#ifdef VOILA_T2_TRACE
            es.tl_on = blockIdx.x == 0 && ew == 0 && lane == 0 && step >= g_t2_tl_win[0] && step < g_t2_tl_win[1];
#endif
            for (int li = 0; li < n_layers; ++li) {
                const T2Layer l = L[li];
                es.tl_layer = (uint32_t)li;
                if (my_slot >= 0 && (int)l.slot != my_slot) {  // the other set's record: sequence numbers only
                    const bool hid = l.epi == T2_EPI_HIDDEN;
                    es.ev += (hid && !l.one_event) ? (int)(l.n_pad >> 6) : 1;
                    es.ld_seq += hid ? (uint32_t)__popc((unsigned)l.blk_mask) : 1u;
                    if (hid && l.wait_chunks > 0) es.free_seq += ((uint32_t)l.wait_chunks + l.free_nk - 1u) / l.free_nk;
                    continue;
                }
                const float *bias = sbias + l.sbias_off + (l.bias_per_action ? (step & 1) * (int)l.n_pad : 0);
                if (l.epi == T2_EPI_HIDDEN) {
                    const int boff = (int)l.sbias_off + (l.bias_per_action ? (step & 1) * (int)l.n_pad : 0);
                    EpiConst ecs = ec;
                    ecs.taddr0 += (uint32_t)l.col_off;  // accumulators ping-pong between the TMEM halves (narrow models)
                    if (shared_hidden) epi_hidden_layer_par(es, l, boff, ecs, 0);
                    else epi_hidden_layer(es, l, boff, ecs);
                } else if (l.epi == T2_EPI_REWARD) {
                    wait_layer();
                    T2_TL(es.tl_on, (es.tl_kind << 24) | (es.tl_layer << 8) | 0xffu);
                    if (half == 0) {
                        float r = 0.0f;
#pragma unroll
                        for (int g = 0; g < 4; ++g) {
                            if (16 * g < (int)l.n_pad) {
                                uint32_t v[16];
                                tmem_ld16(lane_taddr + (uint32_t)l.col_off + 16 * g, v);
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
                        pay(r);
                    }
                    tc_fence_before();
                    arrive_event();
                    T2_TL(es.tl_on, ((es.tl_kind + 1u) << 24) | (es.tl_layer << 8) | 0xffu);
                } else if (l.epi == T2_EPI_STATE) {
                    // w_Z(t) is independent of the state: draw it while the output layer's MMAs run
                    if (half == 1) gen_noise_call(nz, p.seed, (uint32_t)p_idx, (uint32_t)q, (uint32_t)t, kStreamRolloutZ, Nz);
                    if (t + 1 < p.H) refresh_issue(q, t + 1);
                    else if (unit_i + 1 < n_my_units)
                        refresh_issue((cluster_id + (unit_i + 1) * n_clusters) / p.blocks_per_q, 0);
                    wait_layer();
                    T2_TL(es.tl_on, (es.tl_kind << 24) | (es.tl_layer << 8) | 0xffu);
                    if (half == 0) {
#pragma unroll
                        for (int g = 0; g < 4; ++g) {
                            if (16 * g < (int)l.n_pad) {
                                uint32_t v[16];
                                tmem_ld16(lane_taddr + (uint32_t)l.col_off + 16 * g, v);
                                float4 b[4];
#pragma unroll
                                for (int i = 0; i < 4; ++i) b[i] = *(reinterpret_cast<const float4 *>(bias + 16 * g) + i);
                                tmem_ld_wait();
#pragma unroll
                                for (int i = 0; i < 4; ++i) {
                                    const uint32_t n0 = pack_bf16x2(__uint_as_float(v[4 * i]) + b[i].x,
                                                                    __uint_as_float(v[4 * i + 1]) + b[i].y);
                                    const uint32_t n1 = pack_bf16x2(__uint_as_float(v[4 * i + 2]) + b[i].z,
                                                                    __uint_as_float(v[4 * i + 3]) + b[i].w);
                                    // a row whose episode has ended keeps its state
                                    persist[8 * g + 2 * i] = (MODE == 0 || alive) ? n0 : persist[8 * g + 2 * i];
                                    persist[8 * g + 2 * i + 1] = (MODE == 0 || alive) ? n1 : persist[8 * g + 2 * i + 1];
                                }
                            }
                        }
                    }
                    write_input(0, 1);
                    fence_proxy_async_smem();
                    tc_fence_before();
                    arrive_event();
                    T2_TL(es.tl_on, ((es.tl_kind + 1u) << 24) | (es.tl_layer << 8) | 0xffu);
                } else {  // T2_EPI_OBS: last layer of the step
                    const bool last_step = (t == p.H - 1);
                    if (half == 0 && !last_step)
                        gen_noise_call(nz, p.seed, (uint32_t)p_idx, (uint32_t)q, (uint32_t)(t + 1), kStreamRolloutT, Nz);
                    wait_layer();
                    T2_TL(es.tl_on, (es.tl_kind << 24) | (es.tl_layer << 8) | 0xffu);
                    if (half == 1) {
                        // no observation for a row whose episode ended at or before step t
                        const float disc_w = (MODE == 0 || alive_s[(t & 1) * kT2Rows + row] != 0) ? disc : 0.0f;
#pragma unroll
                        for (int g = 0; g < 4; ++g) {
                            if (16 * g < (int)l.n_pad) {
                                uint32_t v[16];
                                tmem_ld16(lane_taddr + (uint32_t)l.col_off + 16 * g, v);
                                float4 b[4];
#pragma unroll
                                for (int i = 0; i < 4; ++i) b[i] = *(reinterpret_cast<const float4 *>(bias + 16 * g) + i);
                                tmem_ld_wait();
#pragma unroll
                                for (int i = 0; i < 4; ++i) {
                                    const float o0 = __uint_as_float(v[4 * i]) + b[i].x, o1 = __uint_as_float(v[4 * i + 1]) + b[i].y;
                                    const float o2 = __uint_as_float(v[4 * i + 2]) + b[i].z, o3 = __uint_as_float(v[4 * i + 3]) + b[i].w;
                                    const int c0 = 16 * g + 4 * i;
                                    persist[c0] = __float_as_uint(fmaf(disc_w, o0, __uint_as_float(persist[c0])));
                                    persist[c0 + 1] = __float_as_uint(fmaf(disc_w, o1, __uint_as_float(persist[c0 + 1])));
                                    persist[c0 + 2] = __float_as_uint(fmaf(disc_w, o2, __uint_as_float(persist[c0 + 2])));
                                    persist[c0 + 3] = __float_as_uint(fmaf(disc_w, o3, __uint_as_float(persist[c0 + 3])));
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
                                float *fs = p.final_states_out + ((size_t)q * p.P + p_idx) * p.S_io;
#pragma unroll
                                for (int c2 = 0; c2 < 32; ++c2)
                                    if (2 * c2 < p.S_io) {
                                        fs[2 * c2] = bf16lo(persist[c2]);
                                        if (2 * c2 + 1 < p.S_io) fs[2 * c2 + 1] = bf16hi(persist[c2]);
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
                        named_bar_sync(bar_id, 256);
                        // (two-slot: the second slot of a sequence's last pair may lie past the last tile)
                        if (ew == 0 && lane == 0 && blk < p.tiles_per_q)
                            p.part_value[(size_t)q * p.tiles_per_q + blk] = (red_g[0] + red_g[1]) + (red_g[2] + red_g[3]);
                        if (ew == 4 && p.part_witness && blk < p.tiles_per_q) {
                            for (int c = lane; c < O; c += 32)
                                p.part_witness[((size_t)q * p.tiles_per_q + blk) * O + c] =
                                    ((double)red_w[c] + (double)red_w[64 + c]) +
                                    ((double)red_w[128 + c] + (double)red_w[192 + c]);
                        }
                        named_bar_sync(bar_id, 256);
                        ++unit_i;
                        if (unit_i < n_my_units) {
                            load_unit();
                            if (half == 0) gen_noise_call(nz, p.seed, (uint32_t)p_idx, (uint32_t)q, 0u, kStreamRolloutT, Nz);
                        }
                    }
                    if (unit_i < n_my_units) {
                        write_input(0, 0);
                        step_reward();
                    }
                    refresh_store((step + 1) & 1);
                    {
                        T2_TRACE_T0();
                        named_bar_sync(bar_id, 256);
                        T2_TRACE_ADD(es.tr_bar);
                    }
                    fence_proxy_async_smem();
                    tc_fence_before();
                    arrive_event();
                    T2_TL(es.tl_on, ((es.tl_kind + 1u) << 24) | (es.tl_layer << 8) | 0xffu);
                }
            }
        }
#ifdef VOILA_T2_TRACE
        if (cluster_id == 0 && lane == 0) {
            unsigned long long *o = g_t2_trace + 16 + ((int)rank * 8 + ew) * 3;
            o[0] = es.tr_layer;
            o[1] = es.tr_free;
            o[2] = es.tr_bar;
            if (ew == 0 && rank == 0) g_t2_trace[15] = clock64() - tr_start;
        }
#endif
        (void)tr_start;
    }
}

// Epilogue role of the belief-update program: per 256-particle unit
//   input [s_i ; w_i] -> f_T hidden layers -> PROPOSAL: s'_i = D + b -> bf16 -> proposals (HBM),
//   operand = [s'_i] -> g hidden layers -> SCORE: l_i = <e, D + b>, L_i = log w_i + l_i / lambda
//   -> logits, ordered-int running maximum, prior-weight partial sums.
// P = N and H = 1 in T2Params; the action is the same for every particle, so the action-dependent
// bias rows are parked once in slot 0 of the shared-memory bias table.  Rows stream HBM -> operand
// buffer -> HBM: no per-row register state, so a TWO-SLOT program (hdr.n_slots == 2: narrow models)
// keeps two units in flight, each layer record naming its slot; the epilogue of one unit then
// overlaps the MMAs of the other.
// MODE: 0 the belief update, 1 progressive widening (per-row action / embedding / child maximum),
// 2 diffusion teacher (one denoiser call + DDIM step).  Compile-time: as runtime tests these branches
// cost the plain belief update 8 % (CFG4 propose+score 611 -> 660 us).
template <int MODE>
__device__ __forceinline__ void t2_bu_epilogue(const T2Params &p, const T2Layer *L, uint32_t a_u32, uint32_t tmem_base,
                                               uint64_t *evt, uint64_t *layer_done, float *sbias, int warp, int lane,
                                               uint32_t rank, int cluster_id, int n_clusters, int n_my_units,
                                               int my_slot) {
    // my_slot < 0: this set of eight epilogue warps serves every slot in program order;
    // my_slot = 0 | 1 (16 epilogue warps): it serves one slot and only keeps the books (event,
    // accumulator-block and chunk-free sequence numbers) for the other slot's layer records.
    const int n_layers = p.hdr.n_layers, n_slots = p.hdr.n_slots;
    const int ew = (warp - 4) & 7, qd = warp & 3, half = ew >> 2;
    const uint32_t bar_id = 1u + (uint32_t)(my_slot > 0 ? my_slot : 0);
    const int row = qd * 32 + lane;
    const uint32_t lane_taddr = tmem_base + ((uint32_t)(qd * 32) << 16);
    const int S = p.S, Nz = p.Nz;
    const int in_units = p.hdr.in_chunks * 8;   // f_T input operand, 8-column units
    const int g_units = p.hdr.g_in_chunks * 8;  // g input operand
    const float *e_s = sbias + p.hdr.e_off;
    EpiSync es;
    es.evt_cl = mapa_u32(smem_u32(evt), 0u);
    es.layer_done = layer_done;
    es.cfree = layer_done + kT2AccRing;
    es.lane = lane;
    const EpiConst ec = make_epi_const(a_u32, lane_taddr, sbias, row, half);

    // one-time: action rows of the bias table (slot 0), e = f(o)
    {
        const int tid_e = ((int)threadIdx.x - 128) & 255;  // each set of epilogue warps writes the (same) values
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int li = p.hdr.pa_layer[i];
            if (li >= 0)
                for (int c = tid_e; c < (int)L[li].n_pad; c += 256)
                    sbias[L[li].sbias_off + c] = __ldg(p.bias + L[li].bias_off + (size_t)p.bu_action * L[li].n_pad + c);
        }
        // (MODE 0: e = f(o) comes from the kernel launched just before this one; it is copied at the
        //  first SCORE epilogue, after griddepcontrol.wait: programmatic dependent launch)
        if (MODE != 0)
            for (int c = tid_e; c < p.hdr.e_pad; c += 256) sbias[p.hdr.e_off + c] = 0.0f;
    }

    // particle index of this thread's row in (unit, slot)
    auto row_index = [&](int unit_local, int slot) {
        const int unit = cluster_id + unit_local * n_clusters;
        return ((unit * n_slots + slot) * 2 + (int)rank) * kT2Rows + row;
    };
    // f_T input [s_i ; w_i ; 0] of a row straight into the slot's operand chunks (half 0 warps)
    // (worker: the half of the warps that does it -- a row belongs to one thread of each half)
    auto load_input = [&](int unit_local, int slot, uint32_t a_slot, int worker = 0) {
        if (half != worker) return;
        const int i_idx = row_index(unit_local, slot);
        if (MODE == 4) {  // [bf16(obs)] of a stored branch
            const bool ok = i_idx < p.P && (i_idx % p.slot_M) < __ldg(p.slot_count + i_idx / p.slot_M);
            for (int u = 0; u < in_units; ++u) {
                uint4 v = make_uint4(0u, 0u, 0u, 0u);
                if (ok && 8 * u < p.O) {
                    const float4 *xp = reinterpret_cast<const float4 *>(p.slot_obs + (size_t)i_idx * p.O) + 2 * u;
                    const float4 x0 = __ldg(xp), x1 = __ldg(xp + 1);
                    v = make_uint4(pack_bf16x2(x0.x, x0.y), pack_bf16x2(x0.z, x0.w), pack_bf16x2(x1.x, x1.y),
                                   pack_bf16x2(x1.z, x1.w));
                }
                st_shared_v4(a_unit_addr(a_slot, row, u), v.x, v.y, v.z, v.w);
            }
            return;
        }
        if (MODE == 3) {  // [s_src ; w_T(src) ; onehot(a_g)] of the simulation that opened the slot
            const int src = i_idx < p.P ? __ldg(p.slot_src + i_idx) : -1;
            const int a_row = src >= 0 ? __ldg(p.slot_action + i_idx / p.slot_M) : -1;
            int un = 0;
            for (int u = 0; u < (S >> 3); ++u, ++un) {
                uint4 v = make_uint4(0u, 0u, 0u, 0u);
                if (src >= 0) v = load_row_unit(p.particles + (size_t)src * p.S_io, p.S_io, u);
                st_shared_v4(a_unit_addr(a_slot, row, un), v.x, v.y, v.z, v.w);
            }
            for (int u = 0; u < (Nz >> 3); ++u, ++un) {
                const uint4 v = noise_unit8(p.seed, (uint32_t)(src >= 0 ? src : 0), 0u, 0u, kStreamBeliefT, (uint32_t)u);
                st_shared_v4(a_unit_addr(a_slot, row, un), v.x, v.y, v.z, v.w);
            }
            for (int u = 0; u < ((p.A + 7) >> 3); ++u, ++un) {
                const bool here = a_row >= 0 && (a_row >> 3) == u;
                const int wsel = (a_row & 7) >> 1;
                const uint32_t one = (a_row & 1) ? 0x3F800000u : 0x00003F80u;
                st_shared_v4(a_unit_addr(a_slot, row, un), (here && wsel == 0) ? one : 0u, (here && wsel == 1) ? one : 0u,
                             (here && wsel == 2) ? one : 0u, (here && wsel == 3) ? one : 0u);
            }
            for (; un < in_units; ++un) st_shared_v4(a_unit_addr(a_slot, row, un), 0u, 0u, 0u, 0u);
            return;
        }
        const bool valid = i_idx < p.P;
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (8 * u < S) {
                uint4 v = make_uint4(0u, 0u, 0u, 0u);
                if (valid) v = load_row_unit(p.particles + (size_t)i_idx * p.S_io, p.S_io, u);
                st_shared_v4(a_unit_addr(a_slot, row, u), v.x, v.y, v.z, v.w);
            }
        }
        const int u0 = S >> 3;
        int u_next = u0;
        if (MODE == 2) {
            // diffusion teacher: the current x (bf16 operand copy of the fp32 state; omega at the first step)
            for (int u = 0; u < (p.diff_D >> 3); ++u) {
                uint4 v = make_uint4(0u, 0u, 0u, 0u);
                if (p.diff_first) {
                    v = noise_unit8(p.seed, (uint32_t)i_idx, 0u, 0u, kStreamDiffusion, (uint32_t)u);
                } else if (valid) {
                    const float4 *xp = reinterpret_cast<const float4 *>(p.diff_x + (size_t)i_idx * p.diff_D) + 2 * u;
                    const float4 x0 = __ldg(xp), x1 = __ldg(xp + 1);
                    v = make_uint4(pack_bf16x2(x0.x, x0.y), pack_bf16x2(x0.z, x0.w), pack_bf16x2(x1.x, x1.y),
                                   pack_bf16x2(x1.z, x1.w));
                }
                st_shared_v4(a_unit_addr(a_slot, row, u0 + u), v.x, v.y, v.z, v.w);
            }
            u_next = u0 + (p.diff_D >> 3);
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (8 * u < Nz) {
                    const uint4 v = noise_unit8(p.seed, (uint32_t)i_idx, 0u, 0u, kStreamBeliefT, (uint32_t)u);
                    st_shared_v4(a_unit_addr(a_slot, row, u0 + u), v.x, v.y, v.z, v.w);
                }
            }
            u_next = u0 + (Nz >> 3);
        }
        if (MODE >= 1) {
            // per-row action: the one-hot block is part of the operand, columns [S + Nz, S + Nz + A)
            const int a_row = valid ? __ldg(p.pw_sim_action + i_idx) : -1;
            const int n_u = (p.A + 7) >> 3;
            for (int u = 0; u < n_u; ++u) {
                // bf16 1.0 at column a_row of the block (selects, no dynamically indexed array: that went to local memory)
                const bool here = a_row >= 0 && (a_row >> 3) == u;
                const int wsel = (a_row & 7) >> 1;
                const uint32_t one = (a_row & 1) ? 0x3F800000u : 0x00003F80u;
                st_shared_v4(a_unit_addr(a_slot, row, u_next + u), (here && wsel == 0) ? one : 0u,
                             (here && wsel == 1) ? one : 0u, (here && wsel == 2) ? one : 0u,
                             (here && wsel == 3) ? one : 0u);
            }
            u_next += n_u;
        }
        for (int u = u_next; u < in_units; ++u) st_shared_v4(a_unit_addr(a_slot, row, u), 0u, 0u, 0u, 0u);
    };

    if (n_my_units > 0) {
        for (int s = 0; s < n_slots; ++s) {  // one initial event per slot (hdr.init_events)
            if (my_slot >= 0 && s != my_slot) {
                ++es.ev;
                continue;
            }
            load_input(0, s, a_u32 + (uint32_t)(s * p.hdr.slot_chunks) * kT2ChunkBytes);
            named_bar_sync(bar_id, 256);  // also orders the bias-table writes above before their first use
            fence_proxy_async_smem();
            es.arrive_event();
        }
    }
    es.tl_kind = my_slot > 0 ? 5u : 3u;
    for (int step = 0; step < n_my_units; ++step) {
#ifdef VOILA_T2_TRACE
        es.tl_on = blockIdx.x == 0 && ew == 0 && lane == 0 && step >= g_t2_tl_win[0] && step < g_t2_tl_win[1];
#endif
        for (int li = 0; li < n_layers; ++li) {
            const T2Layer l = L[li];
            es.tl_layer = (uint32_t)li;
            const int slot = l.slot;
            const float *bias = sbias + l.sbias_off;
            const uint32_t a_slot = a_u32 + (uint32_t)l.chunk_off * kT2ChunkBytes;
            const uint32_t taddr = lane_taddr + (uint32_t)l.col_off;
            if (my_slot >= 0 && p.hdr.split_hidden && l.epi == T2_EPI_HIDDEN) {
                // both sets share the layer: this set takes the chunks of its parity (four epilogue
                // warps per scheduler on every layer instead of two: a set alone is latency-bound)
                EpiConst ecs = ec;
                ecs.st_base += (uint32_t)l.chunk_off * kT2ChunkBytes;
                ecs.taddr0 += (uint32_t)l.col_off;
                epi_hidden_layer_par(es, l, (int)l.sbias_off, ecs, my_slot);
                continue;
            }
            if (my_slot >= 0 && slot != my_slot) {  // the other set's record: sequence numbers only
                const bool hid = l.epi == T2_EPI_HIDDEN;
                es.ev += (hid && !l.one_event) ? (int)(l.n_pad >> 6) : 1;
                es.ld_seq += hid ? (uint32_t)__popc((unsigned)l.blk_mask) : 1u;
                if (hid && l.wait_chunks > 0) es.free_seq += ((uint32_t)l.wait_chunks + l.free_nk - 1u) / l.free_nk;
                continue;
            }
            if (l.epi == T2_EPI_HIDDEN) {
                EpiConst ecs = ec;
                ecs.st_base += (uint32_t)l.chunk_off * kT2ChunkBytes;
                ecs.taddr0 += (uint32_t)l.col_off;
                epi_hidden_layer(es, l, (int)l.sbias_off, ecs);
            } else if (MODE < 2 && l.epi == T2_EPI_PROPOSAL) {
                const int i_idx = row_index(step, slot);
                const bool valid = i_idx < p.P;
                es.wait_layer();
                T2_TL(es.tl_on, (es.tl_kind << 24) | (es.tl_layer << 8) | 0xffu);
                if (half == 0) {
                    // the stored particle is what the filter carries forward: bf16(s'); 16 columns
                    // at a time: TMEM -> + bias -> bf16 -> operand buffer (g's input) and HBM
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        if (16 * g < (int)l.n_pad) {
                            uint32_t v[16], o[8];
                            tmem_ld16(taddr + 16 * g, v);
                            float4 b[4];
#pragma unroll
                            for (int i = 0; i < 4; ++i) b[i] = *(reinterpret_cast<const float4 *>(bias + 16 * g) + i);
                            tmem_ld_wait();
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                o[2 * i] = pack_bf16x2(__uint_as_float(v[4 * i]) + b[i].x,
                                                       __uint_as_float(v[4 * i + 1]) + b[i].y);
                                o[2 * i + 1] = pack_bf16x2(__uint_as_float(v[4 * i + 2]) + b[i].z,
                                                           __uint_as_float(v[4 * i + 3]) + b[i].w);
                            }
#pragma unroll
                            for (int h2 = 0; h2 < 2; ++h2) {
                                const int u = 2 * g + h2;
                                if (8 * u < S) {
                                    st_shared_v4(a_unit_addr(a_slot, row, u), o[4 * h2], o[4 * h2 + 1], o[4 * h2 + 2],
                                                 o[4 * h2 + 3]);
                                    if (valid)
                                        store_row_unit(p.bu_proposals + (size_t)i_idx * p.S_io, p.S_io, u,
                                                       make_uint4(o[4 * h2], o[4 * h2 + 1], o[4 * h2 + 2], o[4 * h2 + 3]));
                                }
                            }
                        }
                    }
                } else {
                    for (int u = S >> 3; u < g_units; ++u) st_shared_v4(a_unit_addr(a_slot, row, u), 0u, 0u, 0u, 0u);
                }
                fence_proxy_async_smem();
                tc_fence_before();
                es.arrive_event();
                T2_TL(es.tl_on, ((es.tl_kind + 1u) << 24) | (es.tl_layer << 8) | 0xffu);
            } else if (MODE == 3 && l.epi == T2_EPI_CHAIN) {
                // opened branches: s' -> bf16 -> the state units of f_Z's input; the other half of the warps
                // writes w_Z(src) (stream 5), the one-hot block and the zero padding
                const int i_idx = row_index(step, slot);
                const int src = i_idx < p.P ? __ldg(p.slot_src + i_idx) : -1;
                es.wait_layer();
                if (half == 0) {
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        if (16 * g < (int)l.n_pad) {
                            uint32_t v[16], o[8];
                            tmem_ld16(taddr + 16 * g, v);
                            float4 b[4];
#pragma unroll
                            for (int i = 0; i < 4; ++i) b[i] = *(reinterpret_cast<const float4 *>(bias + 16 * g) + i);
                            tmem_ld_wait();
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                o[2 * i] = pack_bf16x2(__uint_as_float(v[4 * i]) + b[i].x, __uint_as_float(v[4 * i + 1]) + b[i].y);
                                o[2 * i + 1] = pack_bf16x2(__uint_as_float(v[4 * i + 2]) + b[i].z, __uint_as_float(v[4 * i + 3]) + b[i].w);
                            }
#pragma unroll
                            for (int h2 = 0; h2 < 2; ++h2) {
                                const int u = 2 * g + h2;
                                if (8 * u < S)
                                    st_shared_v4(a_unit_addr(a_slot, row, u), o[4 * h2], o[4 * h2 + 1], o[4 * h2 + 2], o[4 * h2 + 3]);
                            }
                        }
                    }
                } else {
                    const int a_row = src >= 0 ? __ldg(p.slot_action + i_idx / p.slot_M) : -1;
                    int un = S >> 3;
                    for (int u = 0; u < (Nz >> 3); ++u, ++un) {
                        const uint4 v = noise_unit8(p.seed, (uint32_t)(src >= 0 ? src : 0), 0u, 0u, kStreamPwObs, (uint32_t)u);
                        st_shared_v4(a_unit_addr(a_slot, row, un), v.x, v.y, v.z, v.w);
                    }
                    for (int u = 0; u < ((p.A + 7) >> 3); ++u, ++un) {
                        const bool here = a_row >= 0 && (a_row >> 3) == u;
                        const int wsel = (a_row & 7) >> 1;
                        const uint32_t one = (a_row & 1) ? 0x3F800000u : 0x00003F80u;
                        st_shared_v4(a_unit_addr(a_slot, row, un), (here && wsel == 0) ? one : 0u, (here && wsel == 1) ? one : 0u,
                                     (here && wsel == 2) ? one : 0u, (here && wsel == 3) ? one : 0u);
                    }
                    for (; un < in_units; ++un) st_shared_v4(a_unit_addr(a_slot, row, un), 0u, 0u, 0u, 0u);
                }
                fence_proxy_async_smem();
                tc_fence_before();
                es.arrive_event();
            } else if (MODE >= 3) {  // T2_EPI_OBS_STORE (MODE 3) | T2_EPI_EMB_STORE (MODE 4): last layer of the unit
                const int i_idx = row_index(step, slot);
                bool ok = i_idx < p.P;
                if (MODE == 3) ok = ok && __ldg(p.slot_src + i_idx) >= 0;
                else ok = ok && (i_idx % p.slot_M) < __ldg(p.slot_count + i_idx / p.slot_M);
                const int width = MODE == 3 ? p.O : p.d;
                float *dst = (MODE == 3 ? p.slot_obs : p.slot_emb) + (size_t)i_idx * width;
                es.wait_layer();
                if (half == 0) {
#pragma unroll
                    for (int g = 0; g < 8; ++g) {
                        if (16 * g < (int)l.n_pad) {
                            uint32_t v[16];
                            tmem_ld16(taddr + 16 * g, v);
                            float4 b[4];
#pragma unroll
                            for (int i = 0; i < 4; ++i) b[i] = *(reinterpret_cast<const float4 *>(bias + 16 * g) + i);
                            tmem_ld_wait();
#pragma unroll
                            for (int i = 0; i < 4; ++i)
                                if (ok && 16 * g + 4 * i < width)
                                    *(reinterpret_cast<float4 *>(dst) + 4 * g + i) =
                                        make_float4(__uint_as_float(v[4 * i]) + b[i].x, __uint_as_float(v[4 * i + 1]) + b[i].y,
                                                    __uint_as_float(v[4 * i + 2]) + b[i].z, __uint_as_float(v[4 * i + 3]) + b[i].w);
                        }
                    }
                }
                if (step + 1 < n_my_units) load_input(step + 1, slot, a_slot);
                named_bar_sync(bar_id, 256);
                fence_proxy_async_smem();
                tc_fence_before();
                es.arrive_event();
            } else if (MODE == 2) {  // T2_EPI_DIFFUSE: diffusion teacher, last (only) network of the unit
                const int i_idx = row_index(step, slot);
                const bool valid = i_idx < p.P;
                const int D = p.diff_D;
                es.wait_layer();
                T2_TL(es.tl_on, (es.tl_kind << 24) | (es.tl_layer << 8) | 0xffu);
                if (half == 0) {
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        if (16 * g < (int)l.n_pad) {
                            uint32_t v[16];
                            tmem_ld16(taddr + 16 * g, v);
                            float4 b[4], x[4];
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                b[i] = *(reinterpret_cast<const float4 *>(bias + 16 * g) + i);
                                x[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                                if (16 * g + 4 * i < D) {
                                    if (p.diff_first) {
                                        x[i] = normals_f4(p.seed, (uint32_t)i_idx, 0u, 0u, kStreamDiffusion,
                                                          (uint32_t)(4 * g + i));
                                    } else if (valid) {
                                        x[i] = __ldg(reinterpret_cast<const float4 *>(p.diff_x + (size_t)i_idx * D) + 4 * g + i);
                                    }
                                }
                            }
                            tmem_ld_wait();
                            // v-prediction and the DDIM step (eta = 0) per element
                            auto upd = [&](float xx, uint32_t d, float bb) {
                                const float vv = __uint_as_float(d) + bb;
                                const float x0_hat = p.al * xx - p.si * vv, eps_hat = p.si * xx + p.al * vv;
                                return p.al_n * x0_hat + p.si_n * eps_hat;
                            };
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                if (valid && 16 * g + 4 * i < D) {
                                    const float4 o = make_float4(upd(x[i].x, v[4 * i], b[i].x), upd(x[i].y, v[4 * i + 1], b[i].y),
                                                                 upd(x[i].z, v[4 * i + 2], b[i].z), upd(x[i].w, v[4 * i + 3], b[i].w));
                                    *(reinterpret_cast<float4 *>(p.diff_x + (size_t)i_idx * D) + 4 * g + i) = o;
                                }
                            }
                        }
                    }
                }
                if (step + 1 < n_my_units) load_input(step + 1, slot, a_slot);
                named_bar_sync(bar_id, 256);
                fence_proxy_async_smem();
                tc_fence_before();
                es.arrive_event();
                T2_TL(es.tl_on, ((es.tl_kind + 1u) << 24) | (es.tl_layer << 8) | 0xffu);
            } else {  // T2_EPI_SCORE: last layer of the slot's unit
                const int i_idx = row_index(step, slot);
                const bool valid = i_idx < p.P;
                float w = 1.0f, lw = 0.0f;
                if (half == 0 && p.weights) {
                    w = valid ? __ldg(p.weights + i_idx) : 0.0f;
                    lw = w > 0.0f ? logf(w) : -INFINITY;
                }
                // progressive widening: the row's own embedding (rows of e_pad floats, zero-padded)
                const float *e_row = nullptr;
                int seg = 0;
                if (MODE == 1 && half == 0) {
                    seg = valid ? __ldg(p.pw_sim_seg + i_idx) : 0;
                    e_row = p.pw_E + (size_t)seg * (size_t)p.hdr.e_pad;
                }
                if (MODE == 0 && step == 0) {
                    // everything the previous kernel produced (e, the reset running maximum) is needed from
                    // here on only: wait for it now, park e in shared memory
                    asm volatile("griddepcontrol.wait;" ::: "memory");
                    const int tid_e = ((int)threadIdx.x - 128) & 255;
                    for (int c = tid_e; c < p.hdr.e_pad; c += 256)
                        sbias[p.hdr.e_off + c] = c < p.d ? p.bu_e[c] : 0.0f;
                    named_bar_sync(bar_id, 256);
                }
                es.wait_layer();
                T2_TL(es.tl_on, (es.tl_kind << 24) | (es.tl_layer << 8) | 0xffu);
                if (half == 0) {
                    float ell = 0.0f;
#pragma unroll
                    for (int g = 0; g < 8; ++g) {
                        if (16 * g < (int)l.n_pad) {
                            uint32_t v[16];
                            tmem_ld16(taddr + 16 * g, v);
                            float4 b[4], e4[4];
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                b[i] = *(reinterpret_cast<const float4 *>(bias + 16 * g) + i);
                                e4[i] = MODE == 1 ? __ldg(reinterpret_cast<const float4 *>(e_row + 16 * g) + i)
                                                  : *(reinterpret_cast<const float4 *>(e_s + 16 * g) + i);
                            }
                            tmem_ld_wait();
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                ell = fmaf(e4[i].x, __uint_as_float(v[4 * i]) + b[i].x, ell);
                                ell = fmaf(e4[i].y, __uint_as_float(v[4 * i + 1]) + b[i].y, ell);
                                ell = fmaf(e4[i].z, __uint_as_float(v[4 * i + 2]) + b[i].z, ell);
                                ell = fmaf(e4[i].w, __uint_as_float(v[4 * i + 3]) + b[i].w, ell);
                            }
                        }
                    }
                    const float Lg = lw + ell * p.inv_lambda;
                    int ord = float_to_ordered(valid ? Lg : -INFINITY);
                    if (valid) p.bu_logits[i_idx] = Lg;
                    if (MODE == 1) {  // the maximum of the row's own child belief; no evidence sums
                        if (valid) atomicMax(p.pw_seg_max + seg, ord);
                        ord = (int)0x80000000;
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) ord = max(ord, __shfl_xor_sync(0xffffffffu, ord, o));
                    double ws = valid ? (double)w : 0.0;
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) ws += __shfl_xor_sync(0xffffffffu, ws, o);
                    const int i0 = i_idx - lane;  // first particle of this warp's 32 rows
                    if (MODE == 0 && lane == 0 && i0 < p.P) {
                        atomicMax(p.bu_max_ordered, ord);
                        p.bu_part_wsum[i0 >> 5] = ws;
                    }
                }
                // this slot's next unit: its input goes into the slot's operand chunks with this event; the
                // warps that had no part in the score fetch the rows and draw the noise meanwhile
                if (step + 1 < n_my_units) load_input(step + 1, slot, a_slot, 1);
                named_bar_sync(bar_id, 256);
                fence_proxy_async_smem();
                tc_fence_before();
                es.arrive_event();
                T2_TL(es.tl_on, ((es.tl_kind + 1u) << 24) | (es.tl_layer << 8) | 0xffu);
            }
        }
    }
}

// NTHREADS: 384 (8 epilogue warps) or 640 (16: one set of 8 per slot of a two-slot program).
// R_LOW / R_HIGH: registers per thread of the producer/issuer warpgroup and of the epilogue
// warpgroups after `setmaxnreg` (their total must fit the launch allocation).
// R_HELP: registers of the second set of epilogue warps (warps 12-19 of a 640-thread kernel);
// > 0: raised to R_HELP, < 0: lowered to -R_HELP.
template <bool BELIEF, int NTHREADS, int R_LOW, int R_HIGH, int R_HELP, int MODE>
__device__ __forceinline__ void tc2_body(const T2Params &p, const CUtensorMap &wmap) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw_u32 = smem_u32(smem_raw);
    uint8_t *smem = smem_raw + (((raw_u32 + 1023u) & ~1023u) - raw_u32);
    const Smem2 map = smem2_map(p.hdr);
    T2Layer *L = reinterpret_cast<T2Layer *>(smem + map.layers);
    T2TileDev *T = reinterpret_cast<T2TileDev *>(smem + map.tiles);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + map.bars);
    uint64_t *empty = full + 8;
    uint64_t *evt = empty + 8;
    uint64_t *layer_done = evt + kT2EvtRing;
    uint32_t *tmem_ptr = reinterpret_cast<uint32_t *>(smem + map.misc);
    double *red_g = reinterpret_cast<double *>(smem + map.misc + 16);                 // [2 slots][4]
    float *red_w = reinterpret_cast<float *>(smem + map.misc + 16 + 2 * 4 * 8);       // [2 slots][4][64]
    uint8_t *alive_s = smem + map.misc + 16 + 2 * 4 * 8 + 2 * 4 * 64 * 4;             // [2 slots][2][128]
    float *sbias = reinterpret_cast<float *>(smem + map.sbias);
    const uint32_t a_u32 = smem_u32(smem + map.a), ring_u32 = smem_u32(smem + map.ring);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int n_layers = p.hdr.n_layers, n_tiles = p.hdr.n_tiles, n_stages = p.hdr.n_stages;

    // ---- one-time setup: program -> smem, zero the operand buffer, barriers, TMEM ----
    {
        const uint32_t *src = reinterpret_cast<const uint32_t *>(p.layers);
        uint32_t *dst = reinterpret_cast<uint32_t *>(L);
        for (int i = threadIdx.x; i < n_layers * (int)(sizeof(T2Layer) / 4); i += NTHREADS) dst[i] = src[i];
        src = reinterpret_cast<const uint32_t *>(p.tiles);
        dst = reinterpret_cast<uint32_t *>(T);
        for (int i = threadIdx.x; i < n_tiles * (int)(sizeof(T2TileDev) / 4); i += NTHREADS) dst[i] = src[i];
        for (int i = threadIdx.x; i < p.hdr.sbias_floats; i += NTHREADS) sbias[i] = p.sbias_init[i];
        uint4 *az = reinterpret_cast<uint4 *>(smem + map.a);
        for (int i = threadIdx.x; i < p.hdr.a_chunks * kT2ChunkBytes / 16; i += NTHREADS)
            az[i] = make_uint4(0u, 0u, 0u, 0u);
        fence_proxy_async_smem();
    }
    if (warp == 0 && lane == 0) tma_prefetch_desc(&wmap);
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < 8; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 1);
        }
        for (int i = 0; i < kT2EvtRing; ++i) mbar_init(&evt[i], 16);  // 8 epilogue warps x 2 CTAs
        for (int i = 0; i < kT2AccRing + kT2FreeRing; ++i) mbar_init(&layer_done[i], 1);  // + cfree ring
        fence_barrier_init();
    }
    if (warp == 2) {
        tmem_alloc_2cta(tmem_ptr, (uint32_t)p.hdr.tmem_cols);
        tmem_relinquish_2cta();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();  // the peer's barriers and TMEM exist before anything signals them
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    const int cluster_id = (int)blockIdx.x >> 1, n_clusters = (int)gridDim.x >> 1;
    const int n_my_units = (p.n_units - cluster_id + n_clusters - 1) / n_clusters;
    const int total_steps = n_my_units * p.H;

    // the epilogue warpgroups take the registers the producer / issuer warpgroup does not need
    if (warp < 4) {
    setmaxnreg_dec<R_LOW>();
    if (warp == 0) {
        // ===== producer: this CTA's half of every weight tile, in issue order, once per step =====
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            const uint32_t stage_bytes = (uint32_t)p.hdr.stage_rows * 128u;
            long long tr_empty = 0;
            const long long tr_start = clock64();
            for (int step = 0; step < total_steps; ++step) {
                for (int i = 0; i < n_tiles; ++i) {
                    const uint32_t src_row = T[i].src_row;
                    const int rows = (int)(T[i].misc >> 16);
                    {
                        T2_TRACE_T0();
                        mbar_wait(&empty[stage], phase ^ 1u);
                        T2_TRACE_ADD(tr_empty);
                    }
                    if (rank == 0) mbar_arrive_expect_tx(&full[stage], 2u * stage_bytes);
                    tma_load_2d_2cta(smem + map.ring + stage * stage_bytes, &wmap, &full[stage], 0,
                                     (int32_t)src_row + (int32_t)rank * rows);
                    if (++stage == (uint32_t)n_stages) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
            }
#ifdef VOILA_T2_TRACE
            if (cluster_id == 0) {
                g_t2_trace[(int)rank * 2] = tr_empty;
                g_t2_trace[(int)rank * 2 + 1] = clock64() - tr_start;
            }
#endif
            (void)tr_empty; (void)tr_start;
        }
    } else if (warp == 1) {
        // ===== MMA issuer: leader CTA only.  The whole warp walks the tile program (waits are
        // warp-uniform); one elected lane issues the MMAs and commits.  (A second issuer warp taking the
        // tiles of the other slot / of the odd accumulator blocks was built and measured: no gain, and
        // its per-tile ownership test alone cost the one-issuer kernel 3 % -- every instruction of this
        // loop is on the critical path.) =====
        if (rank == 0) {
            uint32_t stage = 0, phase = 0;
            uint32_t tl_n = 0;
            (void)tl_n;
            int waited0 = -1, waited1 = -1;  // latest event waited for, per publishing set (T2Tile::need2)
            const uint32_t a_desc_lo = (uint32_t)umma_desc_sw128(a_u32), ring_desc_lo = (uint32_t)umma_desc_sw128(ring_u32);
            const uint32_t desc_hi = (uint32_t)(umma_desc_sw128(0u) >> 32);
            const uint32_t stage_b16 = (uint32_t)p.hdr.stage_rows * 8u;  // stage bytes / 16 (descriptor units)
            uint32_t b_stage = ring_desc_lo;  // descriptor low word of the current ring stage (kept running: a
                                              // multiply here sat between the weight wait and the first MMA)
            int base = p.hdr.init_events, blk_base = 0;
            uint32_t free_seq = 0;
            uint64_t *cfree = layer_done + kT2AccRing;
            long long tr_evt = 0, tr_full = 0, tr_mma = 0, tr_commit = 0;
            const long long tr_start = clock64();
            // the next tile's record is fetched while the current tile waits / issues (its shared-memory
            // latency is otherwise at the head of every tile's dependent chain)
            uint4 r0n = *reinterpret_cast<const uint4 *>(T), r1n = *(reinterpret_cast<const uint4 *>(T) + 1);
            for (int step = 0; step < total_steps; ++step) {
                for (int i = 0; i < n_tiles; ++i) {
                    const uint4 r0 = r0n, r1 = r1n;
                    {
                        const int ni = i + 1 < n_tiles ? i + 1 : 0;
                        r0n = *reinterpret_cast<const uint4 *>(T + ni);
                        r1n = *(reinterpret_cast<const uint4 *>(T + ni) + 1);
                    }
#ifdef VOILA_T2_TRACE
                    const bool tl_on = cluster_id == 0 && lane == 0 && step >= g_t2_tl_win[0] && step < g_t2_tl_win[1];
#endif
                    // events needed from epilogue set 0 and set 1 (-100000: nothing to wait for)
                    const int n0 = base + (int)r1.x, n1 = base + (int)r1.y;
                    T2_TL_ISSUER(tl_on, (7u << 24) | (uint32_t)i);
                    if (n0 > waited0) {
                        T2_TRACE_T0();
                        mbar_wait(&evt[n0 & (kT2EvtRing - 1)], (uint32_t)(n0 / kT2EvtRing) & 1u);
                        T2_TRACE_ADD(tr_evt);
                        waited0 = n0;
                    }
                    if (n1 > waited1) {
                        T2_TRACE_T0();
                        mbar_wait(&evt[n1 & (kT2EvtRing - 1)], (uint32_t)(n1 / kT2EvtRing) & 1u);
                        T2_TRACE_ADD(tr_evt);
                        waited1 = n1;
                    }
                    T2_TL_ISSUER(tl_on, (8u << 24) | (uint32_t)i);
                    {
                        T2_TRACE_T0();
                        mbar_wait(&full[stage], phase);
                        T2_TRACE_ADD(tr_full);
                    }
                    T2_TL_ISSUER(tl_on, (9u << 24) | (uint32_t)i);
                    tc_fence_after();
                    T2_TL_ISSUER(tl_on, (1u << 24) | (uint32_t)i);
                    const uint32_t misc = r1.w;
                    if (elect_one_sync()) {
                    const uint32_t d = tmem_base + r0.w;
                    const uint32_t nk = misc & 15u;
                    uint32_t acc = (misc & 16u) ? 0u : 1u;
#ifdef VOILA_T2_TRACE
                    const long long tm0 = clock64();
#endif
                    // descriptors differ only in their 14-bit address field (units of 16 bytes): add
                    // offsets to the low word instead of rebuilding them (the rebuilt form was ~100
                    // uniform-datapath instructions per tile)
                    uint32_t a_lo = a_desc_lo + r0.z;
                    uint32_t b_lo = b_stage;
#pragma unroll
                    for (int c = 0; c < 4; ++c) {  // a stage holds up to 4 K chunks
                        if (c >= (int)nk) break;
#pragma unroll
                        for (int k = 0; k < 4; ++k) {  // 64-wide chunk = 4 x (K = 16); +32 bytes per K step
                            umma_ss_2cta(d, ((uint64_t)desc_hi << 32) | (a_lo + 2u * k),
                                         ((uint64_t)desc_hi << 32) | (b_lo + 2u * k), r0.y, acc);
                            acc = 1u;
                        }
                        a_lo += kT2ChunkBytes >> 4;
                        b_lo += r1.z;
                    }
#ifdef VOILA_T2_TRACE
                    const long long tm1 = clock64();
                    tr_mma += tm1 - tm0;
#endif
                    umma_commit_2cta(&empty[stage], 3);
                    if (misc & 64u) umma_commit_2cta(&cfree[free_seq & (kT2FreeRing - 1)], 3);
                    if (misc & 32u)
                        umma_commit_2cta(&layer_done[((uint32_t)blk_base + ((misc >> 8) & 255u)) & (kT2AccRing - 1)], 3);
#ifdef VOILA_T2_TRACE
                    tr_commit += clock64() - tm1;
#endif
                    }
                    __syncwarp();
                    T2_TL_ISSUER(tl_on, (2u << 24) | (uint32_t)i);
                    free_seq += (misc >> 6) & 1u;
                    b_stage += stage_b16;
                    if (++stage == (uint32_t)n_stages) {
                        stage = 0;
                        phase ^= 1u;
                        b_stage = ring_desc_lo;
                    }
                }
                base += p.hdr.evt_per_step;
                blk_base += p.hdr.blocks_per_step;
            }
#ifdef VOILA_T2_TRACE
            if (cluster_id == 0 && elect_one_sync()) {
                g_t2_trace[4] = tr_evt;
                g_t2_trace[5] = tr_full;
                g_t2_trace[6] = clock64() - tr_start;
                g_t2_trace[7] = tr_mma;
                g_t2_trace[8] = tr_commit;
            }
#endif
            (void)tr_evt; (void)tr_full; (void)tr_start; (void)tr_mma; (void)tr_commit;
        }
    }
    } else if (NTHREADS == kT2Threads || warp < 12) {
        setmaxnreg_inc<R_HIGH>();
        if (BELIEF)
            t2_bu_epilogue<BELIEF ? MODE : 0>(p, L, a_u32, tmem_base, evt, layer_done, sbias, warp, lane, rank, cluster_id, n_clusters,
                           n_my_units, NTHREADS == kT2Threads ? -1 : 0);
        else
            t2_epilogue<BELIEF ? 0 : MODE>(p, L, a_u32, tmem_base, evt, layer_done, red_g, red_w, alive_s, sbias, warp, lane, rank,
                        cluster_id, n_clusters, n_my_units, total_steps, NTHREADS != kT2Threads && R_HELP < 0,
                        (NTHREADS != kT2Threads && R_HELP > 0) ? 0 : -1);
    } else {
        // second set of epilogue warps (640-thread kernels)
        if (R_HELP > 0) setmaxnreg_inc<(R_HELP > 0 ? R_HELP : 24)>();
        else setmaxnreg_dec<(R_HELP < 0 ? -R_HELP : 24)>();
        if (BELIEF)
            t2_bu_epilogue<BELIEF ? MODE : 0>(p, L, a_u32, tmem_base, evt, layer_done, sbias, warp, lane, rank, cluster_id, n_clusters,
                           n_my_units, 1);
        else if (R_HELP > 0)  // two-slot rollout: the second slot's own set of stateful epilogue warps
            t2_epilogue<BELIEF ? 0 : MODE>(p, L, a_u32, tmem_base, evt, layer_done, red_g, red_w, alive_s, sbias, warp, lane, rank,
                        cluster_id, n_clusters, n_my_units, total_steps, false, 1);
        else
            t2_helper_epilogue(p, L, a_u32, tmem_base, evt, layer_done, sbias, warp, lane, total_steps);
    }

    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 2) tmem_dealloc_2cta(tmem_base, (uint32_t)p.hdr.tmem_cols);
}

// MODE: rollout kernels 0 | 1 (terminal regions); belief-style kernels 0 | 1 | 2 (see t2_bu_epilogue).
template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kT2Threads, 1)
    rollout_tc2_kernel(const T2Params p, const __grid_constant__ CUtensorMap wmap) {
    tc2_body<false, kT2Threads, 56, 224, 0, MODE>(p, wmap);
}
template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kT2Threads, 1)
    belief_tc2_kernel(const T2Params p, const __grid_constant__ CUtensorMap wmap) {
    tc2_body<true, kT2Threads, 56, 224, 0, MODE>(p, wmap);
}
// Two-slot belief program with one set of eight epilogue warps PER SLOT (20 warps): the two units'
// epilogues run concurrently, four epilogue warps per scheduler hide each other's latencies.
constexpr int kT2ThreadsDual = 640;
template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kT2ThreadsDual, 1)
    belief_tc2_dual_kernel(const T2Params p, const __grid_constant__ CUtensorMap wmap) {
    tc2_body<true, kT2ThreadsDual, 40, 104, 104, MODE>(p, wmap);
}
// Rollout with a second set of epilogue warps that takes the odd chunks of every hidden layer: the
// layer's epilogue (TMEM read, activation, pack, store) runs on 16 warps, four per scheduler.
template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kT2ThreadsDual, 1)
    rollout_tc2x_kernel(const T2Params p, const __grid_constant__ CUtensorMap wmap) {
    tc2_body<false, kT2ThreadsDual, 32, 168, -56, MODE>(p, wmap);
}
// Two-slot rollout (generators whose layers are all <= 256 wide): two 256-particle blocks of one
// sequence in flight per CTA pair, each with its own set of eight stateful epilogue warps (state /
// witness in registers), so that one block's epilogue overlaps the other block's MMAs.
template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kT2ThreadsDual, 1)
    rollout_tc2d_kernel(const T2Params p, const __grid_constant__ CUtensorMap wmap) {
    tc2_body<false, kT2ThreadsDual, 32, 112, 112, MODE>(p, wmap);
}

}  // namespace

// =====================================================================================
// Host side: program construction (weight packing, block shapes, issue order), launcher
// =====================================================================================
namespace {

constexpr size_t kMaxDynSmem2 = 232448;  // 227 KB per CTA on sm_100

uint16_t h_bf16_bits(float x) {
    uint32_t u;
    std::memcpy(&u, &x, 4);
    if ((u & 0x7f800000u) != 0x7f800000u) u += 0x7fffu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}
float h_bf16_round(float x) {
    const uint32_t u = (uint32_t)h_bf16_bits(x) << 16;
    float y;
    std::memcpy(&y, &u, 4);
    return y;
}
int rup(int x, int m) { return (x + m - 1) / m * m; }

// Accumulator block widths of a hidden layer of width n (multiple of 64).  Narrow blocks first:
// the next layer's MMAs may start as soon as the epilogue has drained the first block, and a
// block's tiles all wait for the block's LAST column to be drained.
std::vector<int> hidden_blocks(int n, int policy) {
    std::vector<int> b;
    int left = n;
    if (policy == 0 && n <= 256) policy = 2;  // a 256-wide layer as two 128 blocks: the epilogue of the
                                              // first overlaps the MMAs of the second (measured, CFG3)
    if (policy == 4 && n > 256) {  // 256s, then the last 256 columns as two 128 blocks (short last epilogue)
        while (left > 256) { b.push_back(256); left -= 256; }
        while (left >= 128) { b.push_back(128); left -= 128; }
    }
    if (policy == 0 || policy == 3 || policy == 4) {  // all 256 (N < 256 MMAs run below the tensor pipe's floor: A re-read)
        while (left >= 256) { b.push_back(256); left -= 256; }
    } else if (policy == 2) {  // all 128
        while (left >= 128) { b.push_back(128); left -= 128; }
    } else {  // 1: 128, 128, then 256s
        for (int i = 0; i < 2 && left >= 128; ++i) { b.push_back(128); left -= 128; }
        while (left >= 256) { b.push_back(256); left -= 256; }
    }
    while (left >= 128) { b.push_back(128); left -= 128; }
    if (left > 0) b.push_back(left);  // 64
    return b;
}

struct Builder2 {
    std::vector<T2Layer> layers;
    std::vector<T2Tile> tiles;
    std::vector<uint8_t> wstream;  // rows of 128 bytes
    std::vector<float> bias;        // global: every bias row (SiLU hidden layers pre-halved)
    std::vector<float> sbias_init;  // shared-memory table image: constant rows; 2 empty rows per action layer
    int pa_layer[2] = {-1, -1};
    bool too_many_pa = false;
    bool bad_order = false;
    int evt = 0;
    int col_free[512];
    int a_ready[8];
    int a_chunks = 1;
    // current slot (two-slot programs): operand chunk / TMEM column offsets of the layers added next
    int slot = 0, chunk_off = 0, col_off = 0, slot_chunks = 8;
    int n_blocks = 0;  // accumulator blocks of the step so far (each is handed to the epilogues on its own)
    int policy = 0;
    int stage_rows = 128;  // weight rows per CTA per ring stage (T2Header::stage_rows)

    Builder2() {
        for (int &c : col_free) c = -1;
        for (int &a : a_ready) a = -1;
        if (const char *e = getenv("VOILA_T2_STAGE_ROWS")) stage_rows = atoi(e) == 256 ? 256 : 128;  // tuning knob
    }

    // Two-slot mode: every layer is added once per slot (slot 1 shares slot 0's biases and weight
    // tiles; its operand chunks / TMEM columns are disjoint, so its dependencies are tracked apart).
    bool pingpong = false;         // see add_layer
    bool par_split = false;        // two sets of epilogue warps share every hidden layer (even / odd chunks)
    std::vector<uint8_t> evt_set;  // set that publishes event e of the step
    bool dual = false;
    std::map<uint32_t, uint32_t> tile_src;  // layer << 16 | block << 8 | first K chunk  ->  src_row of the packed tile
    void set_dual(int chunks_per_slot, int cols_per_slot) {
        dual = true;
        slot_chunks = chunks_per_slot;
        dual_cols = cols_per_slot;
        // two-slot programs: one 256-column accumulator block per layer (one hand-off, no in-place
        // chunk-free waits; the OTHER slot's MMAs overlap this slot's epilogue): measured CFG3 750 -> 759
        // TFLOP/s, CFG4 propose+score 630 -> 616 us against two 128-column blocks
        if (policy == 0) policy = 3;
        // slot 0's input / accumulator were last touched by the event BEFORE the previous step's last
        for (int j = 0; j < chunks_per_slot; ++j) a_ready[j] = -2;
        for (int c = 0; c < cols_per_slot; ++c) col_free[c] = -2;
    }
    int dual_cols = 256;

    // W: [n0][k0] row-major fp32 ("algorithmic" column order); bias_rows x n0 biases.
    void add_layer(const float *W, int n0, int k0, const float *b, int bias_rows, int epi, int act) {
        if (!dual) {
            // narrow single-slot programs: consecutive layers accumulate in alternate halves of TMEM, so a
            // layer's tiles wait only for the operand chunks they read (not for the previous layer's
            // accumulator to be drained) and start chunk by chunk while that epilogue is still running
            if (pingpong) col_off = (int)(layers.size() & 1) * 256;
            add_one(W, n0, k0, b, bias_rows, epi, act, -1);
            return;
        }
        slot = 0; chunk_off = 0; col_off = 0;
        const int li = add_one(W, n0, k0, b, bias_rows, epi, act, -1);
        slot = 1; chunk_off = slot_chunks; col_off = dual_cols;
        add_one(W, n0, k0, b, bias_rows, epi, act, li);
    }

    int add_one(const float *W, int n0, int k0, const float *b, int bias_rows, int epi, int act, int same_as) {
        T2Layer l{};
        const bool hidden = epi == T2_EPI_HIDDEN;
        const int n_pad = hidden ? rup(n0, 64) : rup(n0, 16);  // padded neurons: zero weights, zero bias -> act(0) = 0
        const int kc_n = rup(k0, 64) / 64;
        l.bias_off = (uint32_t)bias.size();
        l.n_pad = (uint16_t)n_pad;
        l.epi = (uint8_t)epi;
        l.act = (uint8_t)act;
        l.bias_per_action = bias_rows > 1;
        const float bscale = (hidden && act == VOILA_ACT_SILU) ? 0.5f : 1.0f;  // see act_biased()
        if (same_as < 0)
            for (int r = 0; r < bias_rows; ++r)
                for (int j = 0; j < n_pad; ++j)
                    bias.push_back((b && j < n0) ? bscale * b[(size_t)r * n0 + j] : 0.0f);
        a_chunks = std::max(a_chunks, chunk_off + std::max(kc_n, hidden ? n_pad / 64 : 1));
        l.slot = (uint8_t)slot;
        l.chunk_off = (uint8_t)chunk_off;
        l.col_off = (uint16_t)col_off;
        const int li = (int)layers.size();
        l.sbias_off = (uint32_t)sbias_init.size();
        if (same_as >= 0) {
            l.bias_off = layers[same_as].bias_off;
            l.sbias_off = layers[same_as].sbias_off;
        } else if (bias_rows > 1) {
            sbias_init.resize(sbias_init.size() + 2 * (size_t)n_pad, 0.0f);
            if (pa_layer[0] < 0) pa_layer[0] = li;
            else if (pa_layer[1] < 0) pa_layer[1] = li;
            else too_many_pa = true;
        } else {
            sbias_init.insert(sbias_init.end(), bias.end() - n_pad, bias.end());
        }
        std::vector<int> blocks = hidden ? hidden_blocks(n_pad, policy) : std::vector<int>{n_pad};
        std::vector<T2Tile> lt;
        int n_start = 0;
        for (size_t bi = 0; bi < blocks.size(); ++bi) {
            const int bn = blocks[bi], half = bn / 2;
            const int nk_max = std::max(1, std::min(4, stage_rows / half));
            int blk_need = -1000;
            for (int c = n_start; c < n_start + bn; ++c) blk_need = std::max(blk_need, col_free[col_off + c]);
            for (int kc0 = 0; kc0 < kc_n; kc0 += nk_max) {
                const int nk = std::min(nk_max, kc_n - kc0);
                T2Tile t{};
                t.src_row = (uint32_t)(wstream.size() / 128);
                t.idesc = umma_idesc_bf16_m256((uint32_t)bn);
                t.d_col16 = (uint8_t)((col_off + n_start) / 16);
                t.blk = (uint8_t)(n_blocks + (int)bi);
                t.kc0 = (uint8_t)(chunk_off + kc0);
                t.nk = (uint8_t)nk;
                t.rows8 = (uint8_t)(half / 8);
                t.pad = (uint8_t)slot;  // two-slot programs: the slot (= the MMA issuer warp that owns the tile)
                int need = blk_need;
                for (int c = 0; c < nk; ++c) need = std::max(need, a_ready[chunk_off + kc0 + c]);
                t.need = (int16_t)need;
                t.flags = (uint8_t)(bi << 4);  // scratch: block index, cleared below
                const uint32_t key_bk = ((uint32_t)bi << 8) | (uint32_t)kc0;
                if (same_as >= 0) {  // slot 1 streams the very tile slot 0 packed
                    t.src_row = tile_src.at(((uint32_t)same_as << 16) | key_bk);
                    lt.push_back(t);
                    continue;
                }
                tile_src[((uint32_t)li << 16) | key_bk] = t.src_row;
                // pack: CTA 0's rows then CTA 1's; per CTA chunk by chunk; 16-byte units XOR (row & 7)
                const size_t base = wstream.size();
                wstream.resize(base + (size_t)2 * nk * half * 128, 0);
                for (int r = 0; r < 2; ++r)
                    for (int c = 0; c < nk; ++c)
                        for (int i = 0; i < half; ++i) {
                            uint8_t *dst = wstream.data() + base + ((size_t)(r * nk + c) * half + i) * 128;
                            const int row = n_start + r * half + i;
                            for (int u = 0; u < 8; ++u)
                                for (int e = 0; e < 8; ++e) {
                                    const int k = (kc0 + c) * 64 + u * 8 + e;
                                    const float v = (row < n0 && k < k0) ? W[(size_t)row * k0 + k] : 0.0f;
                                    const uint16_t h = h_bf16_bits(v);
                                    std::memcpy(dst + ((u ^ (i & 7)) * 16) + e * 2, &h, 2);
                                }
                        }
                lt.push_back(t);
            }
            n_start += bn;
        }
        std::stable_sort(lt.begin(), lt.end(), [](const T2Tile &x, const T2Tile &y) { return x.need < y.need; });
        bool seen[16] = {};
        int last_of[16];
        for (size_t i = 0; i < lt.size(); ++i) {
            const int bi = lt[i].flags >> 4;
            lt[i].flags = seen[bi] ? 0 : 1;
            seen[bi] = true;
            last_of[bi] = (int)i;
        }
        // the last tile of every block hands that block of the accumulator to the epilogues
        for (size_t bi = 0; bi < blocks.size(); ++bi) lt[last_of[bi]].flags |= 2;
        {
            int c = 0;
            for (size_t bi = 0; bi < blocks.size(); ++bi) {
                if (hidden) l.blk_mask |= (uint8_t)(1u << c);
                c += blocks[bi] / 64;
            }
        }
        n_blocks += (int)blocks.size();
        if (hidden && blocks.size() > 1) {
            const int last_bi = (int)blocks.size() - 1, last_half = blocks[last_bi] / 2;
            const int nk_last = std::max(1, std::min(4, stage_rows / last_half));
            const int early = (n_pad - blocks[last_bi]) / 64;
            l.free_nk = (uint8_t)nk_last;
            l.wait_chunks = (uint8_t)std::min(early, kc_n);
            int prev_kc0 = -1, n_sig = 0;
            for (T2Tile &t : lt) {
                if ((int)t.blk != n_blocks - 1) continue;
                if ((int)t.kc0 <= prev_kc0) bad_order = true;  // signals must arrive in chunk order
                prev_kc0 = t.kc0;
                if ((int)t.kc0 - chunk_off < (int)l.wait_chunks) {
                    t.flags |= 4;
                    ++n_sig;
                }
            }
            if (n_sig > kT2FreeRing) bad_order = true;
        }
        tiles.insert(tiles.end(), lt.begin(), lt.end());
        l.one_event = (hidden && dual && !par_split && blocks.size() == 1) ? 1 : 0;
        layers.push_back(l);
        if (hidden && l.one_event) {
            for (int c = 0; c < n_pad; ++c) col_free[col_off + c] = evt;
            for (int j = 0; j < n_pad / 64; ++j) a_ready[chunk_off + j] = evt;
            evt_set.push_back(0);
            ++evt;
        } else if (hidden) {
            for (int j = 0; j < n_pad / 64; ++j) {
                for (int c = 64 * j; c < 64 * j + 64; ++c) col_free[col_off + c] = evt;
                a_ready[chunk_off + j] = evt;
                evt_set.push_back((uint8_t)(par_split ? (j & 1) : 0));
                ++evt;
            }
        } else {
            for (int c = 0; c < n_pad; ++c) col_free[col_off + c] = evt;
            if (epi != T2_EPI_REWARD && epi != T2_EPI_SCORE && epi != T2_EPI_DIFFUSE && epi != T2_EPI_OBS_STORE &&
                epi != T2_EPI_EMB_STORE)  // the next layer-1 input is written with this event
                for (int j = chunk_off; j < std::min(8, chunk_off + slot_chunks); ++j) a_ready[j] = evt;
            evt_set.push_back((uint8_t)((dual && par_split) ? slot : 0));
            ++evt;
        }
        return li;
    }

    // After the last layer: the second wait of every tile (see T2Tile::need2).
    void finish_needs() {
        // events repeat with period `evt` (one step); a negative index names an event of the previous step
        auto set_of = [&](int e) { return (int)evt_set[((e % evt) + evt) % evt]; };
        for (T2Tile &t : tiles) {
            const int need = t.need;
            const int set = par_split ? set_of(need) : 0;
            t.need_set = (uint8_t)set;
            int other = -100000;
            if (par_split)
                for (int e = need - 1; e >= need - evt && other < -1000; --e)
                    if (set_of(e) != set) other = e;
            t.need2 = (int16_t)(other > -1000 ? other : need);
        }
    }
};


// One static program resident on the device: tables, packed weight stream, its tensor map.
struct T2Program {
    T2Header hdr{};
    void *d_wstream = nullptr, *d_bias = nullptr, *d_sbias = nullptr, *d_layers = nullptr, *d_tiles = nullptr;
    size_t smem_bytes = 0;
    int max_clusters = 0;
    CUtensorMap wmap;
};

struct T2Handle {
    T2Program roll;    // rollout: [reward] + f_T + f_Z per step
    T2Program belief;       // belief update: f_T + g per 256-particle unit
    T2Program belief_dual;  // the same with two units in flight per CTA pair (narrow models)
    bool has_belief = false, has_belief_dual = false;
    // progressive widening: the belief program with the one-hot block in the operand (per-row actions)
    T2Program pw, pw_dual;
    bool has_pw = false, has_pw_dual = false;
    T2Program pw_open, pw_emb;  // the small passes over the (action node, branch) slots (see T2Params)
    bool has_pw_slots = false;
    // diffusion teachers (0 transition, 1 observation): one denoiser call per launch, [which][dual]
    T2Program diff[2][2];
    bool has_diff[2][2] = {{false, false}, {false, false}};
    float *d_diff_b1[2] = {nullptr, nullptr}, *d_diff_w1t[2] = {nullptr, nullptr};  // layer-1 bias, time-embedding columns
    int diff_n1[2] = {0, 0};
    float diff_scale[2] = {1.0f, 1.0f};
    bool roll_x = false;    // rollout runs the 640-thread kernel (two sets of epilogue warps)
    T2Program roll_dual;    // rollout with two 256-particle blocks in flight per CTA pair (layers <= 256 wide)
    bool has_roll_dual = false;
    int Sp = 0, Nzp = 0;    // operand widths of the state and the noise (public widths rounded up to 8)
};

// Layer 1 of a generator sees the "algorithmic" input [s ; w] (K = S + Nz): the one-hot block is
// folded into a per-action bias row b1 + W1[:, S + a] (R21).
// S, Nz are the PUBLIC widths; in the operand the state occupies rup(S, 8) columns and the noise
// rup(Nz, 8) (paper-shaped states of 39 / 45 coordinates: the pad columns carry zero weights).
void add_generator2(Builder2 &pb, const voila_mlp &f, int S, int A, int Nz, int last_epi) {
    const int Sp = rup(S, 8), Nzp = rup(Nz, 8);
    for (int l = 0; l < f.n_layers; ++l) {
        const int K = f.dims[l], N = f.dims[l + 1];
        const bool last = l == f.n_layers - 1;
        if (l == 0) {
            const int k0 = Sp + Nzp;
            std::vector<float> W((size_t)N * k0, 0.0f), b((size_t)A * N);
            for (int j = 0; j < N; ++j) {
                for (int k = 0; k < S; ++k) W[(size_t)j * k0 + k] = f.W[0][(size_t)j * K + k];
                for (int k = 0; k < Nz; ++k) W[(size_t)j * k0 + Sp + k] = f.W[0][(size_t)j * K + S + A + k];
                for (int a = 0; a < A; ++a)
                    b[(size_t)a * N + j] = f.b[0][j] + h_bf16_round(f.W[0][(size_t)j * K + S + a]);
            }
            pb.add_layer(W.data(), N, k0, b.data(), A, last ? last_epi : T2_EPI_HIDDEN, f.act);
        } else {
            pb.add_layer(f.W[l], N, K, f.b[l], 1, last ? last_epi : T2_EPI_HIDDEN, f.act);
        }
    }
}

// The same generator with the one-hot block kept in the operand, input order [s ; w ; onehot(a)]
// (K = S + Nz + A): rows of a tile may carry different actions (progressive widening).
void add_generator2_dense(Builder2 &pb, const voila_mlp &f, int S, int A, int Nz, int last_epi) {
    for (int l = 0; l < f.n_layers; ++l) {
        const int K = f.dims[l], N = f.dims[l + 1];
        const bool last = l == f.n_layers - 1;
        if (l == 0) {
            const int k0 = S + Nz + A;
            std::vector<float> W((size_t)N * k0);
            for (int j = 0; j < N; ++j) {
                for (int k = 0; k < S; ++k) W[(size_t)j * k0 + k] = f.W[0][(size_t)j * K + k];
                for (int k = 0; k < Nz; ++k) W[(size_t)j * k0 + S + k] = f.W[0][(size_t)j * K + S + A + k];
                for (int a = 0; a < A; ++a) W[(size_t)j * k0 + S + Nz + a] = f.W[0][(size_t)j * K + S + a];
            }
            pb.add_layer(W.data(), N, k0, f.b[0], 1, last ? last_epi : T2_EPI_HIDDEN, f.act);
        } else {
            pb.add_layer(f.W[l], N, K, f.b[l], 1, last ? last_epi : T2_EPI_HIDDEN, f.act);
        }
    }
}

// Denoiser of a diffusion teacher: input order [c ; x ; onehot(a)] (K = S + D + A); the time-embedding
// columns of layer 1 are folded into one bias row per DDIM step (the row is written before the step's
// launch by diffusion_bias_kernel and picked like a per-action row).
constexpr int kT2DiffMaxSteps = 256;
void add_denoiser2(Builder2 &pb, const voila_mlp &f, int S, int A, int D) {
    for (int l = 0; l < f.n_layers; ++l) {
        const int K = f.dims[l], N = f.dims[l + 1];
        const bool last = l == f.n_layers - 1;
        if (l == 0) {
            const int k0 = S + D + A;
            std::vector<float> W((size_t)N * k0);
            for (int j = 0; j < N; ++j) {
                for (int k = 0; k < S; ++k) W[(size_t)j * k0 + k] = f.W[0][(size_t)j * K + k];
                for (int k = 0; k < D; ++k) W[(size_t)j * k0 + S + k] = f.W[0][(size_t)j * K + S + A + k];
                for (int a = 0; a < A; ++a) W[(size_t)j * k0 + S + D + a] = f.W[0][(size_t)j * K + S + a];
            }
            pb.add_layer(W.data(), N, k0, nullptr, kT2DiffMaxSteps, last ? T2_EPI_DIFFUSE : T2_EPI_HIDDEN, f.act);
        } else {
            pb.add_layer(f.W[l], N, K, f.b[l], 1, last ? T2_EPI_DIFFUSE : T2_EPI_HIDDEN, f.act);
        }
    }
}

// bias row of one DDIM step: scale * (b1[j] + sum_e bf16(W1[j][temb e]) * bf16(temb_e)), zero padding
struct TembArg { float v[kTemb]; };
__global__ void diffusion_bias_kernel(float *row, const float *__restrict__ b1, const float *__restrict__ w1t, int n,
                                      int n_pad, float scale, TembArg t) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_pad) return;
    float acc = 0.0f;
    if (j < n) {
        acc = b1[j];
#pragma unroll
        for (int e = 0; e < kTemb; ++e) acc = fmaf(w1t[j * kTemb + e], bf16_round(t.v[e]), acc);
    }
    row[j] = scale * acc;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

// Sizes the program, uploads its tables and weight stream, encodes the tensor map, queries how
// many CTA pairs of `kernel` can be resident.  Returns an empty string on success.
template <typename Kernel>
std::string finish_program(Builder2 &pb, T2Program &g, Kernel kernel, int in_chunks, int sm_count,
                           std::vector<void *> *allocs, int n_threads = kT2Threads) {
    if ((int)pb.layers.size() > kT2MaxLayers || (int)pb.tiles.size() > kT2MaxTiles || pb.too_many_pa || pb.bad_order)
        return "model too deep for the tcgen05 program tables";
    pb.finish_needs();
    // the TMA box is always 128 rows: pad the stream so that the last tile's box stays in bounds
    pb.wstream.resize(pb.wstream.size() + (size_t)pb.stage_rows * 128, 0);
    g.hdr.stage_rows = pb.stage_rows;
    g.hdr.n_layers = (int)pb.layers.size();
    g.hdr.blocks_per_step = pb.n_blocks;
    g.hdr.n_tiles = (int)pb.tiles.size();
    g.hdr.evt_per_step = pb.evt;
    g.hdr.a_chunks = pb.a_chunks;
    g.hdr.in_chunks = in_chunks;
    g.hdr.sbias_floats = (int)pb.sbias_init.size();
    g.hdr.pa_layer[0] = pb.pa_layer[0];
    g.hdr.pa_layer[1] = pb.pa_layer[1];
    int max_n = 32;
    for (const T2Layer &l : pb.layers) max_n = std::max(max_n, (int)l.col_off + (int)l.n_pad);
    g.hdr.init_events = pb.dual ? 2 : 1;
    g.hdr.n_slots = pb.dual ? 2 : 1;
    g.hdr.slot_chunks = pb.dual ? pb.slot_chunks : 0;
    int cols = 32;
    while (cols < max_n) cols *= 2;
    g.hdr.tmem_cols = cols;
    g.hdr.split_hidden = (pb.dual && pb.par_split) ? 1 : 0;
    g.hdr.n_stages = 8;
    if (const char *e = getenv("VOILA_T2_STAGES")) g.hdr.n_stages = std::max(2, std::min(8, atoi(e)));
    while (g.hdr.n_stages > 2 && smem2_map(g.hdr).total + 1024 > kMaxDynSmem2) --g.hdr.n_stages;
    g.smem_bytes = smem2_map(g.hdr).total + 1024;
    if (g.smem_bytes > kMaxDynSmem2) return "model does not fit the shared-memory budget of the tcgen05 pair kernel";
    // device form of the tile records (see T2TileDev)
    std::vector<T2TileDev> dev_tiles;
    for (const T2Tile &t : pb.tiles) {
        T2TileDev d{};
        d.src_row = t.src_row;
        d.idesc = t.idesc;
        d.a_off = (uint32_t)t.kc0 * (uint32_t)(kT2ChunkBytes >> 4);
        d.d_off = (uint32_t)t.d_col16 * 16u;
        const int need = t.need, need2 = t.need2;
        const int s0 = t.need_set ? need2 : need, s1 = t.need_set ? need : need2;
        d.need_s0 = s0;
        d.need_s1 = need2 != need ? s1 : -100000;
        d.chunk_b16 = ((uint32_t)t.rows8 * 1024u) >> 4;
        d.misc = (uint32_t)t.nk | ((uint32_t)(t.flags & 7u) << 4) | ((uint32_t)t.blk << 8) |
                 ((uint32_t)((int)t.nk * (int)t.rows8 * 8) << 16);
        dev_tiles.push_back(d);
    }
    auto upload = [&](const void *src, size_t bytes, void **dst) -> bool {
        if (cudaMalloc(dst, bytes) != cudaSuccess) return false;
        allocs->push_back(*dst);
        return cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess;
    };
    if (!upload(pb.wstream.data(), pb.wstream.size(), &g.d_wstream) ||
        !upload(pb.bias.data(), pb.bias.size() * sizeof(float), &g.d_bias) ||
        !upload(pb.sbias_init.data(), pb.sbias_init.size() * sizeof(float), &g.d_sbias) ||
        !upload(pb.layers.data(), pb.layers.size() * sizeof(T2Layer), &g.d_layers) ||
        !upload(dev_tiles.data(), dev_tiles.size() * sizeof(T2TileDev), &g.d_tiles) ||
        // several programs share one kernel function: ask for the architectural maximum once
        cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxDynSmem2) != cudaSuccess)
        return cudaGetErrorString(cudaGetLastError());
    // weight stream as a 2-D tensor [rows][64 bf16]; box = one ring stage (128 rows x 128 bytes).
    // The tiles are pre-swizzled on the host, so the copy itself does not swizzle.
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess ||
        fn == nullptr || qres != cudaDriverEntryPointSuccess)
        return "cuTensorMapEncodeTiled not available from the driver";
    const cuuint64_t gdim[2] = {64, (cuuint64_t)(pb.wstream.size() / 128)};
    const cuuint64_t gstride[1] = {128};
    const cuuint32_t box[2] = {64, (cuuint32_t)pb.stage_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult cr = reinterpret_cast<EncodeTiledFn>(fn)(
        &g.wmap, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, g.d_wstream, gdim, gstride, box, estr,
        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) return "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)cr);
    // how many CTA pairs can be resident at once (one CTA per SM; normally sm_count / 2)
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)(sm_count & ~1));
    cfg.blockDim = dim3((unsigned)n_threads);
    cfg.dynamicSmemBytes = g.smem_bytes;
    int nc = 0;
    if (cudaOccupancyMaxActiveClusters(&nc, kernel, &cfg) != cudaSuccess || nc < 1) {
        cudaGetLastError();
        nc = sm_count / 2;
    }
    g.max_clusters = std::min(nc, sm_count / 2);
    return std::string();
}

}  // namespace

// The CTA-pair programs pad what the MMA shapes want (state / noise columns to multiples of 8, hidden
// widths to multiples of 64) when the weights are packed; the public buffers keep their widths.
bool tc2_supported(const voila_model_desc *d, std::string *why) {
    auto fail = [&](const char *m) {
        if (why) *why = m;
        return false;
    };
    if (d->prec != VOILA_PREC_BF16) return fail("tcgen05 path is the bf16 mode");
    if (d->state_dim < 1 || d->state_dim > 64) return fail("state_dim must be at most 64");
    if (d->obs_dim < 1 || d->obs_dim > 64) return fail("obs_dim must be at most 64");
    if (d->noise_dim < 1 || d->noise_dim > 32) return fail("noise_dim must be 1 .. 32");
    for (const voila_mlp *f : {&d->f_T, &d->f_Z}) {
        if (f->n_layers < 2) return fail("generator needs at least one hidden layer");
        for (int l = 1; l < f->n_layers; ++l)
            if (f->dims[l] > 512) return fail("hidden widths must be at most 512");
    }
    return true;
}

namespace {
// The state tower g fits the belief program when its hidden widths are MMA-block shaped and the
// embedding fits eight 16-column accumulator groups.
bool tower_fits_tc2(const voila_model_desc *d) {
    const voila_mlp &g = d->lik_state;
    if (g.n_layers < 2 || g.n_layers > 6) return false;
    if (g.dims[0] != d->state_dim + (d->lik_action_cond ? d->n_actions : 0)) return false;
    for (int l = 1; l < g.n_layers; ++l)
        if (g.dims[l] > 512) return false;
    return g.dims[g.n_layers] >= 1 && g.dims[g.n_layers] <= 128;
}
}  // namespace

void *tc2_create(const voila_model_desc *d, int sm_count, std::vector<void *> *allocs, std::string *err) {
    const int S = d->state_dim, A = d->n_actions, Nz = d->noise_dim;
    const int Sp = rup(S, 8), Nzp = rup(Nz, 8);  // operand widths of the state and the noise
    const bool aligned = Sp == S && Nzp == Nz;   // the per-row-action / denoiser programs want aligned widths
    const bool term = d->terminal && d->terminal->n_regions > 0;  // the rollout kernel instance with the alive-flag logic
    int policy = 0;
    if (const char *e = getenv("VOILA_T2_BLOCK_POLICY")) policy = atoi(e);  // tuning knob (0, 1, 2)
    T2Handle *h = new T2Handle();
    h->Sp = Sp;
    h->Nzp = Nzp;
    {
        Builder2 pb;
        pb.policy = policy;
        // The 640-thread kernel (two sets of epilogue warps sharing every hidden layer) is the default:
        // measured +11 % on CFG3, +7 % on CFG2, +2 % on CFG5 over the eight-warp kernel.
        {
            const char *e = getenv("VOILA_T2_ROLLOUT_WARPS");  // "8" | "16": override for A/B runs
            h->roll_x = e ? atoi(e) == 16 : true;
        }
        pb.par_split = h->roll_x;
        {
            int w = 0;
            for (const voila_mlp *f : {&d->f_T, &d->f_Z})
                for (int l = 1; l <= f->n_layers; ++l) w = std::max(w, rup(f->dims[l], 64));
            pb.pingpong = w <= 256 && !getenv("VOILA_T2_NO_PINGPONG");
            // wide generators: 32 KB ring stages, so a tile of a 256-column block holds two K chunks (8 MMAs,
            // ~1000 clk of tensor work per pass of the issuer loop instead of ~500; measured CFG5 +6.8 %, two
            // stages in flight).  Narrow / two-slot programs keep 16 KB stages (more stages in flight: measured
            // CFG3 753 vs 729 TFLOP/s, CFG4 propose+score 624 vs 645 us).
            if (w > 256 && !getenv("VOILA_T2_STAGE_ROWS")) pb.stage_rows = 256;
        }
        if (d->reward.kind == VOILA_R_NEG_QUADRATIC)  // u = M s on the tensor pipe, r = -s^T u in the epilogue
            pb.add_layer(d->reward.param, S, S, nullptr, 1, T2_EPI_REWARD, VOILA_ACT_NONE);
        add_generator2(pb, d->f_T, S, A, Nz, T2_EPI_STATE);
        add_generator2(pb, d->f_Z, S, A, Nz, T2_EPI_OBS);
        // 16 epilogue warps (two sets sharing every hidden layer) unless the 8-warp kernel is asked for
        const std::string m =
            h->roll_x ? (term ? finish_program(pb, h->roll, rollout_tc2x_kernel<1>, rup(Sp + Nzp, 64) / 64, sm_count, allocs, kT2ThreadsDual)
                              : finish_program(pb, h->roll, rollout_tc2x_kernel<0>, rup(Sp + Nzp, 64) / 64, sm_count, allocs, kT2ThreadsDual))
                      : (term ? finish_program(pb, h->roll, rollout_tc2_kernel<1>, rup(Sp + Nzp, 64) / 64, sm_count, allocs)
                              : finish_program(pb, h->roll, rollout_tc2_kernel<0>, rup(Sp + Nzp, 64) / 64, sm_count, allocs));
        if (!m.empty()) {
            if (err) *err = m;
            delete h;
            return nullptr;
        }
    }
    {
        // Two-slot rollout program (narrow generators): 4 operand chunks and 256 TMEM columns per slot,
        // shared weight tiles, the tile program alternating the slots layer by layer.
        int w = Sp + Nzp;
        for (const voila_mlp *f : {&d->f_T, &d->f_Z})
            for (int l = 1; l <= f->n_layers; ++l) w = std::max(w, rup(f->dims[l], l == f->n_layers ? 16 : 64));
        if (w <= 256 && !getenv("VOILA_T2_ROLLOUT_1SLOT")) {
            Builder2 pb;
            pb.policy = policy;
            pb.set_dual(4, 256);
            if (d->reward.kind == VOILA_R_NEG_QUADRATIC)
                pb.add_layer(d->reward.param, S, S, nullptr, 1, T2_EPI_REWARD, VOILA_ACT_NONE);
            add_generator2(pb, d->f_T, S, A, Nz, T2_EPI_STATE);
            add_generator2(pb, d->f_Z, S, A, Nz, T2_EPI_OBS);
            const std::string m =
                term ? finish_program(pb, h->roll_dual, rollout_tc2d_kernel<1>, rup(Sp + Nzp, 64) / 64, sm_count, allocs, kT2ThreadsDual)
                     : finish_program(pb, h->roll_dual, rollout_tc2d_kernel<0>, rup(Sp + Nzp, 64) / 64, sm_count, allocs, kT2ThreadsDual);
            h->has_roll_dual = m.empty();  // (the one-slot program serves if this one does not fit)
        }
    }
    if (tower_fits_tc2(d)) {
        // belief-update program: proposal s' = f_T(s, a, w), then the state tower g(s') and the score.
        // Narrow models (every layer <= 256 wide, every K <= 256) get a second, TWO-SLOT build: two
        // units in flight per CTA pair (4 operand chunks and 256 TMEM columns each), so that the
        // epilogue of one unit overlaps the MMAs of the other; used when there is more than one
        // unit per CTA pair (large N), while small N keeps the one-slot program (lower latency).
        int widest = Sp + Nzp;
        for (int l = 1; l <= d->f_T.n_layers; ++l) widest = std::max(widest, rup(d->f_T.dims[l], 64));
        for (int l = 0; l <= d->lik_state.n_layers; ++l) widest = std::max(widest, l == 0 ? Sp : rup(d->lik_state.dims[l], 64));
        const bool want_dual = widest <= 256 && !getenv("VOILA_T2_BELIEF_1SLOT");
        // pw = 1: the progressive-widening form (one-hot block in the operand; its layer-1 K is
        // S + Nz + A); only without an action-conditioned state tower
        for (int pw = 0; pw <= (d->lik_action_cond ? 0 : 1); ++pw) {
            const int in_cols = Sp + Nzp + (pw ? rup(A, 8) : 0);
            if (pw && (!aligned || A % 8 != 0 || in_cols > 512)) continue;
            const bool dual_ok = want_dual && rup(in_cols, 64) / 64 <= 4;
            for (int dual = 0; dual <= (dual_ok ? 1 : 0); ++dual) {
                Builder2 pb;
                pb.policy = policy;
                if (dual) {
                    pb.set_dual(4, 256);
                    pb.par_split = getenv("VOILA_T2_DUAL_SPLIT") != nullptr;  // measured slower (CFG4 676 vs 645 us): off
                }
                if (pw) add_generator2_dense(pb, d->f_T, S, A, Nz, T2_EPI_PROPOSAL);
                else add_generator2(pb, d->f_T, S, A, Nz, T2_EPI_PROPOSAL);
                const voila_mlp &g = d->lik_state;
                if (d->lik_action_cond) {
                    add_generator2(pb, g, S, A, 0, T2_EPI_SCORE);
                } else {
                    for (int l = 0; l < g.n_layers; ++l)
                        pb.add_layer(g.W[l], g.dims[l + 1], g.dims[l], g.b[l], 1,
                                     l == g.n_layers - 1 ? T2_EPI_SCORE : T2_EPI_HIDDEN, g.act);
                }
                T2Program &prog = pw ? (dual ? h->pw_dual : h->pw) : (dual ? h->belief_dual : h->belief);
                const int dd = g.dims[g.n_layers];
                prog.hdr.g_in_chunks = rup(Sp, 64) / 64;
                prog.hdr.e_pad = rup(dd, 16);
                prog.hdr.e_off = (int)pb.sbias_init.size();
                pb.sbias_init.resize(pb.sbias_init.size() + (size_t)prog.hdr.e_pad, 0.0f);
                const std::string m =
                    dual ? (pw ? finish_program(pb, prog, belief_tc2_dual_kernel<1>, rup(in_cols, 64) / 64, sm_count, allocs, kT2ThreadsDual)
                               : finish_program(pb, prog, belief_tc2_dual_kernel<0>, rup(in_cols, 64) / 64, sm_count, allocs, kT2ThreadsDual))
                         : (pw ? finish_program(pb, prog, belief_tc2_kernel<1>, rup(in_cols, 64) / 64, sm_count, allocs)
                               : finish_program(pb, prog, belief_tc2_kernel<0>, rup(in_cols, 64) / 64, sm_count, allocs));
                // without a one-slot program the CUDA-core kernels serve the call
                bool &flag = pw ? (dual ? h->has_pw_dual : h->has_pw) : (dual ? h->has_belief_dual : h->has_belief);
                flag = m.empty();
            }
        }
    }
    // progressive widening, the slot passes: (f_T -> f_Z) over the opened slots, tower f over the stored ones
    if (h->has_pw && d->obs_dim % 8 == 0 && d->lik_obs.dims[d->lik_obs.n_layers] % 16 == 0 &&
        d->lik_obs.dims[d->lik_obs.n_layers] <= 128) {
        bool ok = true;
        for (int l = 1; l < d->lik_obs.n_layers; ++l) ok = ok && d->lik_obs.dims[l] <= 512;
        std::string m1 = "x", m2 = "x";
        if (ok) {
            const int in_cols = Sp + Nzp + rup(A, 8);
            Builder2 pb;
            pb.policy = policy;
            add_generator2_dense(pb, d->f_T, S, A, Nz, T2_EPI_CHAIN);
            add_generator2_dense(pb, d->f_Z, S, A, Nz, T2_EPI_OBS_STORE);
            h->pw_open.hdr.e_off = (int)pb.sbias_init.size();
            m1 = finish_program(pb, h->pw_open, belief_tc2_kernel<3>, rup(in_cols, 64) / 64, sm_count, allocs);
            Builder2 pe;
            pe.policy = policy;
            const voila_mlp &f = d->lik_obs;
            for (int l = 0; l < f.n_layers; ++l)
                pe.add_layer(f.W[l], f.dims[l + 1], f.dims[l], f.b[l], 1,
                             l == f.n_layers - 1 ? T2_EPI_EMB_STORE : T2_EPI_HIDDEN, f.act);
            h->pw_emb.hdr.e_off = (int)pe.sbias_init.size();
            m2 = finish_program(pe, h->pw_emb, belief_tc2_kernel<4>, rup(d->obs_dim, 64) / 64, sm_count, allocs);
        }
        h->has_pw_slots = m1.empty() && m2.empty();
    }
    // diffusion teachers: one program per denoiser (one- and two-slot)
    for (int which = 0; which < 2; ++which) {
        const voila_mlp &f = which == 0 ? d->denoise_T : d->denoise_Z;
        const int D = which == 0 ? S : d->obs_dim;
        if (f.n_layers < 2 || f.n_layers > 8 || D % 8 != 0 || D > 64 || !aligned) continue;
        bool fits = S + D + rup(A, 8) <= 512;
        int widest = S + D + rup(A, 8);
        for (int l = 1; l < f.n_layers; ++l) {
            fits = fits && f.dims[l] % 64 == 0 && f.dims[l] <= 512;
            widest = std::max(widest, f.dims[l]);
        }
        if (!fits) continue;
        const int in_cols = S + D + rup(A, 8);
        for (int dual = 0; dual <= ((widest <= 256 && rup(in_cols, 64) / 64 <= 4) ? 1 : 0); ++dual) {
            Builder2 pb;
            pb.policy = policy;
            if (dual) {
                    pb.set_dual(4, 256);
                    pb.par_split = getenv("VOILA_T2_DUAL_SPLIT") != nullptr;  // measured slower (CFG4 676 vs 645 us): off
                }
            add_denoiser2(pb, f, S, A, D);
            T2Program &prog = h->diff[which][dual];
            prog.hdr.g_in_chunks = 0;
            prog.hdr.e_pad = 0;
            prog.hdr.e_off = (int)pb.sbias_init.size();
            const std::string m =
                dual ? finish_program(pb, prog, belief_tc2_dual_kernel<2>, rup(in_cols, 64) / 64, sm_count, allocs, kT2ThreadsDual)
                     : finish_program(pb, prog, belief_tc2_kernel<2>, rup(in_cols, 64) / 64, sm_count, allocs);
            h->has_diff[which][dual] = m.empty();
        }
        if (h->has_diff[which][0]) {
            const int N1 = f.dims[1], K = f.dims[0];
            std::vector<float> b1(f.b[0], f.b[0] + N1), w1t((size_t)N1 * kTemb);
            for (int j = 0; j < N1; ++j)
                for (int e = 0; e < kTemb; ++e) w1t[(size_t)j * kTemb + e] = h_bf16_round(f.W[0][(size_t)j * K + S + A + D + e]);
            void *p1 = nullptr, *p2 = nullptr;
            if (cudaMalloc(&p1, b1.size() * 4) == cudaSuccess && cudaMalloc(&p2, w1t.size() * 4) == cudaSuccess) {
                allocs->push_back(p1);
                allocs->push_back(p2);
                cudaMemcpy(p1, b1.data(), b1.size() * 4, cudaMemcpyHostToDevice);
                cudaMemcpy(p2, w1t.data(), w1t.size() * 4, cudaMemcpyHostToDevice);
                h->d_diff_b1[which] = reinterpret_cast<float *>(p1);
                h->d_diff_w1t[which] = reinterpret_cast<float *>(p2);
                h->diff_n1[which] = N1;
                h->diff_scale[which] = f.act == VOILA_ACT_SILU ? 0.5f : 1.0f;  // SiLU layers carry pre-halved biases
            } else {
                h->has_diff[which][0] = h->has_diff[which][1] = false;
            }
        }
    }
    return h;
}

void tc2_destroy(void *tc) { delete reinterpret_cast<T2Handle *>(tc); }

bool tc2_has_belief(const void *tc) { return tc && reinterpret_cast<const T2Handle *>(tc)->has_belief; }
bool tc2_has_diffusion(const void *tc, int which) {
    return tc && reinterpret_cast<const T2Handle *>(tc)->has_diff[which][0];
}
bool tc2_has_pw_slots(const void *tc) { return tc && reinterpret_cast<const T2Handle *>(tc)->has_pw_slots; }
bool tc2_has_pw(const void *tc) { return tc && reinterpret_cast<const T2Handle *>(tc)->has_pw; }
int tc2_pw_e_stride(const void *tc) { return reinterpret_cast<const T2Handle *>(tc)->pw.hdr.e_pad; }

namespace {
T2Params base_params(const T2Program &g, const ModelDev &m) {
    T2Params p{};
    p.bias = reinterpret_cast<const float *>(g.d_bias);
    p.sbias_init = reinterpret_cast<const float *>(g.d_sbias);
    p.layers = reinterpret_cast<const T2Layer *>(g.d_layers);
    p.tiles = reinterpret_cast<const T2TileDev *>(g.d_tiles);
    p.hdr = g.hdr;
    p.S = rup(m.S, 8); p.O = m.O; p.A = m.A; p.Nz = rup(m.Nz, 8);
    p.S_io = m.S;
    p.gamma = m.gamma;
    p.reward_kind = m.reward.kind;
    p.reward_param = m.reward.param;
    p.action_cost = m.reward.action_cost;
    p.term = m.term;
    return p;
}
}  // namespace

cudaError_t launch_rollout_tc2(void *tc, const ModelDev &m, const RolloutArgs &a, cudaStream_t st,
                               std::string *kernel_name, int *n_launches) {
    const T2Handle *h = reinterpret_cast<const T2Handle *>(tc);
    // two blocks in flight per CTA pair: when a sequence has an even number of 256-particle blocks (no
    // idle slot) or at least five, and every CTA pair gets more than one pair of blocks
    const int blocks = (a.P + 2 * kT2Rows - 1) / (2 * kT2Rows);
    // (an odd block count leaves the second slot of a sequence's last pair empty -- its rows are invalid --:
    //  worth it from five blocks on, 1.27 x 5 / 6 against the one-block kernel)
    const int pairs = (blocks + 1) / 2;
    const bool dual = h->has_roll_dual && (blocks % 2 == 0 || blocks >= 5) && pairs * a.Q > h->roll_dual.max_clusters;
    const T2Program &g = dual ? h->roll_dual : h->roll;
    T2Params p = base_params(g, m);
    p.particles = reinterpret_cast<const uint16_t *>(a.particles);
    p.seqs = a.action_seqs;
    p.weights = a.weights;
    p.P = a.P; p.Q = a.Q; p.H = a.H;
    p.seed = a.seed;
    p.part_value = a.part_value;
    p.part_witness = a.part_witness;
    p.returns_out = a.returns_out;
    p.final_states_out = a.final_states_out;
    p.blocks_per_q = dual ? pairs : blocks;  // work units of a CTA pair per sequence
    p.tiles_per_q = a.tiles;  // = 2 * blocks (see rollout_tile_count)
    p.n_units = p.blocks_per_q * a.Q;
    const int clusters = std::min(g.max_clusters, p.n_units);
    const bool term = m.term.n > 0;
    if (dual) {
        if (term) rollout_tc2d_kernel<1><<<2 * clusters, kT2ThreadsDual, g.smem_bytes, st>>>(p, g.wmap);
        else rollout_tc2d_kernel<0><<<2 * clusters, kT2ThreadsDual, g.smem_bytes, st>>>(p, g.wmap);
        if (kernel_name) *kernel_name = "rollout_tc2d_kernel<tcgen05 cta_group::2 bf16, two blocks in flight>";
        if (n_launches) *n_launches = 1;
        return cudaGetLastError();
    }
    if (h->roll_x) {
        if (term) rollout_tc2x_kernel<1><<<2 * clusters, kT2ThreadsDual, g.smem_bytes, st>>>(p, g.wmap);
        else rollout_tc2x_kernel<0><<<2 * clusters, kT2ThreadsDual, g.smem_bytes, st>>>(p, g.wmap);
    } else {
        if (term) rollout_tc2_kernel<1><<<2 * clusters, kT2Threads, g.smem_bytes, st>>>(p, g.wmap);
        else rollout_tc2_kernel<0><<<2 * clusters, kT2Threads, g.smem_bytes, st>>>(p, g.wmap);
    }
    if (kernel_name)
        *kernel_name = h->roll_x ? "rollout_tc2x_kernel<tcgen05 cta_group::2 bf16, 16 epilogue warps>"
                                 : "rollout_tc2_kernel<tcgen05 cta_group::2 bf16>";
    if (n_launches) *n_launches = 1;
    return cudaGetLastError();
}

// Belief update, propose + score on the CTA-pair tcgen05 program.
// part_wsum gets one entry per 32 particles.
cudaError_t launch_bu_propose_score_tc2(void *tc, const ModelDev &m, const BeliefArgs &a, cudaStream_t st,
                                        int *n_launches, std::string *kernel_name) {
    const T2Handle *h = reinterpret_cast<const T2Handle *>(tc);
    // two units in flight per CTA pair pay off once a pair has more than one unit to process
    const bool dual = h->has_belief_dual && a.N > 2 * kT2Rows * h->belief.max_clusters;
    const T2Program &g = dual ? h->belief_dual : h->belief;
    T2Params p = base_params(g, m);
    p.particles = reinterpret_cast<const uint16_t *>(a.particles);
    p.weights = a.weights;
    p.P = a.N; p.Q = 1; p.H = 1;
    p.seed = a.seed;
    const int unit_rows = 2 * kT2Rows * g.hdr.n_slots;  // particles per work unit of a CTA pair
    p.n_units = (a.N + unit_rows - 1) / unit_rows;
    p.bu_action = a.action;
    p.bu_e = a.e;
    p.bu_proposals = reinterpret_cast<uint16_t *>(a.proposals);
    p.bu_logits = a.logits;
    p.bu_max_ordered = a.max_ordered;
    p.bu_part_wsum = a.part_wsum;
    p.inv_lambda = 1.0f / m.lambda;
    p.d = m.mlp[3].dims[m.mlp[3].n_layers];
    const int clusters = std::min(g.max_clusters, p.n_units);
    // programmatic dependent launch: may start while the observation-tower kernel in front of it still runs
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)(2 * clusters));
    cfg.blockDim = dim3((unsigned)(dual ? kT2ThreadsDual : kT2Threads));
    cfg.dynamicSmemBytes = g.smem_bytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const cudaError_t le = dual ? cudaLaunchKernelEx(&cfg, belief_tc2_dual_kernel<0>, p, g.wmap)
                                : cudaLaunchKernelEx(&cfg, belief_tc2_kernel<0>, p, g.wmap);
    if (le != cudaSuccess) return le;
    if (kernel_name)
        *kernel_name = dual ? "belief_tc2_dual_kernel<tcgen05 cta_group::2 bf16, two units in flight>"
                            : "belief_tc2_kernel<tcgen05 cta_group::2 bf16>";
    if (n_launches) *n_launches = 1;
    return cudaGetLastError();
}

// Progressive widening, propose + score of every simulation (voila_pw_update) on the CTA-pair tcgen05
// program: per-row actions (one-hot block in the operand), per-row tower embeddings, child maxima.
cudaError_t launch_pw_propose_score_tc2(void *tc, const ModelDev &m, const PwArgs &a, const int32_t *sim_action,
                                        const int32_t *sim_seg, cudaStream_t st, std::string *kernel_name) {
    const T2Handle *h = reinterpret_cast<const T2Handle *>(tc);
    const bool dual = h->has_pw_dual && a.N > 2 * kT2Rows * h->pw.max_clusters;
    const T2Program &g = dual ? h->pw_dual : h->pw;
    T2Params p = base_params(g, m);
    p.particles = reinterpret_cast<const uint16_t *>(a.particles);
    p.weights = a.weights;
    p.P = a.N; p.Q = 1; p.H = 1;
    p.seed = a.seed;
    const int unit_rows = 2 * kT2Rows * g.hdr.n_slots;
    p.n_units = (a.N + unit_rows - 1) / unit_rows;
    p.bu_action = 0;
    p.bu_e = nullptr;
    p.bu_proposals = reinterpret_cast<uint16_t *>(a.proposals);
    p.bu_logits = a.logits;
    p.bu_max_ordered = nullptr;
    p.bu_part_wsum = nullptr;
    p.inv_lambda = 1.0f / m.lambda;
    p.d = m.mlp[3].dims[m.mlp[3].n_layers];
    p.pw_sim_action = sim_action;
    p.pw_sim_seg = sim_seg;
    p.pw_E = a.E;
    p.pw_seg_max = a.seg_max;
    const int clusters = std::min(g.max_clusters, p.n_units);
    if (dual) belief_tc2_dual_kernel<1><<<2 * clusters, kT2ThreadsDual, g.smem_bytes, st>>>(p, g.wmap);
    else belief_tc2_kernel<1><<<2 * clusters, kT2Threads, g.smem_bytes, st>>>(p, g.wmap);
    if (kernel_name)
        *kernel_name = dual ? "belief_tc2_dual_kernel<tcgen05 cta_group::2 bf16, two units in flight, per-row actions>"
                            : "belief_tc2_kernel<tcgen05 cta_group::2 bf16, per-row actions>";
    return cudaGetLastError();
}

// Progressive widening, the two small passes over the (action node, branch) slots on the tensor cores:
// sampled observations of the slots opened in this call, then the tower f over every stored branch.
cudaError_t launch_pw_slots_tc2(void *tc, const ModelDev &m, const PwArgs &a, cudaStream_t st) {
    const T2Handle *h = reinterpret_cast<const T2Handle *>(tc);
    const int slots = a.G * a.M_max;
    for (int pass = 0; pass < 2; ++pass) {
        const T2Program &g = pass == 0 ? h->pw_open : h->pw_emb;
        T2Params p = base_params(g, m);
        p.particles = reinterpret_cast<const uint16_t *>(a.particles);
        p.P = slots; p.Q = 1; p.H = 1;
        p.seed = a.seed;
        p.n_units = (slots + 2 * kT2Rows - 1) / (2 * kT2Rows);
        p.d = m.mlp[3].dims[m.mlp[3].n_layers];
        p.slot_src = a.new_src;
        p.slot_action = a.group_action;
        p.slot_count = a.branch_count;
        p.slot_obs = a.branch_obs;
        p.slot_emb = a.E;
        p.slot_M = a.M_max;
        const int clusters = std::min(g.max_clusters, p.n_units);
        if (pass == 0) belief_tc2_kernel<3><<<2 * clusters, kT2Threads, g.smem_bytes, st>>>(p, g.wmap);
        else belief_tc2_kernel<4><<<2 * clusters, kT2Threads, g.smem_bytes, st>>>(p, g.wmap);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// One DDIM-ODE step of a diffusion teacher on the CTA-pair tcgen05 program (2 launches: the step's
// bias row with the time embedding folded in, then the denoiser + update over all samples).
cudaError_t launch_diffusion_step_tc2(void *tc, const ModelDev &m, const DiffusionArgs &a, int k, cudaStream_t st,
                                      std::string *kernel_name) {
    const T2Handle *h = reinterpret_cast<const T2Handle *>(tc);
    const int w = a.which;
    const bool dual = h->has_diff[w][1] && a.N > 2 * kT2Rows * h->diff[w][0].max_clusters;
    const T2Program &g = h->diff[w][dual ? 1 : 0];
    // layer 1 is the program's first layer record: its per-step bias rows start at offset 0 of the
    // program's bias buffer; hidden widths are multiples of 64, so n_pad = N1
    const int n_pad = h->diff_n1[w];
    float *row = reinterpret_cast<float *>(g.d_bias) + (size_t)k * n_pad;
    TembArg t;
    for (int e = 0; e < kTemb; ++e) t.v[e] = a.temb[e];
    diffusion_bias_kernel<<<(n_pad + 127) / 128, 128, 0, st>>>(row, h->d_diff_b1[w], h->d_diff_w1t[w], h->diff_n1[w], n_pad,
                                                               h->diff_scale[w], t);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    T2Params p = base_params(g, m);
    p.particles = reinterpret_cast<const uint16_t *>(a.cond);
    p.weights = nullptr;
    p.P = a.N; p.Q = 1; p.H = 1;
    p.seed = a.seed;
    const int unit_rows = 2 * kT2Rows * g.hdr.n_slots;
    p.n_units = (a.N + unit_rows - 1) / unit_rows;
    p.bu_action = k;  // the step's bias row
    p.pw_sim_action = a.actions;
    p.diff_x = a.x;
    p.diff_D = a.D;
    p.diff_first = a.first;
    p.al = a.al; p.si = a.si; p.al_n = a.al_n; p.si_n = a.si_n;
    const int clusters = std::min(g.max_clusters, p.n_units);
    if (dual) belief_tc2_dual_kernel<2><<<2 * clusters, kT2ThreadsDual, g.smem_bytes, st>>>(p, g.wmap);
    else belief_tc2_kernel<2><<<2 * clusters, kT2Threads, g.smem_bytes, st>>>(p, g.wmap);
    if (kernel_name)
        *kernel_name = dual ? "belief_tc2_dual_kernel<tcgen05 cta_group::2 bf16, two units in flight, denoiser + DDIM step>"
                            : "belief_tc2_kernel<tcgen05 cta_group::2 bf16, denoiser + DDIM step>";
    return cudaGetLastError();
}

}  // namespace voila

#ifdef VOILA_T2_TRACE
extern "C" __attribute__((visibility("default"))) int voila_debug_t2_trace(unsigned long long *out64) {
    return (int)cudaMemcpyFromSymbol(out64, voila::g_t2_trace, sizeof(unsigned long long) * 64);
}
// Timeline: sets the recorded step window and clears the buffer / reads it back (returns the count).
extern "C" __attribute__((visibility("default"))) int voila_debug_t2_timeline_arm(int step0, int step1) {
    const int win[2] = {step0, step1};
    const unsigned zero = 0;
    cudaMemcpyToSymbol(voila::g_t2_tl_win, win, sizeof(win));
    void *p = nullptr;
    cudaGetSymbolAddress(&p, voila::g_t2_tl);
    cudaMemset(p, 0, sizeof(unsigned long long) * 2 * voila::kT2TlCap);
    return (int)cudaMemcpyToSymbol(voila::g_t2_tl_n, &zero, sizeof(zero));
}
extern "C" __attribute__((visibility("default"))) int voila_debug_t2_timeline_read(unsigned long long *out, int cap_pairs) {
    // regions are zero-filled by arm(); unused entries stay (0, 0)
    unsigned n = voila::kT2TlCap;
    if ((int)n > cap_pairs) n = (unsigned)cap_pairs;
    cudaMemcpyFromSymbol(out, voila::g_t2_tl, sizeof(unsigned long long) * 2 * n);
    return (int)n;
}
#endif
