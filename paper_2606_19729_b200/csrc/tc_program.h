// tc_program.h -- the static "program" the tcgen05 kernels execute: a per-step list of layers and a
// per-step list of weight tiles in issue order, built once per model on the host (rollout_tc.cu).
//
// One CTA owns a tile of 128 rows (particles of ONE action sequence / of the belief).  Activations
// live in ONE shared-memory operand buffer that every layer rewrites IN PLACE (chunk j = columns
// [64j, 64j+64) of the 128-row operand, 16 KB, canonical 128-byte-swizzle K-major layout) and the
// accumulator of the running layer lives in TMEM columns [0, N).  Weight tiles (BN output neurons x
// 64 inputs, pre-swizzled on the host) stream from L2 through a ring of 16 KB stages.
//
// Because operand and accumulator are rewritten in place, a weight tile (layer l+1, block n,
// K-chunk k) may be issued as soon as the epilogue of layer l has (a) written operand chunk k and
// (b) drained the accumulator columns block n will overwrite.  The epilogue publishes its progress
// as a sequence of numbered EVENTS (one per 64-column chunk); every tile carries the index of the
// event it needs (`need`, relative to the step's first event; -1 = last event of the previous
// step) and tiles are issued in order of need.  That lets the tensor pipe work on the lower
// triangle of layer l+1 while the epilogue of layer l is still running.
#pragma once
#include <stdint.h>

namespace voila {

constexpr int kTcRows = 128;          // rows per CTA tile (UMMA M)
constexpr int kTcChunkCols = 64;      // K chunk: 64 bf16 = 128 bytes (one swizzle row)
constexpr int kTcChunkBytes = kTcRows * 128;  // 16 KB
constexpr int kTcStageBytes = 128 * 128;      // ring stage: up to 128 neurons x 64 inputs
constexpr int kTcMaxLayers = 24;
constexpr int kTcMaxTiles = 512;
constexpr int kTcEvtRing = 32;
constexpr int kTcThreads = 384;       // warps 0-3: producer / MMA / TMEM alloc / spare; 4-11 epilogue

enum TcEpi : int {
    TC_EPI_HIDDEN = 0,   // y = act(D + bias) -> bf16 -> operand chunks (in place)
    TC_EPI_REWARD = 1,   // rollout: u = M s; r = -s^T u (quadratic reward on the tensor pipe)
    TC_EPI_STATE = 2,    // rollout: s' = D + bias (f_T output); next operand = [s' ; w_Z]
    TC_EPI_OBS = 3,      // rollout: o = D + bias (f_Z output) -> witness; next operand = [s' ; w_T]
    TC_EPI_PROPOSAL = 4, // belief: s' = D + bias -> proposals; next operand = [s']
    TC_EPI_SCORE = 5     // belief: l = <e, D + bias> -> logits, running max
};

struct TcLayer {
    uint32_t idesc;      // tcgen05 instruction descriptor (M = 128, N = bn)
    uint32_t bias_off;   // float offset into the bias buffer
    uint16_t n_pad;      // padded output width
    uint16_t bn;         // accumulator block width of one weight tile
    uint16_t kc;         // number of 64-wide K chunks of the input operand
    uint8_t epi;         // TcEpi
    uint8_t act;         // voila_act of a hidden layer
    uint8_t bias_per_action;  // bias row = action (one-hot block folded into the bias)
    uint8_t pad[3];
};

struct TcTile {
    uint32_t src_off;    // byte offset of the packed tile in the weight stream
    uint32_t bytes;      // bn * 128
    int16_t need;        // event this tile waits for, relative to the step's first event
    uint8_t layer;
    uint8_t n;           // accumulator block
    uint8_t kc;          // operand chunk
    uint8_t first;       // first tile of its accumulator block (accumulate = 0)
    uint8_t last;        // last tile of its layer (commit -> layer_done)
    uint8_t pad;
};

struct TcProgramHeader {
    int n_layers, n_tiles, evt_per_step, a_chunks;  // a_chunks: operand buffer size in chunks
    int tmem_cols, n_stages, in_chunks, reserved;   // in_chunks: chunks of the step's input operand
};

}  // namespace voila
