// tc2_program.h -- the static program of the CTA-PAIR tcgen05 kernels (rollout_tc2.cu).
//
// Two CTAs of a cluster (two SMs of one TPC) own 256 rows (particles of ONE action sequence / of
// the belief), 128 each.  Every tcgen05.mma is issued with cta_group::2 by the leader CTA: M = 256,
// each CTA supplies its own 128 operand rows and HALF of the weight tile's output neurons, and
// receives its 128 accumulator rows x N columns in its own TMEM.  Per CTA that halves both the
// weight bytes streamed from L2 and the shared-memory operand reads per flop.
//
// As in tc_program.h the activations live in ONE operand buffer per CTA that every layer's
// epilogue rewrites in place (64-column chunks, 16 KB, 128-byte-swizzle K-major) and the running
// layer's accumulator lives in TMEM columns [0, N).  A weight tile may be issued once the epilogues
// of BOTH CTAs have written the operand chunks it reads and drained the accumulator block it
// overwrites; progress is published as numbered events on the leader's mbarriers (16 arrivals: 8
// epilogue warps x 2 CTAs).  Accumulator blocks are handed to the epilogues one by one
// (`layer_done` ring, multicast tcgen05.commit), so the epilogue of block n overlaps the MMAs of
// block n+1.  Because the operand buffer is rewritten in place, the epilogue of an earlier block
// may store output chunk c only after the LAST block's tile that reads operand chunk c has
// retired: those tiles commit "operand chunk free" signals (`cfree` ring) in chunk order.
//
// Two refinements share this program format:
//  * two SETS of epilogue warps (640-thread kernels): the second set takes the odd chunks of every
//    hidden layer.  A set publishes its events in order, the sets are not ordered with respect to
//    each other, so a tile names two events to wait for (T2Tile::need / need2);
//  * two SLOTS (belief update of narrow models): two independent 256-row units in flight per CTA
//    pair, each with its own operand chunks and TMEM columns (T2Layer::slot / chunk_off / col_off),
//    the program alternating the slots layer by layer, one set of epilogue warps per slot.
#pragma once
#include <stdint.h>

namespace voila {

constexpr int kT2Rows = 128;              // rows per CTA (256 per pair)
constexpr int kT2ChunkBytes = 128 * 128;  // one 64-column operand chunk
constexpr int kT2StageBytes = 128 * 128;  // smallest weight ring stage per CTA (TMA box: 128 rows x 128 B);
                                          // a program's stage is T2Header::stage_rows x 128 B (128 | 256 rows)
constexpr int kT2MaxLayers = 24;
constexpr int kT2MaxTiles = 512;
constexpr int kT2EvtRing = 32;
constexpr int kT2AccRing = 8;
constexpr int kT2FreeRing = 8;
constexpr int kT2Threads = 384;  // warp 0 producer, 1 MMA issuer (leader), 2 TMEM, 3 spare, 4-11 epilogue

enum T2Epi : int {
    T2_EPI_HIDDEN = 0,    // y = act(D + bias) -> bf16 -> operand chunks (in place)
    T2_EPI_REWARD = 1,    // rollout: u = M s ; r = -s^T u
    T2_EPI_STATE = 2,     // rollout: s' = D + bias ; next operand = [s' ; w_Z]
    T2_EPI_OBS = 3,       // rollout: o = D + bias -> witness ; next operand = [s' ; w_T]
    T2_EPI_PROPOSAL = 4,  // belief: s' = D + bias -> proposals (HBM) ; next operand = [s']
    T2_EPI_SCORE = 5,     // belief: logit = <e, D + bias>/lambda + log w -> logits, running max
    T2_EPI_DIFFUSE = 6,   // diffusion teacher: v = D + bias ; x <- DDIM-ODE step(x, v) (fp32 state in HBM)
    T2_EPI_CHAIN = 7,     // progressive widening, opened branches: s' = D + bias ; next operand = [s' ; w_Z ; onehot(a)]
    T2_EPI_OBS_STORE = 8, // ... o = D + bias -> the branch's stored observation (fp32, HBM)
    T2_EPI_EMB_STORE = 9  // tower f over stored observations: e = D + bias -> embedding table (fp32, HBM)
};

struct T2Layer {  // what the epilogue needs to know about a layer
    uint32_t bias_off;   // float offset into the global bias buffer (per-action layers: A rows)
    uint32_t sbias_off;  // float offset into the shared-memory bias table (per-action layers: 2 rows)
    uint16_t n_pad;     // padded output width
    uint8_t free_nk;    // K chunks per tile of the layer's LAST accumulator block (see wait_chunks)
    uint8_t wait_chunks;  // output chunks [0, wait_chunks) belong to earlier blocks and overwrite operand
                          // chunks the last block's MMAs still read: chunk c may be stored once
                          // c / free_nk + 1 "operand chunk free" signals of this layer have arrived
    uint8_t epi;        // T2Epi
    uint8_t act;        // voila_act of a hidden layer
    uint8_t bias_per_action;
    uint8_t blk_mask;   // hidden layers: bit c set = 64-column chunk c is the first of an accumulator block
    // Two-slot programs (belief update of narrow models): two independent 256-row units are in
    // flight per CTA pair, each with its own operand chunks and TMEM columns, so the epilogue of
    // one unit overlaps the MMAs of the other.  A layer record belongs to one slot.
    uint8_t slot;        // 0 | 1
    uint8_t chunk_off;   // first operand chunk of the slot
    uint16_t col_off;    // first TMEM column of the slot
    // Hidden layer of a two-slot program with ONE accumulator block: every tile of the next layer waits for
    // the layer's last chunk anyway (the block must be drained), so the epilogue publishes one event for
    // the whole layer instead of one per 64-column chunk (a proxy fence + a cluster arrive each).
    uint8_t one_event;
    uint8_t pad[3];
};
static_assert(sizeof(T2Layer) == 24, "T2Layer is copied to shared memory as 32-bit words");

struct T2Tile {  // one weight-ring stage: nk K-chunks of one accumulator block (20 bytes)
    uint32_t src_row;  // first 128-byte row of the tile in the weight stream (CTA r: + r * rows)
    uint32_t idesc;    // tcgen05 instruction descriptor (M = 256, N = bn)
    uint8_t d_col16;   // first accumulator column of the block / 16
    uint8_t blk;       // index of the accumulator block among the step's blocks (epilogue order)
    int16_t need;      // event the tile waits for, relative to the step's first event
    uint8_t kc0;       // first operand chunk
    uint8_t nk;        // number of 64-wide K chunks held by the stage
    uint8_t rows8;     // weight rows per CTA per chunk / 8 (= bn / 16)
    uint8_t flags;     // bit 0: first tile of its block (overwrite); bit 1: last tile of its block;
                       // bit 2: commit an "operand chunk free" signal after this tile
    // Events are published in order by each SET of epilogue warps, not across sets (the 640-thread
    // rollout kernel has two sets sharing every hidden layer: even chunks / odd chunks).  "Every
    // event <= need has happened" therefore takes two waits: `need` (set `need_set`) and `need2`,
    // the latest earlier event of the OTHER set (= need when there is one set only).
    int16_t need2;
    uint8_t need_set;  // 0 | 1: the set that publishes event `need`
    uint8_t pad;       // host scratch: the tile's slot in a two-slot program
};
static_assert(sizeof(T2Tile) == 20, "T2Tile is copied to shared memory as 32-bit words");

// The tile record as the device reads it (32 bytes = two 16-byte shared-memory loads, every field
// a ready-to-use 32-bit word: the MMA issuer's loop is a dependent chain that shares its scheduler
// with four epilogue warps, and ncu showed a quarter of its time in the byte / halfword loads and
// unpacking of the 20-byte host record).
struct T2TileDev {
    uint32_t src_row;   // producer: first 128-byte row of the tile in the weight stream
    uint32_t idesc;     // tcgen05 instruction descriptor
    uint32_t a_off;     // operand descriptor offset of the first K chunk (16-byte units)
    uint32_t d_off;     // accumulator column offset in TMEM
    int32_t need_s0;    // event of epilogue set 0 to wait for (relative to the step), -100000: none
    int32_t need_s1;    // event of epilogue set 1 to wait for, -100000: none
    uint32_t chunk_b16; // weight bytes of one K chunk in the stage / 16 (descriptor units)
    uint32_t misc;      // nk | flags << 4 | blk << 8 | rows << 16   (rows = weight rows per CTA in the stage)
};
static_assert(sizeof(T2TileDev) == 32, "T2TileDev is read with two 16-byte loads");

struct T2Header {
    int n_layers, n_tiles, evt_per_step, a_chunks;
    int tmem_cols, n_stages, in_chunks, blocks_per_step;  // accumulator blocks (hand-offs) per step
    int sbias_floats;     // size of the shared-memory bias table
    int pa_layer[2];      // layers whose bias row depends on the action (-1: none)
    int init_events;      // events published before the first step (one per slot)
    int n_slots;          // 1 | 2 units in flight per CTA pair (see T2Layer::slot)
    int slot_chunks;      // operand chunks per slot
    int g_in_chunks;      // belief program: operand chunks of the state tower's input
    int e_off, e_pad;     // belief program: f(o) in the shared-memory table (float offset, padded length)
    int split_hidden;     // two-slot programs: 1 = both sets of epilogue warps share EVERY hidden layer of both
                          // slots (even / odd chunks), a slot's other layers go to the set of its number;
                          // 0 = one set per slot
    int stage_rows;       // weight rows (128 bytes each) per CTA per ring stage = rows of the TMA box: 128 | 256
};

}  // namespace voila
