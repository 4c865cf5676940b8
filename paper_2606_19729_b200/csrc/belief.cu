// belief.cu -- weight normalisation, prefix sum and systematic resampling of the SIR belief update
// (O5-O7; PAPER.md:77 "before resampling", :128 only relative weights matter, :137).
//
//   weight_scan    v_i = exp(L_i - m) (max-shifted), q_i = floor(v_i 2^32) as
//                  uint64, inclusive scan C_i in ONE pass: warp shuffles inside a 4096-element tile,
//                  block-wide decoupled look-back across tiles (512 predecessors per round).  Integer addition is associative, so the CDF is
//                  independent of tiling and the resampled indices are bit-exact (reading R6).
//   bu_finalize    W = C_{N-1}, comb offset U = (x0 W) >> 32 from one Philox word, log evidence,
//                  degenerate-weight status.
//   resample_gather  i_k = min{ i : N C_i > k W + U } with 128-bit compares: ancestors are
//                  non-decreasing in k, so a CTA brackets its 256 outputs with two searches of the
//                  L2-resident CDF, stages that CDF segment in shared memory and searches there;
//                  then coalesced vectorised row gathers.
// HBM-bound; no tensor-core work here.
#include "voila_device.cuh"
#include <atomic>

#include "voila_kernels.h"

namespace voila {

namespace {

typedef unsigned long long u64;
constexpr int kScanThreads = 512;
constexpr int kItems = kScanTile / kScanThreads;  // 8
constexpr unsigned kFlagEmpty = 0u, kFlagAggregate = 1u, kFlagInclusive = 2u;

__global__ void bu_init_kernel(ScanBuffers sb, int tiles) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < tiles) sb.tile_flag[i] = kFlagEmpty;
    if (i == 0) {
        ScanState z;
        z.total_q = 0; z.offset_u = 0; z.sum_v = 0.0; z.sum_w = 0.0;
        z.max_logit = 0.0f; z.status = 0; z.tile_counter = 0; z.done_counter = 0; z.resample = 1; z.ess = 0.0; z.inv_sum_v = 0.0;
        *sb.state = z;
        *sb.max_ordered = (int)0x80000000;
    }
}

// bu_init + the observation tower e = f(o) for ONE observation:
// a chain of GEMVs, so one CTA; the K range of every layer is split over kObsThreads / N thread
// groups (coalesced reads of the k-major weights, independent loads), partial sums meet in shared
// memory.  bf16 mode rounds the operands like every other kernel of the library.
constexpr int kObsThreads = 1024;
constexpr int kObsMaxWidth = 1024;
template <bool EMU>
__global__ void __launch_bounds__(kObsThreads) bu_init_obs_kernel(ScanBuffers sb, int tiles, MlpDev f,
                                                                  const float *__restrict__ obs, float *e_out) {
    __shared__ float xs[2][kObsMaxWidth];
    __shared__ float part[kObsThreads];
    const int tid = threadIdx.x;
    // programmatic dependent launch: the propose+score kernel may start now (its proposal layers need
    // nothing from here); it waits (griddepcontrol.wait) before it reads e or touches the running maximum
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    for (int i = tid; i < tiles; i += kObsThreads) sb.tile_flag[i] = kFlagEmpty;
    if (tid == 0) {
        ScanState z;
        z.total_q = 0; z.offset_u = 0; z.sum_v = 0.0; z.sum_w = 0.0;
        z.max_logit = 0.0f; z.status = 0; z.tile_counter = 0; z.done_counter = 0; z.resample = 1; z.ess = 0.0; z.inv_sum_v = 0.0;
        *sb.state = z;
        *sb.max_ordered = (int)0x80000000;
    }
    // pull every layer's weights towards L2 now: the layers below then pay L2, not HBM, latency
    for (int l = 0; l < f.n_layers; ++l) {
        const size_t lines = ((size_t)f.dims[l] * f.dims[l + 1] * sizeof(float) + 127) / 128;
        const char *w = reinterpret_cast<const char *>(f.Wt[l]);
        for (size_t i = tid; i < lines; i += kObsThreads) asm volatile("prefetch.global.L2 [%0];" ::"l"(w + i * 128));
    }
    for (int k = tid; k < f.dims[0]; k += kObsThreads) xs[0][k] = EMU ? bf16_round(obs[k]) : obs[k];
    __syncthreads();
    int cur = 0;
    for (int l = 0; l < f.n_layers; ++l) {
        const int K = f.dims[l], N = f.dims[l + 1];
        const bool last = l == f.n_layers - 1;
        // G groups of N threads; group g sums k = g, g + G, ...
        int G = kObsThreads / N;
        if (G < 1) G = 1;
        if (G > K) G = K;
        const float *__restrict__ Wt = f.Wt[l];
        for (int j0 = 0; j0 < N; j0 += kObsThreads) {  // one pass unless N > kObsThreads
            const int g = tid / N, j = j0 + tid - g * N;
            float acc = 0.0f;
            if (g < G && j < N) {
                // batches of 8 predicated loads in flight (a plain unrolled loop serialises them
                // behind its exit tests)
                const int per = (K + G - 1) / G;
                for (int kk = 0; kk < per; kk += 8) {
                    float w[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int k = g + (kk + u) * G;
                        w[u] = k < K ? __ldg(Wt + (size_t)k * N + j) : 0.0f;
                    }
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int k = g + (kk + u) * G;
                        acc = fmaf(w[u], k < K ? xs[cur][k] : 0.0f, acc);
                    }
                }
            }
            part[tid] = acc;
            __syncthreads();
            if (tid < N - j0 && tid < kObsThreads) {
                const int jj = j0 + tid;
                float t = 0.0f;
                for (int gg = 0; gg < G; ++gg) t += part[gg * N + tid];
                t += __ldg(f.b[l] + jj);
                if (!last) {
                    t = act_apply(t, f.act);
                    if (EMU) t = bf16_round(t);
                    xs[cur ^ 1][jj] = t;
                } else {
                    e_out[jj] = t;
                }
            }
            __syncthreads();
        }
        cur ^= 1;
    }
}

__device__ __forceinline__ unsigned ld_flag(const unsigned *p) {  // acquire: orders the value load after it
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_flag(unsigned *p, unsigned v) {  // release: the value store is visible first
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ u64 ld_u64_volatile(const u64 *p) {
    return *reinterpret_cast<const volatile u64 *>(p);
}

// q = floor(v * 2^32) for v in [0,1]; v > 1 clamps to 2^32, NaN and negatives give 0 (O7).
__device__ __forceinline__ u64 quantise_weight(float v) {
    if (!(v > 0.0f)) return 0ull;
    if (v >= 1.0f) return 1ull << 32;
    return __float2ull_rz(v * 4294967296.0f);  // power-of-two scaling is exact
}

// W = C_{N-1}, comb offset U, log evidence, status, the ESS decision: run by ONE CTA of T threads once
// every scan tile is published (the last scan CTA, or bu_finalize_kernel).  Fixed-order double sums.
template <int T>
__device__ __forceinline__ void finalize_block(const ScanBuffers &sb, int N, int tiles, const FinalizeArgs &f,
                                               double *sh /* [T] shared */) {
    const int tid = threadIdx.x;
    // prior-weight partials (one per 32 particles: 32768 at N = 2^20): 8 independent loads per round
    // (the loop is latency-bound); fixed order, so the sum is bit-reproducible
    double acc = 0.0;
    if (f.has_prior) {
        int i = tid;
        for (; i + 7 * T < f.n_wsum_parts; i += 8 * T) {
            double t[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) t[u] = __ldcg(sb.part_wsum + i + u * T);
            acc += ((t[0] + t[1]) + (t[2] + t[3])) + ((t[4] + t[5]) + (t[6] + t[7]));
        }
        for (; i < f.n_wsum_parts; i += T) acc += __ldcg(sb.part_wsum + i);
    }
    sh[tid] = acc;
    __syncthreads();
    for (int o = T / 2; o > 0; o >>= 1) {
        if (tid < o) sh[tid] += sh[tid + o];
        __syncthreads();
    }
    const double sum_wp = sh[0];
    __syncthreads();
    // sum v (threads [0, T/2)) and sum v^2 (threads [T/2, T)) of the scan tiles: two trees at once
    constexpr int Hh = T / 2;
    acc = 0.0;
    for (int i = tid & (Hh - 1); i < tiles; i += Hh) acc += __ldcg(sb.tile_sumv + (tid < Hh ? 0 : tiles) + i);
    sh[tid] = acc;
    __syncthreads();
    for (int o = Hh / 2; o > 0; o >>= 1) {
        if ((tid & (Hh - 1)) < o) sh[tid] += sh[tid + o];
        __syncthreads();
    }
    const double sum_v = sh[0], sum_v2 = sh[Hh];
    if (tid == 0) {
        const double sum_w = f.has_prior ? sum_wp : (double)N;
        const u64 W = ld_u64_volatile(&sb.state->total_q);
        float m = 0.0f;
        int status = 0;
        if (f.from_logits) {
            m = ordered_to_float(*reinterpret_cast<volatile int *>(sb.max_ordered));
            if (!(fabsf(m) < INFINITY)) status = 1;
        }
        if (W == 0ull) status = 1;
        const uint4 x = noise_words(f.seed, 0u, 0u, 0u, kStreamResample, 0u);
        const u64 x0 = (u64)x.x;
        // U = (x0 * W) >> 32 from the 96-bit product
        const u64 lo = x0 * W, hi = __umul64hi(x0, W);
        sb.state->offset_u = (hi << 32) | (lo >> 32);
        sb.state->sum_v = sum_v;
        sb.state->inv_sum_v = sum_v > 0.0 ? 1.0 / sum_v : 0.0;
        sb.state->sum_w = sum_w;
        sb.state->max_logit = m;
        sb.state->status = status;
        // adaptive resampling: resample iff ESS < ess_threshold * N (+inf: always)
        const double ess = (status == 0 && sum_v2 > 0.0) ? sum_v * sum_v / sum_v2 : 0.0;
        const int resample = status == 0 && (isinf(f.ess_threshold) || ess < (double)f.ess_threshold * (double)N);
        sb.state->ess = ess;
        sb.state->resample = resample;
        if (f.ess_out) *f.ess_out = (float)ess;
        if (f.resampled_out) *f.resampled_out = resample;
        if (f.dev_status_out) *f.dev_status_out = status;
        if (f.log_evidence_out)
            *f.log_evidence_out = status ? -INFINITY : (float)((double)m + log(sum_v) - log(sum_w));
    }
}

template <bool FROM_LOGITS>
__global__ void __launch_bounds__(kScanThreads) weight_scan_kernel(ScanBuffers sb,
                                                                   const float *__restrict__ in, int N,
                                                                   float *post_weights_out, const FinalizeArgs fin) {
    constexpr int kWarpsS = kScanThreads / 32;
    __shared__ double fin_sh[kScanThreads];
    __shared__ int tile_s, last_s;
    __shared__ u64 warp_tot[kWarpsS];
    __shared__ u64 look_tot[kWarpsS];
    __shared__ int look_first[kWarpsS];
    __shared__ double dsum[kWarpsS], dsum2[kWarpsS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // Tile = ticket taken at start: a look-back only waits for tiles whose CTA has already started,
    // whatever order the hardware dispatches the CTAs in.
    if (tid == 0) tile_s = (int)atomicAdd(&sb.state->tile_counter, 1u);
    __syncthreads();
    const int tile = tile_s;
    const int base = tile * kScanTile + tid * kItems;

    float m = 0.0f;
    bool bad = false;
    if (FROM_LOGITS) {
        m = ordered_to_float(*sb.max_ordered);
        bad = !(fabsf(m) < INFINITY);  // -inf (all weights zero), +inf or NaN scores
    }
    float x[kItems];
    if (base + kItems <= N) {
        const float4 a = __ldcs(reinterpret_cast<const float4 *>(in + base));
        const float4 b = __ldcs(reinterpret_cast<const float4 *>(in + base) + 1);
        x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w;
        x[4] = b.x; x[5] = b.y; x[6] = b.z; x[7] = b.w;
    } else {
#pragma unroll
        for (int i = 0; i < kItems; ++i) x[i] = (base + i < N) ? in[base + i] : (FROM_LOGITS ? -INFINITY : 0.0f);
    }
    u64 c[kItems];
    u64 run = 0;
    double sv = 0.0, sv2 = 0.0;  // sum v, sum v^2 (effective sample size)
#pragma unroll
    for (int i = 0; i < kItems; ++i) {
        float v = x[i];
        if (FROM_LOGITS) v = bad ? 0.0f : expf(x[i] - m);
        if (base + i >= N) v = 0.0f;
        x[i] = v;
        sv += (double)v;
        sv2 += (double)v * (double)v;
        run += quantise_weight(v);
        c[i] = run;
    }
    // block-wide inclusive scan of the per-thread totals
    u64 incl = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u64 t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sv += __shfl_xor_sync(0xffffffffu, sv, o);
        sv2 += __shfl_xor_sync(0xffffffffu, sv2, o);
    }
    if (lane == 31) warp_tot[warp] = incl;
    if (lane == 0) {
        dsum[warp] = sv;
        dsum2[warp] = sv2;
    }
    __syncthreads();
    u64 warp_prefix = 0, agg = 0;
#pragma unroll
    for (int w = 0; w < kWarpsS; ++w) {
        if (w < warp) warp_prefix += warp_tot[w];
        agg += warp_tot[w];
    }
    const u64 thread_excl = warp_prefix + (incl - run);

    // publish this tile's aggregate (tile 0: its inclusive prefix) before looking back
    if (tid == 0) {
        if (tile == 0) {
            sb.tile_incl[0] = agg;
            st_flag(sb.tile_flag, kFlagInclusive);
        } else {
            sb.tile_agg[tile] = agg;
            st_flag(sb.tile_flag + tile, kFlagAggregate);
        }
        double t = 0.0, t2 = 0.0;
#pragma unroll
        for (int w = 0; w < kWarpsS; ++w) {
            t += dsum[w];
            t2 += dsum2[w];
        }
        sb.tile_sumv[tile] = t;
        sb.tile_sumv[gridDim.x + tile] = t2;
    }
    // Decoupled look-back, one predecessor per THREAD and round (kScanThreads per round): when all
    // tiles of a launch are co-resident nobody owns an inclusive prefix early, and a 32-wide
    // look-back would walk tiles/32 dependent rounds of L2 latency; this walks tiles/512.
    // Every predecessor holds a smaller ticket, i.e. has started: the spin cannot deadlock.
    u64 excl = 0;
    for (int j = tile - 1; j >= 0; j -= kScanThreads) {
        const int idx = j - tid;
        unsigned f = kFlagInclusive;
        u64 val = 0;
        if (idx >= 0) {
            while ((f = ld_flag(sb.tile_flag + idx)) == kFlagEmpty) __nanosleep(40);
            val = ld_u64_volatile(f == kFlagInclusive ? sb.tile_incl + idx : sb.tile_agg + idx);
        }
        // nearest predecessor (smallest tid) that already owns an inclusive prefix
        const unsigned inc_mask = __ballot_sync(0xffffffffu, f == kFlagInclusive);
        if (lane == 0) look_first[warp] = inc_mask ? warp * 32 + (__ffs(inc_mask) - 1) : kScanThreads;
        __syncthreads();
        int first = kScanThreads;
#pragma unroll
        for (int w = kWarpsS - 1; w >= 0; --w)
            if (look_first[w] < kScanThreads) first = look_first[w];
        u64 contrib = (tid <= first) ? val : 0ull;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) contrib += __shfl_xor_sync(0xffffffffu, contrib, o);
        if (lane == 0) look_tot[warp] = contrib;
        __syncthreads();
#pragma unroll
        for (int w = 0; w < kWarpsS; ++w) excl += look_tot[w];
        if (first < kScanThreads) break;  // uniform: every thread read the same look_first[]
    }
    if (tid == 0) {
        if (tile > 0) {
            sb.tile_incl[tile] = excl + agg;
            st_flag(sb.tile_flag + tile, kFlagInclusive);
        }
        if (tile == (N + kScanTile - 1) / kScanTile - 1) sb.state->total_q = excl + agg;
    }
    const u64 off = excl + thread_excl;
    if (base + kItems <= N) {
        ulonglong2 *dst = reinterpret_cast<ulonglong2 *>(sb.cdf + base);
#pragma unroll
        for (int i = 0; i < kItems / 2; ++i) dst[i] = make_ulonglong2(off + c[2 * i], off + c[2 * i + 1]);
        if (post_weights_out) {
            float4 *pw = reinterpret_cast<float4 *>(post_weights_out + base);
            pw[0] = make_float4(x[0], x[1], x[2], x[3]);
            pw[1] = make_float4(x[4], x[5], x[6], x[7]);
        }
    } else {
#pragma unroll
        for (int i = 0; i < kItems; ++i)
            if (base + i < N) {
                sb.cdf[base + i] = off + c[i];
                if (post_weights_out) post_weights_out[base + i] = x[i];
            }
    }
    // the last CTA to get here finalises (W, U, evidence, status, ESS): one launch less per update
    if (fin.enabled) {
        __threadfence();
        __syncthreads();
        if (tid == 0) last_s = atomicAdd(&sb.state->done_counter, 1u) == gridDim.x - 1u;
        __syncthreads();
        if (last_s) {
            __threadfence();
            finalize_block<kScanThreads>(sb, N, (int)gridDim.x, fin, fin_sh);
        }
    }
}

constexpr int kFinThreads = 1024;
__global__ void __launch_bounds__(kFinThreads) bu_finalize_kernel(ScanBuffers sb, int N, int tiles, FinalizeArgs fin) {
    __shared__ double sh[kFinThreads];
    finalize_block<kFinThreads>(sb, N, tiles, fin, sh);
}

// N*C > k*W + U as 128-bit integers.
__device__ __forceinline__ bool comb_below(u64 Nn, u64 C, u64 rhs_hi, u64 rhs_lo) {
    const u64 lhs_lo = Nn * C, lhs_hi = __umul64hi(Nn, C);
    return lhs_hi > rhs_hi || (lhs_hi == rhs_hi && lhs_lo > rhs_lo);
}

template <int VEC>
struct VecT;
template <> struct VecT<16> { typedef uint4 type; };
template <> struct VecT<8> { typedef uint2 type; };
template <> struct VecT<4> { typedef uint32_t type; };
template <> struct VecT<2> { typedef uint16_t type; };

constexpr int kSegMax = 2048;  // CDF samples staged per CTA (16 KB)

// first i in [lo, hi] with N*C_i > rhs (the answer is known to lie in the range): one thread
__device__ __forceinline__ int comb_search_global(const u64 *__restrict__ cdf, u64 Nn, int lo, int hi, u64 rhs_hi,
                                                  u64 rhs_lo) {
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (comb_below(Nn, __ldg(cdf + mid), rhs_hi, rhs_lo)) hi = mid;
        else lo = mid + 1;
    }
    return lo;
}

// The same search by a whole warp, 32 probes per round: log32(N) dependent rounds of L2 latency
// instead of log2(N) (4 instead of 20 at N = 2^20).  All lanes return the answer.
__device__ __forceinline__ int comb_search_warp(const u64 *__restrict__ cdf, u64 Nn, int lo, int hi, u64 rhs_hi,
                                                u64 rhs_lo, int lane) {
    while (lo < hi) {
        const long long span = (long long)hi - lo + 1;
        const long long step = (span + 31) / 32;
        long long p = (long long)lo + (lane + 1) * step - 1;
        if (p > hi) p = hi;
        const bool above = comb_below(Nn, __ldg(cdf + p), rhs_hi, rhs_lo);  // answer <= p
        const unsigned mask = __ballot_sync(0xffffffffu, above);             // lane 31 probes hi: mask != 0
        const int f = __ffs(mask) - 1;
        const long long p_f = __shfl_sync(0xffffffffu, p, f);
        const long long p_prev = __shfl_sync(0xffffffffu, p, f > 0 ? f - 1 : 0);
        if (f > 0) lo = (int)p_prev + 1;
        hi = (int)p_f;
    }
    return lo;
}

template <int VEC>
__global__ void __launch_bounds__(256) resample_gather_kernel(ScanBuffers sb, int N,
                                                              const uint8_t *__restrict__ proposals,
                                                              int row_bytes, uint8_t *particles_out,
                                                              float *weights_out, int32_t *ancestors_out,
                                                              const float *__restrict__ w_in, int from_logits) {
    __shared__ int anc_s[256];
    __shared__ int range_s[2];
    __shared__ u64 seg[kSegMax];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int k0 = blockIdx.x * 256, k = k0 + tid;
    const int rows = min(256, N - k0);
    // only the fields needed on the common path stay in registers (the whole struct cost 8 more)
    const u64 W = sb.state->total_q, U = sb.state->offset_u;
    const int st_status = sb.state->status, st_resample = sb.state->resample;
    u64 rhs_lo = (u64)k * W, rhs_hi = __umul64hi((u64)k, W);
    rhs_lo += U;
    rhs_hi += (rhs_lo < U) ? 1ull : 0ull;
    if (st_status == 0 && st_resample) {
        // Ancestors are non-decreasing in k: bracket the CTA's outputs with the ancestors of its
        // first and last output (warps 0 and 1, one cooperative search each).
        if (warp < 2) {
            const int kk = warp == 0 ? k0 : k0 + rows - 1;
            u64 r_lo = (u64)kk * W, r_hi = __umul64hi((u64)kk, W);
            r_lo += U;
            r_hi += (r_lo < U) ? 1ull : 0ull;
            // the answer exists: k*W + U < N*W = N*C_{N-1}
            const int a = comb_search_warp(sb.cdf, (u64)N, 0, N - 1, r_hi, r_lo, lane);
            if (lane == 0) range_s[warp] = a;
        }
        __syncthreads();
        const int a_lo = range_s[0], a_hi = range_s[1];
        const int len = a_hi - a_lo + 1;
        // stage the segment [a_lo, a_hi] in shared memory, every s-th entry when it is longer than
        // kSegMax (sample g = last entry of group g): search the samples, then inside one group
        const int s_ = (len + kSegMax - 1) / kSegMax;
        const int cnt = (len + s_ - 1) / s_;
        for (int i = tid; i < cnt; i += 256) {
            const long long pos = (long long)a_lo + (long long)(i + 1) * s_ - 1;
            seg[i] = __ldg(sb.cdf + (pos < a_hi ? pos : a_hi));
        }
        __syncthreads();
        int a = k;
        if (k < N) {
            int lo = 0, hi = cnt - 1;
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (comb_below((u64)N, seg[mid], rhs_hi, rhs_lo)) hi = mid;
                else lo = mid + 1;
            }
            a = a_lo + lo;
            if (s_ > 1) {
                const long long g_lo = (long long)a_lo + (long long)lo * s_;
                long long g_hi = g_lo + s_ - 1;
                if (g_hi > a_hi) g_hi = a_hi;
                a = comb_search_global(sb.cdf, (u64)N, (int)g_lo, (int)g_hi, rhs_hi, rhs_lo);
            }
        }
        anc_s[tid] = a;
    } else {
        anc_s[tid] = k;  // degenerate weights, or ESS above the threshold: identity
    }
    if (k < N) {
        if (ancestors_out) ancestors_out[k] = anc_s[tid];
        if (weights_out) {
            float w = 1.0f / (float)N;
            if (st_status == 0 && !st_resample) {  // no resampling: carry the normalised weights v_k / sum v
                const float x = w_in[k];
                const float v = from_logits ? expf(x - sb.state->max_logit) : x;
                w = (float)((double)v * sb.state->inv_sum_v);  // one DMUL (a double division here costs 8 registers)
            }
            weights_out[k] = w;
        }
    }
    __syncthreads();
    if (particles_out) {
        typedef typename VecT<VEC>::type V;
        const int cpr = row_bytes / VEC;
        const int total = rows * cpr;
        for (int c = tid; c < total; c += 256) {
            const int j = c / cpr, off = c - j * cpr;
            const V val = *reinterpret_cast<const V *>(proposals + (size_t)anc_s[j] * row_bytes + (size_t)off * VEC);
            __stcs(reinterpret_cast<V *>(particles_out + (size_t)(k0 + j) * row_bytes + (size_t)off * VEC), val);
        }
    }
}

}  // namespace

cudaError_t launch_bu_init(const ScanBuffers &sb, int N, cudaStream_t st) {
    const int tiles = scan_tiles(N);
    bu_init_kernel<<<(tiles + 255) / 256, 256, 0, st>>>(sb, tiles);
    return cudaGetLastError();
}

bool obs_tower_fits(const MlpDev &f) {
    for (int l = 0; l <= f.n_layers; ++l)
        if (f.dims[l] > kObsMaxWidth) return false;
    return true;
}

cudaError_t launch_bu_init_obs(const ScanBuffers &sb, int N, const MlpDev &f, const float *obs, float *e_out,
                               bool bf16, cudaStream_t st) {
    const int tiles = scan_tiles(N);
    if (bf16) bu_init_obs_kernel<true><<<1, kObsThreads, 0, st>>>(sb, tiles, f, obs, e_out);
    else bu_init_obs_kernel<false><<<1, kObsThreads, 0, st>>>(sb, tiles, f, obs, e_out);
    return cudaGetLastError();
}

cudaError_t launch_weight_scan(const ScanBuffers &sb, const float *in, int N, bool from_logits,
                               float *post_weights_out, cudaStream_t st, const FinalizeArgs *fin) {
    const int tiles = scan_tiles(N);
    FinalizeArgs f{};
    if (fin) f = *fin;
    if (from_logits) weight_scan_kernel<true><<<tiles, kScanThreads, 0, st>>>(sb, in, N, post_weights_out, f);
    else weight_scan_kernel<false><<<tiles, kScanThreads, 0, st>>>(sb, in, N, post_weights_out, f);
    return cudaGetLastError();
}

cudaError_t launch_bu_finalize(const ScanBuffers &sb, int N, int n_wsum_parts, bool has_prior,
                               uint64_t seed, float *log_evidence_out, int32_t *dev_status_out,
                               cudaStream_t st, float ess_threshold, float *ess_out, int32_t *resampled_out) {
    // n_wsum_parts < 0 marks the stage-level resampler (weights given directly, no logits)
    FinalizeArgs f{};
    f.enabled = 1;
    f.from_logits = n_wsum_parts >= 0;
    f.n_wsum_parts = n_wsum_parts < 0 ? 0 : n_wsum_parts;
    f.has_prior = has_prior ? 1 : 0;
    f.seed = seed;
    f.ess_threshold = ess_threshold;
    f.log_evidence_out = log_evidence_out; f.ess_out = ess_out;
    f.dev_status_out = dev_status_out; f.resampled_out = resampled_out;
    bu_finalize_kernel<<<1, kFinThreads, 0, st>>>(sb, N, scan_tiles(N), f);
    return cudaGetLastError();
}

cudaError_t launch_resample_gather(const ScanBuffers &sb, int N, const void *proposals, int row_bytes,
                                   void *particles_out, float *weights_out, int32_t *ancestors_out,
                                   cudaStream_t st, const float *w_in, bool from_logits) {
    const int grid = (N + 255) / 256;
    const uint8_t *src = reinterpret_cast<const uint8_t *>(proposals);
    uint8_t *dst = reinterpret_cast<uint8_t *>(particles_out);
    if (row_bytes % 16 == 0)
        resample_gather_kernel<16><<<grid, 256, 0, st>>>(sb, N, src, row_bytes, dst, weights_out, ancestors_out, w_in, from_logits ? 1 : 0);
    else if (row_bytes % 8 == 0)
        resample_gather_kernel<8><<<grid, 256, 0, st>>>(sb, N, src, row_bytes, dst, weights_out, ancestors_out, w_in, from_logits ? 1 : 0);
    else if (row_bytes % 4 == 0)
        resample_gather_kernel<4><<<grid, 256, 0, st>>>(sb, N, src, row_bytes, dst, weights_out, ancestors_out, w_in, from_logits ? 1 : 0);
    else
        resample_gather_kernel<2><<<grid, 256, 0, st>>>(sb, N, src, row_bytes, dst, weights_out, ancestors_out, w_in, from_logits ? 1 : 0);
    return cudaGetLastError();
}

// =====================================================================================
// voila_resample_systematic_static: the stage-level resampler for callers that may not allocate
// (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Same three kernels as
// voila_resample_systematic; the scratch they need (the uint64 CDF, the look-back tile records, the
// scan bookkeeping) lives in ONE file-scope device array of a fixed size instead of the ctx
// workspace: 8 MiB + 16 KiB that every GPU loading the library holds until exit, good for
// N <= kStaticMaxN = 2^20 particles (VOILA_STATIC_MAX_N in voila.h).
// In host code `g_static_scratch` is a host-side stand-in for the symbol, not a device address:
// the address the kernels get comes from cudaGetSymbolAddress, once per device, with that device
// current.  Every call shares the array: calls that overlap on the GPU (two streams, two host
// threads) race on it; bu_init_kernel clears what has to start at zero (tile flags, ScanState,
// the running maximum) at the head of every call, the rest is overwritten before it is read.
// =====================================================================================
namespace {

constexpr int kStaticMaxN = 1 << 20;
constexpr int kStaticTiles = kStaticMaxN / kScanTile;
static_assert(kStaticMaxN % kScanTile == 0, "whole tiles");
// layout in 8-byte words, every part 256-byte aligned
constexpr size_t kStOffCdf = 0;                                      // [kStaticMaxN] uint64
constexpr size_t kStOffAgg = kStOffCdf + (size_t)kStaticMaxN;        // [tiles] uint64
constexpr size_t kStOffIncl = kStOffAgg + kStaticTiles;              // [tiles] uint64
constexpr size_t kStOffSumv = kStOffIncl + kStaticTiles;             // [2 * tiles] double
constexpr size_t kStOffFlag = kStOffSumv + 2 * kStaticTiles;         // [tiles] uint32
constexpr size_t kStOffState = kStOffFlag + kStaticTiles / 2;        // ScanState (<= 32 words)
constexpr size_t kStOffMax = kStOffState + 32;                       // [1] int   (32 words)
constexpr size_t kStOffWsum = kStOffMax + 32;                        // [1] double (32 words, unused by this path)
constexpr size_t kStaticWords = kStOffWsum + 32;
static_assert(sizeof(ScanState) <= 32 * 8, "ScanState fits its slot");
static_assert(kStaticTiles % 64 == 0 && (kStOffAgg % 32) == 0 && (kStOffState % 32) == 0, "256-byte aligned parts");

static __device__ __align__(256) unsigned long long g_static_scratch[kStaticWords];

constexpr int kStaticMaxDevices = 64;
std::atomic<unsigned long long *> g_static_addr[kStaticMaxDevices];  // device address of the array, per device

}  // namespace

int static_resample_max_n() { return kStaticMaxN; }
size_t static_scratch_bytes() { return kStaticWords * sizeof(unsigned long long); }

// Runs on the CURRENT device.  No cudaMalloc / cudaFree, no allocating library call; three launches.
cudaError_t launch_resample_systematic_static(const float *v, int N, uint64_t seed, int32_t *ancestors_out,
                                              int32_t *dev_status_out, cudaStream_t st, const char **why) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDevices) {
        if (why) *why = "device ordinal beyond the static scratch table (64 devices)";
        return cudaErrorInvalidDevice;
    }
    unsigned long long *base = g_static_addr[dev].load(std::memory_order_acquire);
    if (!base) {
        // set-up, once per device, with that device current (two threads racing here store the same value)
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_static_scratch);
        if (e != cudaSuccess) {
            if (why) *why = "cudaGetSymbolAddress(g_static_scratch) failed";
            return e;
        }
        base = reinterpret_cast<unsigned long long *>(ptr);
        g_static_addr[dev].store(base, std::memory_order_release);
    }
    ScanBuffers sb;
    sb.cdf = base + kStOffCdf;
    sb.tile_agg = base + kStOffAgg;
    sb.tile_incl = base + kStOffIncl;
    sb.tile_sumv = reinterpret_cast<double *>(base + kStOffSumv);
    sb.tile_flag = reinterpret_cast<unsigned int *>(base + kStOffFlag);
    sb.state = reinterpret_cast<ScanState *>(base + kStOffState);
    sb.max_ordered = reinterpret_cast<int *>(base + kStOffMax);
    sb.part_wsum = reinterpret_cast<double *>(base + kStOffWsum);
    e = launch_bu_init(sb, N, st);  // clears the tile flags, ScanState and the running maximum of the last call
    if (e != cudaSuccess) return e;
    FinalizeArgs fin{};
    fin.enabled = 1;
    fin.seed = seed;
    fin.ess_threshold = INFINITY;
    fin.dev_status_out = dev_status_out;
    e = launch_weight_scan(sb, v, N, false, nullptr, st, &fin);
    if (e != cudaSuccess) return e;
    return launch_resample_gather(sb, N, nullptr, 16, nullptr, nullptr, ancestors_out, st, v, false);
}

}  // namespace voila
