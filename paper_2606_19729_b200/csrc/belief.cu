// belief.cu -- weight normalisation, prefix sum and systematic resampling of the SIR belief update
// (O5-O7; PAPER.md:77 "before resampling", :128 only relative weights matter, :137).
//
//   weight_scan    v_i = exp(L_i - m) (max-shifted), q_i = floor(v_i 2^32) as
//                  uint64, inclusive scan C_i in ONE pass: warp shuffles inside a 2048-element tile,
//                  decoupled look-back across tiles.  Integer addition is associative, so the CDF is
//                  independent of tiling and the resampled indices are bit-exact (reading R6).
//   bu_finalize    W = C_{N-1}, comb offset U = (x0 W) >> 32 from one Philox word, log evidence,
//                  degenerate-weight status.
//   resample_gather  i_k = min{ i : N C_i > k W + U } by binary search with 128-bit compares
//                  (the 8 N-byte CDF is L2 resident), then coalesced vectorised row gathers.
// HBM-bound; no tensor-core work here.
#include "voila_device.cuh"
#include "voila_kernels.h"

namespace voila {

namespace {

typedef unsigned long long u64;
constexpr int kScanThreads = 256;
constexpr int kItems = kScanTile / kScanThreads;  // 8
constexpr unsigned kFlagEmpty = 0u, kFlagAggregate = 1u, kFlagInclusive = 2u;

__global__ void bu_init_kernel(ScanBuffers sb, int tiles) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < tiles) sb.tile_flag[i] = kFlagEmpty;
    if (i == 0) {
        ScanState z;
        z.total_q = 0; z.offset_u = 0; z.sum_v = 0.0; z.sum_w = 0.0;
        z.max_logit = 0.0f; z.status = 0; z.tile_counter = 0; z.pad = 0;
        *sb.state = z;
        *sb.max_ordered = (int)0x80000000;
    }
}

__device__ __forceinline__ unsigned ld_flag(const unsigned *p) {
    return *reinterpret_cast<const volatile unsigned *>(p);
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

template <bool FROM_LOGITS>
__global__ void __launch_bounds__(kScanThreads) weight_scan_kernel(ScanBuffers sb,
                                                                   const float *__restrict__ in, int N,
                                                                   float *post_weights_out) {
    __shared__ unsigned tile_s;
    __shared__ u64 warp_tot[kScanThreads / 32];
    __shared__ u64 excl_s;
    __shared__ double dsum[kScanThreads / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) tile_s = atomicAdd(&sb.state->tile_counter, 1u);  // ticket: tiles start in order
    __syncthreads();
    const int tile = (int)tile_s;
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
    double sv = 0.0;
#pragma unroll
    for (int i = 0; i < kItems; ++i) {
        float v = x[i];
        if (FROM_LOGITS) v = bad ? 0.0f : expf(x[i] - m);
        if (base + i >= N) v = 0.0f;
        x[i] = v;
        sv += (double)v;
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
    for (int o = 16; o > 0; o >>= 1) sv += __shfl_xor_sync(0xffffffffu, sv, o);
    if (lane == 31) warp_tot[warp] = incl;
    if (lane == 0) dsum[warp] = sv;
    __syncthreads();
    u64 warp_prefix = 0, agg = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) {
        if (w < warp) warp_prefix += warp_tot[w];
        agg += warp_tot[w];
    }
    const u64 thread_excl = warp_prefix + (incl - run);

    if (warp == 0) {
        u64 excl = 0;
        if (tile == 0) {
            if (lane == 0) {
                sb.tile_incl[0] = agg;
                __threadfence();
                *reinterpret_cast<volatile unsigned *>(sb.tile_flag) = kFlagInclusive;
            }
        } else {
            if (lane == 0) {
                sb.tile_agg[tile] = agg;
                __threadfence();
                *reinterpret_cast<volatile unsigned *>(sb.tile_flag + tile) = kFlagAggregate;
            }
            // decoupled look-back, 32 predecessors per round
            int j = tile - 1;
            while (true) {
                const int idx = j - lane;
                unsigned f;
                do {
                    f = idx >= 0 ? ld_flag(sb.tile_flag + idx) : kFlagInclusive;
                } while (__any_sync(0xffffffffu, f == kFlagEmpty));
                __threadfence();
                u64 val = 0;
                if (idx >= 0) val = ld_u64_volatile(f == kFlagInclusive ? sb.tile_incl + idx : sb.tile_agg + idx);
                const unsigned inc_mask = __ballot_sync(0xffffffffu, f == kFlagInclusive);
                const int first = inc_mask ? (__ffs(inc_mask) - 1) : 32;
                u64 contrib = (lane <= first) ? val : 0ull;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) contrib += __shfl_xor_sync(0xffffffffu, contrib, o);
                excl += contrib;
                if (inc_mask) break;
                j -= 32;
            }
            if (lane == 0) {
                sb.tile_incl[tile] = excl + agg;
                __threadfence();
                *reinterpret_cast<volatile unsigned *>(sb.tile_flag + tile) = kFlagInclusive;
            }
        }
        if (lane == 0) {
            excl_s = excl;
            double t = 0.0;
#pragma unroll
            for (int w = 0; w < kScanThreads / 32; ++w) t += dsum[w];
            sb.tile_sumv[tile] = t;
            if (tile == (N + kScanTile - 1) / kScanTile - 1) sb.state->total_q = excl + agg;
        }
    }
    __syncthreads();
    const u64 off = excl_s + thread_excl;
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
}

__global__ void bu_finalize_kernel(ScanBuffers sb, int N, int tiles, int n_wsum_parts, int has_prior,
                                   int from_logits, uint64_t seed, float *log_evidence_out,
                                   int32_t *dev_status_out) {
    __shared__ double sh[256];
    const int tid = threadIdx.x;
    double acc = 0.0;
    for (int i = tid; i < tiles; i += 256) acc += sb.tile_sumv[i];
    sh[tid] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (tid < o) sh[tid] += sh[tid + o];
        __syncthreads();
    }
    const double sum_v = sh[0];
    __syncthreads();
    acc = 0.0;
    if (has_prior) for (int i = tid; i < n_wsum_parts; i += 256) acc += sb.part_wsum[i];
    sh[tid] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (tid < o) sh[tid] += sh[tid + o];
        __syncthreads();
    }
    if (tid == 0) {
        const double sum_w = has_prior ? sh[0] : (double)N;
        const u64 W = sb.state->total_q;
        float m = 0.0f;
        int status = 0;
        if (from_logits) {
            m = ordered_to_float(*sb.max_ordered);
            if (!(fabsf(m) < INFINITY)) status = 1;
        }
        if (W == 0ull) status = 1;
        const uint4 x = noise_words(seed, 0u, 0u, 0u, kStreamResample, 0u);
        const u64 x0 = (u64)x.x;
        // U = (x0 * W) >> 32 from the 96-bit product
        const u64 lo = x0 * W, hi = __umul64hi(x0, W);
        sb.state->offset_u = (hi << 32) | (lo >> 32);
        sb.state->sum_v = sum_v;
        sb.state->sum_w = sum_w;
        sb.state->max_logit = m;
        sb.state->status = status;
        if (dev_status_out) *dev_status_out = status;
        if (log_evidence_out)
            *log_evidence_out = status ? -INFINITY : (float)((double)m + log(sum_v) - log(sum_w));
    }
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

template <int VEC>
__global__ void __launch_bounds__(256) resample_gather_kernel(ScanBuffers sb, int N,
                                                              const uint8_t *__restrict__ proposals,
                                                              int row_bytes, uint8_t *particles_out,
                                                              float *weights_out, int32_t *ancestors_out) {
    __shared__ int anc_s[256];
    const int tid = threadIdx.x;
    const int k0 = blockIdx.x * 256, k = k0 + tid;
    const ScanState st = *sb.state;
    if (k < N) {
        int a = k;
        if (st.status == 0) {
            const u64 W = st.total_q, U = st.offset_u;
            u64 rhs_lo = (u64)k * W, rhs_hi = __umul64hi((u64)k, W);
            rhs_lo += U;
            rhs_hi += (rhs_lo < U) ? 1ull : 0ull;
            int lo = 0, hi = N - 1;  // the answer exists: k*W + U < N*W = N*C_{N-1}
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (comb_below((u64)N, __ldg(sb.cdf + mid), rhs_hi, rhs_lo)) hi = mid;
                else lo = mid + 1;
            }
            a = lo;
        }
        anc_s[tid] = a;
        if (ancestors_out) ancestors_out[k] = a;
        if (weights_out) weights_out[k] = 1.0f / (float)N;
    }
    __syncthreads();
    if (particles_out) {
        typedef typename VecT<VEC>::type V;
        const int rows = min(256, N - k0);
        const int cpr = row_bytes / VEC;
        const int total = rows * cpr;
        for (int c = tid; c < total; c += 256) {
            const int j = c / cpr, off = c - j * cpr;
            const V val = *reinterpret_cast<const V *>(proposals + (size_t)anc_s[j] * row_bytes + (size_t)off * VEC);
            *reinterpret_cast<V *>(particles_out + (size_t)(k0 + j) * row_bytes + (size_t)off * VEC) = val;
        }
    }
}

}  // namespace

cudaError_t launch_bu_init(const ScanBuffers &sb, int N, cudaStream_t st) {
    const int tiles = scan_tiles(N);
    bu_init_kernel<<<(tiles + 255) / 256, 256, 0, st>>>(sb, tiles);
    return cudaGetLastError();
}

cudaError_t launch_weight_scan(const ScanBuffers &sb, const float *in, int N, bool from_logits,
                               float *post_weights_out, cudaStream_t st) {
    const int tiles = scan_tiles(N);
    if (from_logits) weight_scan_kernel<true><<<tiles, kScanThreads, 0, st>>>(sb, in, N, post_weights_out);
    else weight_scan_kernel<false><<<tiles, kScanThreads, 0, st>>>(sb, in, N, post_weights_out);
    return cudaGetLastError();
}

cudaError_t launch_bu_finalize(const ScanBuffers &sb, int N, int n_wsum_parts, bool has_prior,
                               uint64_t seed, float *log_evidence_out, int32_t *dev_status_out,
                               cudaStream_t st) {
    // n_wsum_parts < 0 marks the stage-level resampler (weights given directly, no logits)
    const int from_logits = n_wsum_parts >= 0;
    bu_finalize_kernel<<<1, 256, 0, st>>>(sb, N, scan_tiles(N), n_wsum_parts < 0 ? 0 : n_wsum_parts,
                                          has_prior ? 1 : 0, from_logits, seed, log_evidence_out,
                                          dev_status_out);
    return cudaGetLastError();
}

cudaError_t launch_resample_gather(const ScanBuffers &sb, int N, const void *proposals, int row_bytes,
                                   void *particles_out, float *weights_out, int32_t *ancestors_out,
                                   cudaStream_t st) {
    const int grid = (N + 255) / 256;
    const uint8_t *src = reinterpret_cast<const uint8_t *>(proposals);
    uint8_t *dst = reinterpret_cast<uint8_t *>(particles_out);
    if (row_bytes % 16 == 0)
        resample_gather_kernel<16><<<grid, 256, 0, st>>>(sb, N, src, row_bytes, dst, weights_out, ancestors_out);
    else if (row_bytes % 8 == 0)
        resample_gather_kernel<8><<<grid, 256, 0, st>>>(sb, N, src, row_bytes, dst, weights_out, ancestors_out);
    else if (row_bytes % 4 == 0)
        resample_gather_kernel<4><<<grid, 256, 0, st>>>(sb, N, src, row_bytes, dst, weights_out, ancestors_out);
    else
        resample_gather_kernel<2><<<grid, 256, 0, st>>>(sb, N, src, row_bytes, dst, weights_out, ancestors_out);
    return cudaGetLastError();
}

}  // namespace voila
