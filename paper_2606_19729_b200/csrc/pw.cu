// pw.cu -- vectorised progressive widening with batched likelihood (section 4.3;
// SURVEY 8f f1; readings R26-R29): the bookkeeping kernels of voila_pw_update.
//
//   pw_widen       one warp per action node: the widening criterion |C(a)| < k_o N(a)^alpha_o visit
//                  by visit (a slew-limited tracker of the threshold, evaluated with a warp min-scan),
//                  the branch of every simulation, its rank inside its (action node, branch) child
//                  belief, the members of every child
//   pw_seg_scan    exclusive scan of the child sizes -> child offsets in the sorted order
//   pw_perm        sorted position of every simulation (stable counting sort by child)
//   pw_weights     v = exp(L - max over the child) in sorted order (-> the uint64 scan of belief.cu)
//   pw_resample    per child: exact-integer systematic resampling among its members + row gather
// The MLP work (proposals, sampled observations of the opened branches, observation tower over
// all branch observations, state tower + scores) is in mlp_ffma.cu (pw_*_ffma_kernel).
#include "voila_device.cuh"
#include "voila_kernels.h"

namespace voila {

namespace {

typedef unsigned long long u64;

// T(n) = ceil(k_o n^alpha_o (1 - 1e-9)) in fp64 (reading R27), capped at M_max.
__device__ __forceinline__ int pw_threshold(double k_o, double alpha_o, int n, int M_max) {
    const double x = k_o * pow((double)n, alpha_o) * (1.0 - 1e-9);
    if (!(x < (double)M_max)) return M_max;
    const int t = (int)ceil(x);
    return t < 0 ? 0 : t;
}

constexpr int kWidenWarps = 4;

// One warp per action node.  Serial semantics (per visit j = 0, 1, ... of this batch):
//   n = N0 + j + 1;  if C < min(M_max, T(n)): open branch C, C += 1;  else attach to (x_i C) >> 32.
// C follows the non-decreasing target D'_j = max(min(M_max, T(n)), C0) with slope <= 1:
//   C_j = min(C0 + j + 1, min_{i <= j} (D'_i + j - i)),
// i.e. a prefix minimum of D'_i - i: a warp scan per 32 visits with a running carry.
__global__ void __launch_bounds__(kWidenWarps * 32) pw_widen_kernel(PwArgs a) {
    __shared__ int cnt_s[kWidenWarps][kPwMaxBranches];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = blockIdx.x * kWidenWarps + warp;
    if (g >= a.G) return;
    int *cnt = cnt_s[warp];
    const int M = a.M_max;
    for (int m = lane; m < M; m += 32) {
        cnt[m] = 0;
        a.new_src[(size_t)g * M + m] = -1;
        a.seg_max[(size_t)g * M + m] = (int)0x80000000;
    }
    __syncwarp();
    const int i0 = a.group_off[g], n_g = a.group_off[g + 1] - i0;
    const int C0 = a.branch_count[g], N0 = a.visit_count[g];
    int carry_min = 0x7fffffff;  // min over earlier visits of D'_i - i
    int c_prev_chunk = C0;       // C after the last visit of the previous chunk
    for (int base = 0; base < n_g; base += 32) {
        const int j = base + lane;
        const bool act = j < n_g;
        int val = 0x7fffffff;
        if (act) {
            int D = pw_threshold(a.k_o, a.alpha_o, N0 + j + 1, M);
            if (D < C0) D = C0;
            val = D - j;
        }
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, val, o);
            if (lane >= o) val = min(val, t);
        }
        val = min(val, carry_min);
        int C = act ? min(C0 + j + 1, val + j) : 0;
        int C_before = __shfl_up_sync(0xffffffffu, C, 1);
        if (lane == 0) C_before = c_prev_chunk;
        const int i = i0 + j;
        int b = 0;
        bool opened = false;
        if (act) {
            opened = C > C_before;
            if (opened) {
                b = C_before;
                a.new_src[(size_t)g * M + b] = i;
            } else {
                const uint4 x = noise_words(a.seed, (uint32_t)i, 0u, 0u, kStreamPwAttach, 0u);
                b = (int)(((u64)x.x * (u64)C_before) >> 32);
            }
        }
        // rank inside the (action node, branch) child: members of earlier chunks + earlier lanes
        const unsigned peers = __match_any_sync(0xffffffffu, act ? b : -1 - lane);
        if (act) {
            const int rank = cnt[b] + __popc(peers & ((1u << lane) - 1u));
            a.sim_group[i] = g;
            a.sim_branch[i] = b;
            a.sim_rank[i] = rank;
            if (a.opened_out) a.opened_out[i] = opened ? 1 : 0;
        }
        __syncwarp();
        if (act && (peers & ((1u << lane) - 1u)) == 0u) cnt[b] += __popc(peers);  // lowest lane of each child
        __syncwarp();
        carry_min = __shfl_sync(0xffffffffu, val, 31);
        const int last = min(31, n_g - 1 - base);
        c_prev_chunk = __shfl_sync(0xffffffffu, C, last);
    }
    for (int m = lane; m < M; m += 32) a.seg_count[(size_t)g * M + m] = cnt[m];
    if (lane == 0) {
        a.branch_count[g] = n_g > 0 ? c_prev_chunk : C0;
        a.visit_count[g] = N0 + n_g;
    }
}

// Exclusive scan of the child sizes (n = G * M_max entries), one CTA: every WARP scans a contiguous
// run of the array 32 entries at a time (coalesced, shuffles only, the running prefix in a register),
// one block scan of the 32 run totals, then the run offsets are added in a second coalesced sweep.
// (The first version scanned 1024 entries per round with three block barriers each: 36 us for 2^15
// entries.  Integer sums, so the grouping does not change a bit.)
__global__ void __launch_bounds__(1024) pw_seg_scan_kernel(const int32_t *__restrict__ cnt, int n, int32_t *off) {
    __shared__ int warp_tot[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int per = ((n + 1023) / 1024) * 32;  // entries per warp, a multiple of 32
    const int lo = min(n, warp * per), hi = min(n, lo + per);
    int carry = 0;
    for (int base = lo; base < hi; base += 32) {
        const int idx = base + lane;
        const int v = idx < hi ? __ldg(cnt + idx) : 0;
        int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (idx < hi) off[idx] = carry + incl - v;
        carry += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) warp_tot[warp] = carry;
    __syncthreads();
    if (warp == 0) {
        const int t = warp_tot[lane];
        int w_incl = t;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int u = __shfl_up_sync(0xffffffffu, w_incl, o);
            if (lane >= o) w_incl += u;
        }
        warp_tot[lane] = w_incl - t;  // exclusive prefix of the run totals
        if (lane == 31) off[n] = w_incl;
    }
    __syncthreads();
    const int add = warp_tot[warp];
    if (add != 0)
        for (int idx = lo + lane; idx < hi; idx += 32) off[idx] += add;
}

__global__ void pw_perm_kernel(PwArgs a) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.N) return;
    const int seg = a.sim_group[i] * a.M_max + a.sim_branch[i];
    const int pos = a.seg_off[seg] + a.sim_rank[i];
    a.perm[pos] = i;
    a.seg_of_pos[pos] = seg;
    a.sim_seg[i] = seg;
    a.sim_action[i] = a.group_action[a.sim_group[i]];
    if (a.sim_branch_out) a.sim_branch_out[i] = a.sim_branch[i];
}

// v in sorted order; a child whose maximum is not finite (all weights zero, NaN / inf scores) gets
// v = 0 everywhere, which the resampler turns into the identity + status.
__global__ void pw_weights_kernel(PwArgs a) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= a.N) return;
    const int i = a.perm[p];
    const float m = ordered_to_float(a.seg_max[a.seg_of_pos[p]]);
    const float v = (fabsf(m) < INFINITY) ? expf(a.logits[i] - m) : 0.0f;
    a.v_sorted[p] = v;
    if (a.post_weights_out) a.post_weights_out[i] = v;
}

__device__ __forceinline__ bool comb_gt(u64 n, u64 c, u64 rhs_hi, u64 rhs_lo) {
    const u64 lo = n * c, hi = __umul64hi(n, c);
    return hi > rhs_hi || (hi == rhs_hi && lo > rhs_lo);
}

// Position p of the sorted order belongs to child seg with members [lo, hi): draw k = p - lo,
//   r = min{ r in [lo, hi) : n (C_r - base) > k W + U },  U = (x0 W) >> 32,  x0 = Philox word of the child.
template <int VEC>
__global__ void __launch_bounds__(256) pw_resample_kernel(PwArgs a, const u64 *__restrict__ cdf, int row_bytes) {
    __shared__ int anc_s[256], dst_s[256];
    const int tid = threadIdx.x;
    const int p0 = blockIdx.x * 256, p = p0 + tid;
    const int rows = min(256, a.N - p0);
    if (p < a.N) {
        const int seg = a.seg_of_pos[p];
        const int lo = a.seg_off[seg], hi = a.seg_off[seg + 1];
        const u64 n = (u64)(hi - lo);
        const u64 base = lo > 0 ? cdf[lo - 1] : 0ull;
        const u64 W = cdf[hi - 1] - base;
        const int i = a.perm[p];
        int anc = i;
        if (W == 0ull) {
            if (p == lo && a.seg_status_out) a.seg_status_out[seg] = 1;
        } else {
            const uint4 x = noise_words(a.seed, (uint32_t)seg, 0u, 0u, kStreamResample, 0u);
            const u64 x0 = (u64)x.x;
            const u64 ulo = x0 * W, uhi = __umul64hi(x0, W);
            const u64 U = (uhi << 32) | (ulo >> 32);
            const u64 k = (u64)(p - lo);
            u64 rhs_lo = k * W, rhs_hi = __umul64hi(k, W);
            rhs_lo += U;
            rhs_hi += (rhs_lo < U) ? 1ull : 0ull;
            int l = lo, h = hi - 1;  // the answer exists: k W + U < n W
            while (l < h) {
                const int mid = (l + h) >> 1;
                if (comb_gt(n, cdf[mid] - base, rhs_hi, rhs_lo)) h = mid;
                else l = mid + 1;
            }
            anc = a.perm[l];
            if (p == lo && a.seg_status_out) a.seg_status_out[seg] = 0;
        }
        anc_s[tid] = anc;
        dst_s[tid] = i;
        if (a.ancestors_out) a.ancestors_out[i] = anc;
        if (a.weights_out) a.weights_out[i] = 1.0f / (float)n;
    }
    __syncthreads();
    if (a.particles_out) {
        typedef typename std::conditional<VEC == 16, uint4, typename std::conditional<VEC == 8, uint2, typename std::conditional<VEC == 4, uint32_t, uint16_t>::type>::type>::type V;
        const int cpr = row_bytes / VEC;
        const uint8_t *src = reinterpret_cast<const uint8_t *>(a.proposals);
        uint8_t *dst = reinterpret_cast<uint8_t *>(a.particles_out);
        for (int c = tid; c < rows * cpr; c += 256) {
            const int j = c / cpr, off = c - j * cpr;
            const V val = *reinterpret_cast<const V *>(src + (size_t)anc_s[j] * row_bytes + (size_t)off * VEC);
            *reinterpret_cast<V *>(dst + (size_t)dst_s[j] * row_bytes + (size_t)off * VEC) = val;
        }
    }
}

// child status of EMPTY children (no member this batch): 0
__global__ void pw_clear_status_kernel(int32_t *st, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) st[i] = 0;
}

}  // namespace

cudaError_t launch_pw_widen(const PwArgs &a, cudaStream_t st) {
    pw_widen_kernel<<<(a.G + kWidenWarps - 1) / kWidenWarps, kWidenWarps * 32, 0, st>>>(a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    pw_seg_scan_kernel<<<1, 1024, 0, st>>>(a.seg_count, a.G * a.M_max, a.seg_off);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    pw_perm_kernel<<<(a.N + 255) / 256, 256, 0, st>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_pw_weights(const PwArgs &a, cudaStream_t st) {
    pw_weights_kernel<<<(a.N + 255) / 256, 256, 0, st>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_pw_resample(const PwArgs &a, const unsigned long long *cdf, int row_bytes, cudaStream_t st) {
    if (a.seg_status_out) {
        const int n = a.G * a.M_max;
        pw_clear_status_kernel<<<(n + 255) / 256, 256, 0, st>>>(a.seg_status_out, n);
    }
    const int grid = (a.N + 255) / 256;
    if (row_bytes % 16 == 0) pw_resample_kernel<16><<<grid, 256, 0, st>>>(a, cdf, row_bytes);
    else if (row_bytes % 8 == 0) pw_resample_kernel<8><<<grid, 256, 0, st>>>(a, cdf, row_bytes);
    else if (row_bytes % 4 == 0) pw_resample_kernel<4><<<grid, 256, 0, st>>>(a, cdf, row_bytes);
    else pw_resample_kernel<2><<<grid, 256, 0, st>>>(a, cdf, row_bytes);
    return cudaGetLastError();
}

}  // namespace voila
