// mlp_ffma.cu -- CUDA-core path of libvoila: the fp32 parity mode (north_star: relative 1e-4)
// and a dims-agnostic bf16 mode (operands rounded to bf16, fp32 accumulate) used when the model
// does not fit the tcgen05 kernels.
//
// One CTA = one tile of kTileRows particles of ONE action sequence, so the one-hot action block of
// the generator input is the same for every row of the tile: it is never multiplied, the column
// W1[:, S + a_t] is added instead (same sum, same order as the
// definition since 0*w contributes exactly 0).  Activations live in shared memory transposed
// ([k][row]) so a thread reads 16 rows of one k with four 128-bit loads; weights are stored
// transposed ([k][j]) so lanes read consecutive output neurons j.  The horizon loop never touches
// HBM except for weights (L2-resident).
#include "voila_device.cuh"
#include "voila_kernels.h"

namespace voila {

namespace {

constexpr int R = kTileRows;  // 32
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

// y[j][r] = act(sum_k Wt[k][j] x[k][r] + b[j]) for the tile's R rows.
// Rows k in [skip_lo, skip_hi) of the input are skipped (the one-hot block) and row a_row of Wt is
// added in their place (a_row < 0: nothing added).
// RPT rows per thread: 16 (two threads per neuron) for wide layers; 8 (four threads per neuron) when a
// layer has fewer than kThreads / 2 neurons (config 1's 64-wide layers left half the CTA idle).
template <bool EMU, int RPT>
__device__ __forceinline__ void mlp_layer_rpt(const float *__restrict__ Wt, const float *__restrict__ bias,
                                              int K, int N, int act, bool last, const float *xin,
                                              float *xout, int skip_lo, int skip_hi, int a_row) {
    constexpr int kParts = R / RPT;
    for (int item = threadIdx.x; item < kParts * N; item += kThreads) {
        const int part = item / N, j = item - part * N;
        // accumulators as fp32 PAIRS: sm_100's packed FFMA2 (fma.rn.f32x2) does two rows per instruction,
        // each component an ordinary IEEE fma (the same bits as two fmaf)
        float2 acc2[RPT / 2];
#pragma unroll
        for (int i = 0; i < RPT / 2; ++i) acc2[i] = make_float2(0.0f, 0.0f);
        const float *xp = xin + RPT * part;
        auto fma_row = [&](int k) {
            const float w = __ldg(Wt + (size_t)k * N + j);
            const float2 w2 = make_float2(w, w);
            const float4 *x4 = reinterpret_cast<const float4 *>(xp + k * R);
#pragma unroll
            for (int v = 0; v < RPT / 4; ++v) {
                const float4 x = x4[v];
                acc2[2 * v] = __ffma2_rn(w2, make_float2(x.x, x.y), acc2[2 * v]);
                acc2[2 * v + 1] = __ffma2_rn(w2, make_float2(x.z, x.w), acc2[2 * v + 1]);
            }
        };
        const int k_end0 = skip_lo < K ? skip_lo : K;
#pragma unroll 4
        for (int k = 0; k < k_end0; ++k) fma_row(k);
        if (a_row >= 0) {
            const float w = __ldg(Wt + (size_t)a_row * N + j);
#pragma unroll
            for (int i = 0; i < RPT / 2; ++i) {
                acc2[i].x += w;
                acc2[i].y += w;
            }
        }
#pragma unroll 4
        for (int k = skip_hi; k < K; ++k) fma_row(k);
        const float bj = __ldg(bias + j);
        float4 *o4 = reinterpret_cast<float4 *>(xout + j * R + RPT * part);
#pragma unroll
        for (int v = 0; v < RPT / 4; ++v) {
            float y[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float2 a2 = acc2[2 * v + (i >> 1)];
                float t = ((i & 1) ? a2.y : a2.x) + bj;
                if (!last) {
                    t = act_apply(t, act);
                    if (EMU) t = bf16_round(t);  // the next layer's operand is bf16
                }
                y[i] = t;
            }
            o4[v] = make_float4(y[0], y[1], y[2], y[3]);
        }
    }
}
template <bool EMU>
__device__ __forceinline__ void mlp_layer(const float *__restrict__ Wt, const float *__restrict__ bias,
                                          int K, int N, int act, bool last, const float *xin,
                                          float *xout, int skip_lo, int skip_hi, int a_row) {
    // (same sums in the same order either way: a row's accumulation never crosses threads)
    if (2 * N < kThreads) mlp_layer_rpt<EMU, 8>(Wt, bias, K, N, act, last, xin, xout, skip_lo, skip_hi, a_row);
    else mlp_layer_rpt<EMU, 16>(Wt, bias, K, N, act, last, xin, xout, skip_lo, skip_hi, a_row);
}

// Input in bufA ([dims[0]][R]); hidden activations ping-pong bufB/bufA; the last layer writes out.
template <bool EMU>
__device__ __forceinline__ void mlp_chain(const MlpDev &f, float *bufA, float *bufB, float *out,
                                          int skip_lo, int skip_hi, int a_row) {
    float *in = bufA, *other = bufB;
    for (int l = 0; l < f.n_layers; ++l) {
        const bool last = (l == f.n_layers - 1);
        float *dst = last ? out : other;
        const int K = f.dims[l];
        mlp_layer<EMU>(f.Wt[l], f.b[l], K, f.dims[l + 1], f.act, last, in, dst,
                       l == 0 ? skip_lo : K, l == 0 ? skip_hi : K, l == 0 ? a_row : -1);
        __syncthreads();
        other = in;
        in = dst;
    }
}

// x[(base + j)][r] = j-th standard normal of (seed; p0 + r, q, t, stream) for j < Nz.
template <bool EMU>
__device__ __forceinline__ void fill_noise(float *x, int base, int Nz, uint64_t seed, uint32_t p0,
                                           uint32_t q, uint32_t t, uint32_t stream) {
    const int nblk = (Nz + 3) >> 2;
    for (int idx = threadIdx.x; idx < R * nblk; idx += kThreads) {
        const int r = idx & (R - 1), blk = idx / R;
        float z[4];
        normals4<false>(seed, p0 + r, q, t, stream, blk, z);
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (4 * blk + i < Nz) x[(base + 4 * blk + i) * R + r] = EMU ? bf16_round(z[i]) : z[i];
    }
}

template <bool EMU>
__device__ __forceinline__ void copy_state(float *x, const float *s, int S) {
    for (int idx = threadIdx.x; idx < S * R; idx += kThreads) x[idx] = EMU ? bf16_round(s[idx]) : s[idx];
}

// R(s, a) for the tile's rows, warps splitting the state index; result (before discounting) is
// returned by warp 0's lanes (lane = row).  red = [kWarps][R] scratch.
__device__ __forceinline__ float tile_reward(const RewardDev &rw, int S, const float *s, int a,
                                             float *red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float part = 0.0f;
    if (rw.kind == VOILA_R_NEG_L2_GOAL) {
        for (int i = warp; i < S; i += kWarps) {
            const float d = s[i * R + lane] - __ldg(rw.param + i);
            part = fmaf(d, d, part);
        }
    } else if (rw.kind == VOILA_R_NEG_QUADRATIC) {
        for (int i = warp; i < S; i += kWarps) {
            float row = 0.0f;
            for (int j = 0; j < S; ++j) row = fmaf(__ldg(rw.param + i * S + j), s[j * R + lane], row);
            part = fmaf(s[i * R + lane], row, part);
        }
    } else {
        for (int i = warp; i < S; i += kWarps) part = fmaf(__ldg(rw.param + i), s[i * R + lane], part);
    }
    red[warp * R + lane] = part;
    __syncthreads();
    float r = 0.0f;
    if (warp == 0) {
        float tot = 0.0f;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) tot += red[w * R + lane];
        if (rw.kind == VOILA_R_NEG_L2_GOAL) r = -sqrtf(tot);
        else if (rw.kind == VOILA_R_NEG_QUADRATIC) r = -tot;
        else r = tot + __ldg(rw.param + S);
        if (rw.action_cost) r += __ldg(rw.action_cost + a);
    }
    return r;
}

template <bool EMU>
__device__ __forceinline__ void load_particles(const void *particles, int S, int n_rows_total,
                                               int row0, float *s) {
    for (int idx = threadIdx.x; idx < S * R; idx += kThreads) {
        const int r = idx / S, i = idx - r * S;
        float v = 0.0f;
        if (row0 + r < n_rows_total) {
            const size_t g = (size_t)(row0 + r) * S + i;
            v = EMU ? bf16_to_float(reinterpret_cast<const uint16_t *>(particles)[g])
                    : reinterpret_cast<const float *>(particles)[g];
        }
        s[i * R + r] = v;
    }
}

__device__ __forceinline__ double warp_sum_double(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <bool EMU>
__global__ void __launch_bounds__(kThreads) rollout_ffma_kernel(const ModelDev m, const RolloutArgs a) {
    extern __shared__ __align__(16) float smem[];
    const int S = m.S, O = m.O, A = m.A, Nz = m.Nz, KW = m.max_width;
    float *xa = smem, *xb = xa + KW * R, *s = xb + KW * R, *sn = s + S * R, *wit = sn + S * R;
    float *obs = wit + O * R, *red = obs + O * R, *G = red + kWarps * R;
    float *alive = G + R;  // 1 while the row's episode runs (terminal regions, voila_terminal)
    const int tile = blockIdx.y, q = blockIdx.x, p0 = tile * R;  // q on x: no 65535 limit on the sequences
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    load_particles<EMU>(a.particles, S, a.P, p0, s);
    for (int idx = threadIdx.x; idx < O * R; idx += kThreads) wit[idx] = 0.0f;
    if (threadIdx.x < R) {
        G[threadIdx.x] = 0.0f;
        alive[threadIdx.x] = 1.0f;
    }
    __syncthreads();

    float disc = 1.0f;
    for (int t = 0; t < a.H; ++t) {
        const int act_t = clamp_action(__ldg(a.action_seqs + (size_t)q * a.H + t), A);
        // reward on the CURRENT state (reading R7)
        const float rew = tile_reward(m.reward, S, s, act_t, red);
        if (warp == 0) {
            // terminal regions (reading R25): every region holding s_t pays; a stopping one ends the
            // episode here (no step reward, state frozen, nothing accrues afterwards)
            float bonus = 0.0f;
            bool stop = false;
            for (int k = 0; k < m.term.n; ++k) {
                float d2 = 0.0f;
                for (int j = 0; j < m.term.dim[k]; ++j) {
                    const float sj = EMU ? bf16_round(s[j * R + lane]) : s[j * R + lane];
                    const float d = sj - __ldg(m.term.centers + m.term.off[k] + j);
                    d2 = fmaf(d, d, d2);
                }
                if (d2 <= m.term.r2[k]) {
                    bonus += m.term.reward[k];
                    stop |= m.term.stop[k] != 0;
                }
            }
            if (alive[lane] != 0.0f) {
                G[lane] = fmaf(disc, stop ? bonus : bonus + rew, G[lane]);
                if (stop) alive[lane] = 0.0f;
            }
        }
        // s' = f_T([s ; onehot(a) ; w_T])
        copy_state<EMU>(xa, s, S);
        fill_noise<EMU>(xa, S + A, Nz, a.seed, p0, q, t, kStreamRolloutT);
        __syncthreads();
        mlp_chain<EMU>(m.mlp[0], xa, xb, sn, S, S + A, S + act_t);
        // o = f_Z([s' ; onehot(a) ; w_Z])
        copy_state<EMU>(xa, sn, S);
        fill_noise<EMU>(xa, S + A, Nz, a.seed, p0, q, t, kStreamRolloutZ);
        __syncthreads();
        mlp_chain<EMU>(m.mlp[1], xa, xb, obs, S, S + A, S + act_t);
        // rows whose episode has ended take no step: no observation, state frozen
        for (int idx = threadIdx.x; idx < O * R; idx += kThreads)
            if (alive[idx & (R - 1)] != 0.0f) wit[idx] = fmaf(disc, obs[idx], wit[idx]);
        for (int idx = threadIdx.x; idx < S * R; idx += kThreads)
            if (alive[idx & (R - 1)] != 0.0f) s[idx] = sn[idx];
        disc *= m.gamma;
        __syncthreads();
    }

    // weighted partial sums for this (q, tile); fixed order => bit-reproducible
    const bool valid = (p0 + lane) < a.P;
    const float wl = valid ? (a.weights ? __ldg(a.weights + p0 + lane) : 1.0f) : 0.0f;
    if (warp == 0) {
        const double v = warp_sum_double((double)wl * (double)G[lane]);
        if (lane == 0) a.part_value[(size_t)q * a.tiles + tile] = v;
        if (a.returns_out && valid) a.returns_out[(size_t)q * a.P + p0 + lane] = G[lane];
        red[lane] = wl;
    }
    __syncthreads();
    if (a.part_witness) {
        for (int i = threadIdx.x; i < O; i += kThreads) {
            double acc = 0.0;
            for (int r = 0; r < R; ++r) acc += (double)red[r] * (double)wit[i * R + r];
            a.part_witness[((size_t)q * a.tiles + tile) * O + i] = acc;
        }
    }
    if (a.final_states_out) {
        for (int idx = threadIdx.x; idx < S * R; idx += kThreads) {
            const int r = idx / S, i = idx - r * S;
            if (p0 + r < a.P) a.final_states_out[((size_t)q * a.P + p0 + r) * S + i] = s[i * R + r];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Progressive widening (voila_pw_update): the MLP stages on the CUDA cores.
// Every row carries its own action (simulations of different action nodes share a tile), so the
// one-hot block is part of the operand here (same sum: the zeros contribute exactly 0 and the block
// sits between the state and the noise rows, where the folded form adds its weight row).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void fill_onehot(float *x, int base, int A, const int *act_row) {
    for (int idx = threadIdx.x; idx < A * R; idx += kThreads) {
        const int r = idx & (R - 1), k = idx / R;
        x[(base + k) * R + r] = (k == act_row[r]) ? 1.0f : 0.0f;
    }
}
template <bool EMU>
__device__ __forceinline__ void load_rows(const void *rows_in, int S, const int *src_row, float *x) {
    for (int idx = threadIdx.x; idx < S * R; idx += kThreads) {
        const int r = idx / S, i = idx - r * S;
        float v = 0.0f;
        if (src_row[r] >= 0) {
            const size_t g = (size_t)src_row[r] * S + i;
            v = EMU ? bf16_to_float(reinterpret_cast<const uint16_t *>(rows_in)[g])
                    : reinterpret_cast<const float *>(rows_in)[g];
        }
        x[i * R + r] = v;
    }
}

// s'_i = f_T(s_i, a_g(i), w_T(i)): stream 3, counter (i, 0, 0), as the belief update draws it.
template <bool EMU>
__global__ void __launch_bounds__(kThreads) pw_propose_ffma_kernel(const ModelDev m, const PwArgs a) {
    extern __shared__ __align__(16) float smem[];
    __shared__ int act_row[R], src_row[R];
    const int S = m.S, A = m.A, Nz = m.Nz, KW = m.max_width;
    float *xa = smem, *xb = xa + KW * R, *sn = xb + KW * R;
    const int i0 = blockIdx.x * R;
    if (threadIdx.x < R) {
        const int i = i0 + threadIdx.x;
        src_row[threadIdx.x] = i < a.N ? i : -1;
        act_row[threadIdx.x] = i < a.N ? __ldg(a.group_action + a.sim_group[i]) : 0;
    }
    __syncthreads();
    load_rows<EMU>(a.particles, S, src_row, xa);
    fill_onehot(xa, S, A, act_row);
    fill_noise<EMU>(xa, S + A, Nz, a.seed, i0, 0u, 0u, kStreamBeliefT);
    __syncthreads();
    const int K0 = S + A + Nz;
    mlp_chain<EMU>(m.mlp[0], xa, xb, sn, K0, K0, -1);
    for (int idx = threadIdx.x; idx < S * R; idx += kThreads) {
        const int r = idx / S, i = idx - r * S;
        if (i0 + r < a.N) {
            const float v = sn[i * R + r];
            const size_t gidx = (size_t)(i0 + r) * S + i;
            if (EMU) reinterpret_cast<uint16_t *>(a.proposals)[gidx] = bf16_bits(v);
            else reinterpret_cast<float *>(a.proposals)[gidx] = v;
        }
    }
}

// o_i = f_Z(s'_i, a, w_Z(i)) (stream 5) for the simulations that opened a branch: one row per
// (action node, branch) slot, stored as the branch's observation.
template <bool EMU>
__global__ void __launch_bounds__(kThreads) pw_obs_ffma_kernel(const ModelDev m, const PwArgs a) {
    extern __shared__ __align__(16) float smem[];
    __shared__ int act_row[R], src_row[R];
    const int S = m.S, O = m.O, A = m.A, Nz = m.Nz, KW = m.max_width;
    float *xa = smem, *xb = xa + KW * R, *out = xb + KW * R;
    const int gm0 = blockIdx.x * R, n_slots = a.G * a.M_max;
    if (threadIdx.x < R) {
        const int gm = gm0 + threadIdx.x;
        src_row[threadIdx.x] = gm < n_slots ? a.new_src[gm] : -1;
        act_row[threadIdx.x] = gm < n_slots ? __ldg(a.group_action + gm / a.M_max) : 0;
    }
    __syncthreads();
    bool any = false;
    for (int r = 0; r < R; ++r) any |= src_row[r] >= 0;
    if (!any) return;  // uniform: no branch was opened in this tile of slots
    const int nblk = (Nz + 3) >> 2;
    if (a.obs_from_particles) {
        // the tensor-core pass that stores the proposals runs later: s' of these few rows here
        load_rows<EMU>(a.particles, S, src_row, xa);
        fill_onehot(xa, S, A, act_row);
        for (int idx = threadIdx.x; idx < R * nblk; idx += kThreads) {
            const int r = idx & (R - 1), blk = idx / R;
            float z[4];
            normals4<false>(a.seed, (uint32_t)max(src_row[r], 0), 0u, 0u, kStreamBeliefT, (uint32_t)blk, z);
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (4 * blk + i < Nz) xa[(S + A + 4 * blk + i) * R + r] = EMU ? bf16_round(z[i]) : z[i];
        }
        __syncthreads();
        mlp_chain<EMU>(m.mlp[0], xa, xb, out, S + A + Nz, S + A + Nz, -1);
        copy_state<EMU>(xa, out, S);
        __syncthreads();
    } else {
        load_rows<EMU>(a.proposals, S, src_row, xa);
    }
    fill_onehot(xa, S, A, act_row);
    for (int idx = threadIdx.x; idx < R * nblk; idx += kThreads) {
        const int r = idx & (R - 1), blk = idx / R;
        float z[4];
        normals4<false>(a.seed, (uint32_t)max(src_row[r], 0), 0u, 0u, kStreamPwObs, (uint32_t)blk, z);
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (4 * blk + i < Nz) xa[(S + A + 4 * blk + i) * R + r] = EMU ? bf16_round(z[i]) : z[i];
    }
    __syncthreads();
    const int K0 = S + A + Nz;
    mlp_chain<EMU>(m.mlp[1], xa, xb, out, K0, K0, -1);
    for (int idx = threadIdx.x; idx < O * R; idx += kThreads) {
        const int r = idx / O, k = idx - r * O;
        if (src_row[r] >= 0) a.branch_obs[(size_t)(gm0 + r) * O + k] = out[k * R + r];
    }
}

// L_i = log w_i + <e_{g, b(i)}, g(s'_i [; onehot(a)])> / lambda and the running maximum of its child.
template <bool EMU>
__global__ void __launch_bounds__(kThreads) pw_score_ffma_kernel(const ModelDev m, const PwArgs a) {
    extern __shared__ __align__(16) float smem[];
    __shared__ int act_row[R], src_row[R];
    const int S = m.S, A = m.A, KW = m.max_width;
    const MlpDev &g = m.mlp[3];
    const int d = g.dims[g.n_layers];
    float *xa = smem, *xb = xa + KW * R, *gout = xb + KW * R;
    const int i0 = blockIdx.x * R;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x < R) {
        const int i = i0 + threadIdx.x;
        src_row[threadIdx.x] = i < a.N ? i : -1;
        act_row[threadIdx.x] = i < a.N ? __ldg(a.group_action + a.sim_group[i]) : 0;
    }
    __syncthreads();
    load_rows<EMU>(a.proposals, S, src_row, xa);
    if (m.lik_action_cond) fill_onehot(xa, S, A, act_row);
    __syncthreads();
    const int K0 = S + (m.lik_action_cond ? A : 0);
    mlp_chain<EMU>(g, xa, xb, gout, K0, K0, -1);
    if (warp == 0) {
        const int i = i0 + lane;
        if (i < a.N) {
            const int seg = a.sim_group[i] * a.M_max + a.sim_branch[i];
            const float *e = a.E + (size_t)seg * d;
            float ell = 0.0f;
            for (int k = 0; k < d; ++k) ell += __ldg(e + k) * gout[k * R + lane];
            float lw = 0.0f;
            if (a.weights) {
                const float w = __ldg(a.weights + i);
                lw = w > 0.0f ? logf(w) : -INFINITY;
            }
            const float L = lw + ell / m.lambda;
            a.logits[i] = L;
            atomicMax(a.seg_max + seg, float_to_ordered(L));
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Diffusion teacher (voila_diffusion_sample): one DDIM-ODE step = one call of the
// denoiser v(c, a, x, tau_k) on [c ; onehot(a) ; x ; temb(tau_k)] and the v-prediction update.
// ---------------------------------------------------------------------------------------------
template <bool EMU>
__global__ void __launch_bounds__(kThreads) diffusion_step_ffma_kernel(const ModelDev m, const DiffusionArgs a) {
    extern __shared__ __align__(16) float smem[];
    __shared__ int act_row[R], src_row[R];
    const int S = m.S, A = m.A, D = a.D, KW = m.max_width;
    const MlpDev &f = m.mlp[4 + a.which];
    float *xa = smem, *xb = xa + KW * R, *v = xb + KW * R, *xs = v + D * R;  // xs: the fp32 state [D][R]
    const int i0 = blockIdx.x * R;
    if (threadIdx.x < R) {
        const int i = i0 + threadIdx.x;
        src_row[threadIdx.x] = i < a.N ? i : -1;
        act_row[threadIdx.x] = i < a.N ? __ldg(a.actions + i) : 0;
    }
    __syncthreads();
    load_rows<EMU>(a.cond, S, src_row, xa);
    fill_onehot(xa, S, A, act_row);
    if (a.first) {
        const int nblk = (D + 3) >> 2;
        for (int idx = threadIdx.x; idx < R * nblk; idx += kThreads) {
            const int r = idx & (R - 1), blk = idx / R;
            float z[4];
            normals4<false>(a.seed, (uint32_t)(i0 + r), 0u, 0u, kStreamDiffusion, (uint32_t)blk, z);
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (4 * blk + i < D) xs[(4 * blk + i) * R + r] = z[i];
        }
    } else {
        for (int idx = threadIdx.x; idx < D * R; idx += kThreads) {
            const int r = idx / D, j = idx - r * D;
            xs[j * R + r] = (i0 + r < a.N) ? a.x[(size_t)(i0 + r) * D + j] : 0.0f;
        }
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < D * R; idx += kThreads)
        xa[(S + A) * R + idx] = EMU ? bf16_round(xs[idx]) : xs[idx];
    for (int idx = threadIdx.x; idx < kTemb * R; idx += kThreads) {
        const float t = a.temb[idx / R];
        xa[(S + A + D) * R + idx] = EMU ? bf16_round(t) : t;
    }
    __syncthreads();
    const int K0 = S + A + D + kTemb;
    mlp_chain<EMU>(f, xa, xb, v, K0, K0, -1);
    for (int idx = threadIdx.x; idx < D * R; idx += kThreads) {
        const int r = idx / D, j = idx - r * D;
        if (i0 + r < a.N) {
            const float x = xs[j * R + r], vv = v[j * R + r];
            const float x0_hat = a.al * x - a.si * vv;   // v-prediction
            const float eps_hat = a.si * x + a.al * vv;
            a.x[(size_t)(i0 + r) * D + j] = a.al_n * x0_hat + a.si_n * eps_hat;  // DDIM, eta = 0
        }
    }
}

__global__ void weight_sum_kernel(const float *__restrict__ w, int n, double *out) {
    __shared__ double sh[256];
    double acc = 0.0;
    if (w) {
        for (int i = threadIdx.x; i < n; i += 256) acc += (double)w[i];
    } else if (threadIdx.x == 0) {
        acc = (double)n;
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}

__global__ void rollout_reduce_kernel(const double *__restrict__ part_value,
                                      const double *__restrict__ part_witness, int tiles, int O,
                                      const double *__restrict__ wsum, float *values, float *witness) {
    const int q = blockIdx.x;
    const double inv = 1.0 / *wsum;
    for (int i = threadIdx.x; i < O + 1; i += blockDim.x) {
        double acc = 0.0;
        if (i == O) {
            for (int t = 0; t < tiles; ++t) acc += part_value[(size_t)q * tiles + t];
            values[q] = (float)(acc * inv);
        } else if (witness) {
            for (int t = 0; t < tiles; ++t) acc += part_witness[((size_t)q * tiles + t) * O + i];
            witness[(size_t)q * O + i] = (float)(acc * inv);
        }
    }
}

// q* = argmax_q values[q], ties -> lowest q, NaN never wins; one block.
__global__ void __launch_bounds__(256) best_action_kernel(const float *__restrict__ values,
                                                          const int32_t *__restrict__ seqs, int Q, int H,
                                                          int32_t *best_q, int32_t *best_action) {
    __shared__ float sv[256];
    __shared__ int si[256];
    float bv = -INFINITY;
    int bi = 0x7fffffff;
    for (int q = threadIdx.x; q < Q; q += 256) {
        const float v = values[q];
        if (v == v && (bi == 0x7fffffff || v > bv)) {  // q ascends per thread: strict > keeps the lowest
            bv = v;
            bi = q;
        }
    }
    sv[threadIdx.x] = bv;
    si[threadIdx.x] = bi;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            const float v = sv[threadIdx.x + o];
            const int i = si[threadIdx.x + o];
            if (i != 0x7fffffff && (si[threadIdx.x] == 0x7fffffff || v > sv[threadIdx.x] ||
                                    (v == sv[threadIdx.x] && i < si[threadIdx.x]))) {
                sv[threadIdx.x] = v;
                si[threadIdx.x] = i;
            }
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const int q = si[0] == 0x7fffffff ? 0 : si[0];  // every value NaN: sequence 0
        if (best_q) *best_q = q;
        *best_action = seqs[(size_t)q * H];
    }
}

template <bool EMU>
__global__ void __launch_bounds__(kThreads) mlp_forward_ffma_kernel(const ModelDev m, int which,
                                                                    const float *__restrict__ x,
                                                                    int rows, float *y) {
    extern __shared__ __align__(16) float smem[];
    const MlpDev &f = m.mlp[which];
    const int KW = m.max_width, K0 = f.dims[0], NL = f.dims[f.n_layers];
    float *xa = smem, *xb = xa + KW * R, *out = xb + KW * R;
    const int row0 = blockIdx.x * R;
    for (int idx = threadIdx.x; idx < K0 * R; idx += kThreads) {
        const int r = idx / K0, k = idx - r * K0;
        float v = (row0 + r < rows) ? x[(size_t)(row0 + r) * K0 + k] : 0.0f;
        xa[k * R + r] = EMU ? bf16_round(v) : v;
    }
    __syncthreads();
    mlp_chain<EMU>(f, xa, xb, out, K0, K0, -1);
    for (int idx = threadIdx.x; idx < NL * R; idx += kThreads) {
        const int r = idx / NL, j = idx - r * NL;
        if (row0 + r < rows) y[(size_t)(row0 + r) * NL + j] = out[j * R + r];
    }
}

// Belief update, stage 1 (O5): proposal s' = f_T(s, a, w), score L = log w + <e, g(s')>/lambda.
template <bool EMU>
__global__ void __launch_bounds__(kThreads) bu_propose_score_ffma_kernel(const ModelDev m,
                                                                         const BeliefArgs a) {
    extern __shared__ __align__(16) float smem[];
    const int S = m.S, A = m.A, Nz = m.Nz, KW = m.max_width;
    const MlpDev &g = m.mlp[3];
    const int d = g.dims[g.n_layers];
    float *xa = smem, *xb = xa + KW * R, *s = xb + KW * R, *sn = s + S * R, *gout = sn + S * R;
    const int i0 = blockIdx.x * R;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    load_particles<EMU>(a.particles, S, a.N, i0, s);
    __syncthreads();
    copy_state<EMU>(xa, s, S);
    fill_noise<EMU>(xa, S + A, Nz, a.seed, i0, 0u, 0u, kStreamBeliefT);
    __syncthreads();
    mlp_chain<EMU>(m.mlp[0], xa, xb, sn, S, S + A, S + a.action);
    // the stored particle is what the filter carries forward: in bf16 mode it is bf16(s')
    for (int idx = threadIdx.x; idx < S * R; idx += kThreads) {
        const int r = idx / S, i = idx - r * S;
        if (i0 + r < a.N) {
            const float v = sn[i * R + r];
            const size_t gidx = (size_t)(i0 + r) * S + i;
            if (EMU) reinterpret_cast<uint16_t *>(a.proposals)[gidx] = bf16_bits(v);
            else reinterpret_cast<float *>(a.proposals)[gidx] = v;
        }
    }
    copy_state<EMU>(xa, sn, S);
    __syncthreads();
    if (m.lik_action_cond) mlp_chain<EMU>(g, xa, xb, gout, S, S + A, S + a.action);
    else mlp_chain<EMU>(g, xa, xb, gout, S, S, -1);
    if (warp == 0) {
        float ell = 0.0f;
        for (int k = 0; k < d; ++k) ell += __ldg(a.e + k) * gout[k * R + lane];
        const bool valid = (i0 + lane) < a.N;
        float w = 1.0f, lw = 0.0f;
        if (a.weights) {
            w = valid ? __ldg(a.weights + i0 + lane) : 0.0f;
            lw = w > 0.0f ? logf(w) : -INFINITY;
        }
        const float L = lw + ell / m.lambda;
        int ord = float_to_ordered(valid ? L : -INFINITY);
        if (valid) a.logits[i0 + lane] = L;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ord = max(ord, __shfl_xor_sync(0xffffffffu, ord, o));
        const double ws = warp_sum_double(valid ? (double)w : 0.0);
        if (lane == 0) {
            atomicMax(a.max_ordered, ord);
            a.part_wsum[blockIdx.x] = ws;
        }
    }
}

template <typename K>
cudaError_t set_smem(K kernel, size_t bytes) {
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

}  // namespace

size_t ffma_smem_bytes(const ModelDev &m) {
    const int d = m.mlp[3].dims[m.mlp[3].n_layers];
    const size_t rollout = (size_t)(2 * m.max_width + 2 * m.S + 2 * m.O + kWarps + 2) * R * sizeof(float);
    const size_t belief = (size_t)(2 * m.max_width + 2 * m.S + d) * R * sizeof(float);
    const size_t fwd = (size_t)(3 * m.max_width) * R * sizeof(float);
    const size_t diffusion = (size_t)(2 * m.max_width + 2 * (m.S > m.O ? m.S : m.O)) * R * sizeof(float);
    size_t b = rollout > belief ? rollout : belief;
    b = b > fwd ? b : fwd;
    return b > diffusion ? b : diffusion;
}

template <typename K>
static cudaError_t pw_launch(K kernel, int grid, const ModelDev &m, const PwArgs &a, cudaStream_t st) {
    const size_t smem = ffma_smem_bytes(m);
    cudaError_t e;
    if ((e = set_smem(kernel, smem)) != cudaSuccess) return e;
    kernel<<<grid, kThreads, smem, st>>>(m, a);
    return cudaGetLastError();
}
cudaError_t launch_pw_propose_ffma(const ModelDev &m, const PwArgs &a, bool bf16, cudaStream_t st) {
    const int grid = (a.N + R - 1) / R;
    return bf16 ? pw_launch(pw_propose_ffma_kernel<true>, grid, m, a, st)
                : pw_launch(pw_propose_ffma_kernel<false>, grid, m, a, st);
}
cudaError_t launch_pw_obs_ffma(const ModelDev &m, const PwArgs &a, bool bf16, cudaStream_t st) {
    const int grid = (a.G * a.M_max + R - 1) / R;
    return bf16 ? pw_launch(pw_obs_ffma_kernel<true>, grid, m, a, st)
                : pw_launch(pw_obs_ffma_kernel<false>, grid, m, a, st);
}
cudaError_t launch_pw_score_ffma(const ModelDev &m, const PwArgs &a, bool bf16, cudaStream_t st) {
    const int grid = (a.N + R - 1) / R;
    return bf16 ? pw_launch(pw_score_ffma_kernel<true>, grid, m, a, st)
                : pw_launch(pw_score_ffma_kernel<false>, grid, m, a, st);
}

cudaError_t launch_diffusion_step_ffma(const ModelDev &m, const DiffusionArgs &a, bool bf16, cudaStream_t st) {
    const size_t smem = ffma_smem_bytes(m);
    const int grid = (a.N + R - 1) / R;
    cudaError_t e;
    if (bf16) {
        if ((e = set_smem(diffusion_step_ffma_kernel<true>, smem)) != cudaSuccess) return e;
        diffusion_step_ffma_kernel<true><<<grid, kThreads, smem, st>>>(m, a);
    } else {
        if ((e = set_smem(diffusion_step_ffma_kernel<false>, smem)) != cudaSuccess) return e;
        diffusion_step_ffma_kernel<false><<<grid, kThreads, smem, st>>>(m, a);
    }
    return cudaGetLastError();
}

cudaError_t launch_weight_sum(const float *weights, int n, double *wsum_out, cudaStream_t st) {
    weight_sum_kernel<<<1, 256, 0, st>>>(weights, n, wsum_out);
    return cudaGetLastError();
}

cudaError_t launch_rollout_ffma(const ModelDev &m, const RolloutArgs &a, bool bf16, cudaStream_t st) {
    const size_t smem = ffma_smem_bytes(m);
    dim3 grid(a.Q, a.tiles);
    cudaError_t e;
    if (bf16) {
        if ((e = set_smem(rollout_ffma_kernel<true>, smem)) != cudaSuccess) return e;
        rollout_ffma_kernel<true><<<grid, kThreads, smem, st>>>(m, a);
    } else {
        if ((e = set_smem(rollout_ffma_kernel<false>, smem)) != cudaSuccess) return e;
        rollout_ffma_kernel<false><<<grid, kThreads, smem, st>>>(m, a);
    }
    return cudaGetLastError();
}

cudaError_t launch_rollout_reduce(const RolloutArgs &a, int O, const double *wsum, float *values,
                                  float *witness, cudaStream_t st) {
    rollout_reduce_kernel<<<a.Q, 128, 0, st>>>(a.part_value, witness ? a.part_witness : nullptr,
                                               a.tiles, O, wsum, values, witness);
    return cudaGetLastError();
}

cudaError_t launch_best_action(const float *values, const int32_t *seqs, int Q, int H, int32_t *best_q,
                               int32_t *best_action, cudaStream_t st) {
    best_action_kernel<<<1, 256, 0, st>>>(values, seqs, Q, H, best_q, best_action);
    return cudaGetLastError();
}

cudaError_t launch_mlp_forward_ffma(const ModelDev &m, int which, const float *x, int rows, float *y,
                                    bool bf16, cudaStream_t st) {
    const size_t smem = ffma_smem_bytes(m);
    const int grid = (rows + R - 1) / R;
    cudaError_t e;
    if (bf16) {
        if ((e = set_smem(mlp_forward_ffma_kernel<true>, smem)) != cudaSuccess) return e;
        mlp_forward_ffma_kernel<true><<<grid, kThreads, smem, st>>>(m, which, x, rows, y);
    } else {
        if ((e = set_smem(mlp_forward_ffma_kernel<false>, smem)) != cudaSuccess) return e;
        mlp_forward_ffma_kernel<false><<<grid, kThreads, smem, st>>>(m, which, x, rows, y);
    }
    return cudaGetLastError();
}

cudaError_t launch_bu_propose_score_ffma(const ModelDev &m, const BeliefArgs &a, bool bf16,
                                         cudaStream_t st) {
    const size_t smem = ffma_smem_bytes(m);
    const int grid = (a.N + R - 1) / R;
    cudaError_t e;
    if (bf16) {
        if ((e = set_smem(bu_propose_score_ffma_kernel<true>, smem)) != cudaSuccess) return e;
        bu_propose_score_ffma_kernel<true><<<grid, kThreads, smem, st>>>(m, a);
    } else {
        if ((e = set_smem(bu_propose_score_ffma_kernel<false>, smem)) != cudaSuccess) return e;
        bu_propose_score_ffma_kernel<false><<<grid, kThreads, smem, st>>>(m, a);
    }
    return cudaGetLastError();
}

}  // namespace voila
