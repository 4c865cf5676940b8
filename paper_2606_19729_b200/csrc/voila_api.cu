// voila_api.cu -- the C ABI of libvoila (include/voila.h): context, weight packing, argument
// validation, workspace carving and the launch sequences of the two hot calls.
#include <cmath>
#include <cstring>
#include <new>

#include "voila_kernels.h"

using namespace voila;

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) {
        cudaGetDevice(&prev);
        if (prev != dev) cudaSetDevice(dev);
        else prev = -1;
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

float host_bf16_round(float x) {
    uint32_t u;
    std::memcpy(&u, &x, 4);
    if ((u & 0x7f800000u) != 0x7f800000u) {
        u += 0x7fffu + ((u >> 16) & 1u);
        u &= 0xffff0000u;
    }
    std::memcpy(&x, &u, 4);
    return x;
}

voila_status cuda_fail(voila_ctx *ctx, cudaError_t e) {
    if (ctx) ctx->last_cuda_error = cudaGetErrorString(e);
    return VOILA_ERR_CUDA;
}

bool misaligned(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

bool valid_mlp(const voila_mlp &f, int in_dim, int out_dim) {
    if (f.n_layers < 1 || f.n_layers > kMaxLayers || !f.dims || !f.W || !f.b) return false;
    if (f.act < VOILA_ACT_NONE || f.act > VOILA_ACT_SILU) return false;
    for (int l = 0; l <= f.n_layers; ++l)
        if (f.dims[l] < 1) return false;
    for (int l = 0; l < f.n_layers; ++l)
        if (!f.W[l] || !f.b[l]) return false;
    if (f.dims[0] != in_dim) return false;
    if (out_dim > 0 && f.dims[f.n_layers] != out_dim) return false;
    return true;
}

// Workspace layout for reserved maxima (P, Q, N); all offsets kAlign-aligned.
struct Layout {
    size_t wsum, part_value, part_witness, e, proposals, logits, max_ordered, state, tile_flag,
        tile_agg, tile_incl, tile_sumv, cdf, part_wsum, total;
};

Layout make_layout(const voila_ctx *ctx, int P, int Q, int N) {
    Layout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) {
        const size_t o = off;
        off += align_up(bytes > 0 ? bytes : 1);
        return o;
    };
    const size_t tiles = (size_t)(P + kTileRows - 1) / kTileRows;
    const size_t esize = ctx->prec == VOILA_PREC_BF16 ? 2 : 4;
    const size_t stiles = (size_t)scan_tiles(N > 0 ? N : 1);
    L.wsum = take(sizeof(double));
    L.part_value = take((size_t)Q * tiles * sizeof(double));
    L.part_witness = take((size_t)Q * tiles * ctx->O * sizeof(double));
    L.e = take((size_t)ctx->d * sizeof(float));
    L.proposals = take((size_t)N * ctx->S * esize);
    L.logits = take((size_t)N * sizeof(float));
    L.max_ordered = take(sizeof(int));
    L.state = take(sizeof(ScanState));
    L.tile_flag = take(stiles * sizeof(unsigned));
    L.tile_agg = take(stiles * sizeof(unsigned long long));
    L.tile_incl = take(stiles * sizeof(unsigned long long));
    L.tile_sumv = take(2 * stiles * sizeof(double));  // per tile: sum v, then (at + tiles) sum v^2
    L.cdf = take((size_t)N * sizeof(unsigned long long));
    L.part_wsum = take(((size_t)(N + kTileRows - 1) / kTileRows) * sizeof(double));
    L.total = off;
    return L;
}

ScanBuffers scan_buffers(const voila_ctx *ctx, const Layout &L) {
    uint8_t *w = reinterpret_cast<uint8_t *>(ctx->ws);
    ScanBuffers sb;
    sb.state = reinterpret_cast<ScanState *>(w + L.state);
    sb.tile_flag = reinterpret_cast<unsigned *>(w + L.tile_flag);
    sb.tile_agg = reinterpret_cast<unsigned long long *>(w + L.tile_agg);
    sb.tile_incl = reinterpret_cast<unsigned long long *>(w + L.tile_incl);
    sb.tile_sumv = reinterpret_cast<double *>(w + L.tile_sumv);
    sb.cdf = reinterpret_cast<unsigned long long *>(w + L.cdf);
    sb.max_ordered = reinterpret_cast<int *>(w + L.max_ordered);
    sb.part_wsum = reinterpret_cast<double *>(w + L.part_wsum);
    return sb;
}

// Staging layout of the *_host entry points.
struct Stage {
    size_t particles, actions, weights, values, witness, obs, particles_out, weights_out, ancestors,
        scalars, total;
};

Stage make_stage(const voila_ctx *ctx, int P, int Q, int H, int N) {
    Stage s{};
    size_t off = 0;
    auto take = [&](size_t bytes) {
        const size_t o = off;
        off += align_up(bytes > 0 ? bytes : 1);
        return o;
    };
    const size_t esize = ctx->prec == VOILA_PREC_BF16 ? 2 : 4;
    const size_t rows = (size_t)(P > N ? P : N);
    s.particles = take(rows * ctx->S * esize);
    s.actions = take((size_t)Q * H * sizeof(int32_t));
    s.weights = take(rows * sizeof(float));
    s.values = take((size_t)Q * sizeof(float));
    s.witness = take((size_t)Q * ctx->O * sizeof(float));
    s.obs = take((size_t)ctx->O * sizeof(float));
    s.particles_out = take((size_t)N * ctx->S * esize);
    s.weights_out = take((size_t)N * sizeof(float));
    s.ancestors = take((size_t)N * sizeof(int32_t));
    s.scalars = take(64);
    s.total = off;
    return s;
}

// Brackets one kernel launch with a CUDA event pair when profiling is on.
struct ProfScope {
    voila_ctx *ctx;
    int kind, slot;
    cudaStream_t st;
    ProfScope(voila_ctx *c, int k, cudaStream_t s) : ctx(c), kind(k), slot(-1), st(s) {
        if (!ctx->profiling || ctx->prof_n[kind] >= voila_ctx::kProfRing) return;
        slot = ctx->prof_n[kind];
        if (!ctx->prof_ev[kind][slot][0]) {
            cudaEventCreate(&ctx->prof_ev[kind][slot][0]);
            cudaEventCreate(&ctx->prof_ev[kind][slot][1]);
        }
        cudaEventRecord(ctx->prof_ev[kind][slot][0], st);
    }
    ~ProfScope() {
        if (slot < 0) return;
        cudaEventRecord(ctx->prof_ev[kind][slot][1], st);
        ctx->prof_n[kind] = slot + 1;
    }
};

bool use_tc2(const voila_ctx *ctx) {
    return ctx->prec == VOILA_PREC_BF16 && ctx->tc2 != nullptr &&
           (ctx->kernel == VOILA_KERNEL_AUTO || ctx->kernel == VOILA_KERNEL_TCGEN05_PAIR);
}
bool use_tc(const voila_ctx *ctx) {
    return ctx->prec == VOILA_PREC_BF16 && ctx->tc != nullptr && ctx->kernel != VOILA_KERNEL_FFMA &&
           !use_tc2(ctx);
}

}  // namespace

extern "C" {

const char *voila_status_string(voila_status s) {
    switch (s) {
        case VOILA_OK: return "ok";
        case VOILA_ERR_INVALID_ARG: return "invalid argument";
        case VOILA_ERR_UNSUPPORTED: return "unsupported device or model dimensions";
        case VOILA_ERR_CUDA: return "CUDA error";
        case VOILA_ERR_WORKSPACE: return "sizes exceed the reserved workspace (call voila_reserve)";
    }
    return "unknown status";
}

int voila_version(void) { return 100; }

voila_status voila_set_profiling(voila_ctx *ctx, int on) {
    if (!ctx) return VOILA_ERR_INVALID_ARG;
    ctx->profiling = on != 0;
    return VOILA_OK;
}

int voila_profile_read(voila_ctx *ctx, int which, float *ms_out, int max_n) {
    if (!ctx || which < 0 || which > 3 || !ms_out || max_n < 0) return 0;
    DeviceGuard guard(ctx->device);
    int n = 0;
    for (int i = 0; i < ctx->prof_n[which] && n < max_n; ++i) {
        float ms = 0.0f;
        if (cudaEventSynchronize(ctx->prof_ev[which][i][1]) != cudaSuccess) break;
        if (cudaEventElapsedTime(&ms, ctx->prof_ev[which][i][0], ctx->prof_ev[which][i][1]) != cudaSuccess) break;
        ms_out[n++] = ms;
    }
    ctx->prof_n[which] = 0;
    return n;
}

const char *voila_last_cuda_error(const voila_ctx *ctx) { return ctx ? ctx->last_cuda_error.c_str() : ""; }
uint64_t voila_launch_count(const voila_ctx *ctx) { return ctx ? ctx->launches : 0; }
const char *voila_last_rollout_kernel(const voila_ctx *ctx) {
    return ctx ? ctx->last_rollout_kernel.c_str() : "";
}
const char *voila_last_belief_kernel(const voila_ctx *ctx) {
    return ctx ? ctx->last_belief_kernel.c_str() : "";
}

voila_status voila_create(const voila_model_desc *desc, int device, voila_ctx **out) {
    if (!desc || !out) return VOILA_ERR_INVALID_ARG;
    const int S = desc->state_dim, O = desc->obs_dim, A = desc->n_actions, Nz = desc->noise_dim;
    if (S < 1 || O < 1 || A < 1 || Nz < 0) return VOILA_ERR_INVALID_ARG;
    if (desc->prec != VOILA_PREC_FP32 && desc->prec != VOILA_PREC_BF16) return VOILA_ERR_INVALID_ARG;
    if (!(desc->lik_temperature > 0.0f) || !(desc->discount > 0.0f) || !(desc->discount <= 1.0f))
        return VOILA_ERR_INVALID_ARG;
    if (desc->lik_action_cond != 0 && desc->lik_action_cond != 1) return VOILA_ERR_INVALID_ARG;
    if (!valid_mlp(desc->f_T, S + A + Nz, S) || !valid_mlp(desc->f_Z, S + A + Nz, O) ||
        !valid_mlp(desc->lik_obs, O, -1) ||
        !valid_mlp(desc->lik_state, S + (desc->lik_action_cond ? A : 0), -1))
        return VOILA_ERR_INVALID_ARG;
    const int d = desc->lik_obs.dims[desc->lik_obs.n_layers];
    if (d != desc->lik_state.dims[desc->lik_state.n_layers]) return VOILA_ERR_INVALID_ARG;
    if (desc->denoise_T.n_layers != 0 && !valid_mlp(desc->denoise_T, S + A + S + kTemb, S)) return VOILA_ERR_INVALID_ARG;
    if (desc->denoise_Z.n_layers != 0 && !valid_mlp(desc->denoise_Z, S + A + O + kTemb, O)) return VOILA_ERR_INVALID_ARG;
    if (desc->reward.kind < VOILA_R_NEG_L2_GOAL || desc->reward.kind > VOILA_R_LINEAR || !desc->reward.param)
        return VOILA_ERR_INVALID_ARG;
    const voila_terminal *term = desc->terminal;
    int term_floats = 0;
    if (term && term->n_regions > 0) {
        if (term->n_regions > VOILA_MAX_TERMINAL_REGIONS || !term->dims || !term->centers || !term->radii ||
            !term->rewards || !term->stops)
            return VOILA_ERR_INVALID_ARG;
        for (int k = 0; k < term->n_regions; ++k) {
            if (term->dims[k] < 1 || term->dims[k] > S || !(term->radii[k] >= 0.0f)) return VOILA_ERR_INVALID_ARG;
            term_floats += term->dims[k];
        }
    }

    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) {
        cudaGetLastError();
        return VOILA_ERR_UNSUPPORTED;  // no CPU fallback
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return VOILA_ERR_CUDA;
    if (prop.major != 10) return VOILA_ERR_UNSUPPORTED;  // built for sm_100a only

    voila_ctx *ctx = new (std::nothrow) voila_ctx();
    if (!ctx) return VOILA_ERR_INVALID_ARG;
    ctx->device = device;
    ctx->sm_count = prop.multiProcessorCount;
    ctx->prec = desc->prec;
    ctx->S = S; ctx->O = O; ctx->A = A; ctx->Nz = Nz; ctx->d = d;
    DeviceGuard guard(device);

    ModelDev &m = ctx->model;
    m.S = S; m.O = O; m.A = A; m.Nz = Nz;
    m.lik_action_cond = desc->lik_action_cond;
    m.lambda = desc->lik_temperature;
    m.gamma = desc->discount;
    m.max_width = 1;
    const voila_mlp *src[6] = {&desc->f_T, &desc->f_Z, &desc->lik_obs, &desc->lik_state, &desc->denoise_T,
                               &desc->denoise_Z};
    const bool bf16 = desc->prec == VOILA_PREC_BF16;

    auto upload = [&](const std::vector<float> &h, const float **dst) -> cudaError_t {
        void *p = nullptr;
        cudaError_t e = cudaMalloc(&p, h.size() * sizeof(float));
        if (e != cudaSuccess) return e;
        ctx->dev_allocs.push_back(p);
        *dst = reinterpret_cast<const float *>(p);
        return cudaMemcpy(p, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice);
    };
    cudaError_t e = cudaSuccess;
    for (int w = 0; w < 6 && e == cudaSuccess; ++w) {
        const voila_mlp &f = *src[w];
        MlpDev &g = m.mlp[w];
        g.n_layers = f.n_layers;
        if (w >= 4 && f.n_layers == 0) continue;  // no such diffusion teacher
        g.act = f.act;
        for (int l = 0; l <= f.n_layers; ++l) {
            g.dims[l] = f.dims[l];
            if (f.dims[l] > m.max_width) m.max_width = f.dims[l];
        }
        for (int l = 0; l < f.n_layers && e == cudaSuccess; ++l) {
            const int K = f.dims[l], N = f.dims[l + 1];
            std::vector<float> wt((size_t)K * N), bb(f.b[l], f.b[l] + N);
            for (int j = 0; j < N; ++j)
                for (int k = 0; k < K; ++k) {
                    const float v = f.W[l][(size_t)j * K + k];
                    wt[(size_t)k * N + j] = bf16 ? host_bf16_round(v) : v;  // k-major: lanes read j
                }
            e = upload(wt, &g.Wt[l]);
            if (e == cudaSuccess) e = upload(bb, &g.b[l]);
        }
    }
    if (e == cudaSuccess) {
        const int n = desc->reward.kind == VOILA_R_NEG_L2_GOAL ? S
                      : desc->reward.kind == VOILA_R_NEG_QUADRATIC ? S * S : S + 1;
        m.reward.kind = desc->reward.kind;
        e = upload(std::vector<float>(desc->reward.param, desc->reward.param + n), &m.reward.param);
        m.reward.action_cost = nullptr;
        if (e == cudaSuccess && desc->reward.action_cost)
            e = upload(std::vector<float>(desc->reward.action_cost, desc->reward.action_cost + A),
                       &m.reward.action_cost);
    }
    m.term = TerminalDev{};
    bool term_fits_tc = true;  // the tensor-core epilogue keeps the state packed in registers: leading 8 coordinates
    if (e == cudaSuccess && term_floats > 0) {
        m.term.n = term->n_regions;
        int off = 0;
        for (int k = 0; k < term->n_regions; ++k) {
            m.term.dim[k] = term->dims[k];
            m.term.off[k] = off;
            m.term.stop[k] = term->stops[k] ? 1 : 0;
            m.term.r2[k] = term->radii[k] * term->radii[k];
            m.term.reward[k] = term->rewards[k];
            off += term->dims[k];
            if (term->dims[k] > 8) term_fits_tc = false;
        }
        e = upload(std::vector<float>(term->centers, term->centers + term_floats), &m.term.centers);
    }
    if (e != cudaSuccess) {
        voila_destroy(ctx);
        return VOILA_ERR_CUDA;
    }
    if (ffma_smem_bytes(m) > (size_t)prop.sharedMemPerBlockOptin) {
        voila_destroy(ctx);
        return VOILA_ERR_UNSUPPORTED;
    }
    if (bf16) {
        std::string why;
        if (tc2_supported(desc, &why) && term_fits_tc) {
            // A program that does not fit (tables, shared memory, tensor map) leaves its handle null and
            // AUTO runs the CUDA-core kernels, as voila.h promises; the reason stays readable.
            std::string err;
            if (m.term.n == 0 && tc_supported(desc, &why)) {  // the single-CTA variant: aligned dims, no terminal regions
                ctx->tc = tc_create(desc, ctx->sm_count, &ctx->dev_allocs, &err);
                if (!ctx->tc) ctx->last_cuda_error = "single-CTA tcgen05 program not built: " + err;
            }
            ctx->tc2 = tc2_create(desc, ctx->sm_count, &ctx->dev_allocs, &err);
            if (!ctx->tc2) ctx->last_cuda_error = "CTA-pair tcgen05 program not built: " + err;
        }
    }
    *out = ctx;
    return VOILA_OK;
}

void voila_destroy(voila_ctx *ctx) {
    if (!ctx) return;
    {
        DeviceGuard guard(ctx->device);
        cudaDeviceSynchronize();
        if (ctx->tc) tc_destroy(ctx->tc);
        if (ctx->tc2) tc2_destroy(ctx->tc2);
        for (auto &kind : ctx->prof_ev)
            for (auto &pair : kind)
                for (auto &ev : pair)
                    if (ev) cudaEventDestroy(ev);
        for (void *p : ctx->dev_allocs) cudaFree(p);
        if (ctx->ws) cudaFree(ctx->ws);
        if (ctx->stage) cudaFree(ctx->stage);
        if (ctx->pw_ws) cudaFree(ctx->pw_ws);
    }
    delete ctx;
}

size_t voila_workspace_bytes(const voila_ctx *ctx, int P, int Q, int H, int N) {
    (void)H;
    if (!ctx || P < 0 || Q < 0 || N < 0) return 0;
    return make_layout(ctx, P, Q, N).total;
}

voila_status voila_reserve(voila_ctx *ctx, int P, int Q, int H, int N) {
    if (!ctx || P < 0 || Q < 0 || H < 0 || N < 0) return VOILA_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    cudaDeviceSynchronize();
    const Layout L = make_layout(ctx, P, Q, N);
    const Stage s = make_stage(ctx, P, Q, H, N);
    if (ctx->ws) cudaFree(ctx->ws);
    if (ctx->stage) cudaFree(ctx->stage);
    ctx->ws = ctx->stage = nullptr;
    ctx->res_P = ctx->res_Q = ctx->res_H = ctx->res_N = 0;
    cudaError_t e = cudaMalloc(&ctx->ws, L.total);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->stage, s.total);
    if (e != cudaSuccess) {
        if (ctx->ws) cudaFree(ctx->ws);
        ctx->ws = nullptr;
        return cuda_fail(ctx, e);
    }
    ctx->ws_bytes = L.total;
    ctx->stage_bytes = s.total;
    ctx->res_P = P; ctx->res_Q = Q; ctx->res_H = H; ctx->res_N = N;
    return VOILA_OK;
}

voila_status voila_set_kernel(voila_ctx *ctx, int kernel) {
    if (!ctx || kernel < VOILA_KERNEL_AUTO || kernel > VOILA_KERNEL_TCGEN05_PAIR) return VOILA_ERR_INVALID_ARG;
    if (kernel == VOILA_KERNEL_TCGEN05 && !ctx->tc) return VOILA_ERR_UNSUPPORTED;
    if (kernel == VOILA_KERNEL_TCGEN05_PAIR && !ctx->tc2) return VOILA_ERR_UNSUPPORTED;
    ctx->kernel = kernel;
    return VOILA_OK;
}

int voila_tcgen05_supported(const voila_ctx *ctx) { return ctx && ctx->tc ? 1 : 0; }

voila_status voila_rollout_values(voila_ctx *ctx, const void *particles, int P,
                                  const int32_t *action_seqs, int Q, int H, const float *weights,
                                  uint64_t seed, float *values_out, float *obs_witness_out,
                                  float *returns_out, float *final_states_out, void *cuda_stream) {
    if (!ctx || !particles || !action_seqs || !values_out || P < 1 || Q < 1 || H < 1)
        return VOILA_ERR_INVALID_ARG;
    if (misaligned(particles) || misaligned(action_seqs) || misaligned(weights) ||
        misaligned(values_out) || misaligned(obs_witness_out) || misaligned(returns_out) ||
        misaligned(final_states_out))
        return VOILA_ERR_INVALID_ARG;
    if (!ctx->ws || P > ctx->res_P || Q > ctx->res_Q) return VOILA_ERR_WORKSPACE;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const Layout L = make_layout(ctx, ctx->res_P, ctx->res_Q, ctx->res_N);
    uint8_t *w = reinterpret_cast<uint8_t *>(ctx->ws);

    RolloutArgs a{};
    a.particles = particles;
    a.action_seqs = action_seqs;
    a.weights = weights;
    a.P = P; a.Q = Q; a.H = H;
    a.seed = seed;
    a.part_value = reinterpret_cast<double *>(w + L.part_value);
    a.part_witness = obs_witness_out ? reinterpret_cast<double *>(w + L.part_witness) : nullptr;
    a.returns_out = returns_out;
    a.final_states_out = final_states_out;
    const int tile_rows = use_tc(ctx) ? 128 : kTileRows;
    a.tiles = use_tc2(ctx) ? 2 * ((P + 255) / 256) : (P + tile_rows - 1) / tile_rows;
    if (a.tiles > 65535) return VOILA_ERR_INVALID_ARG;  // grid.y of the CUDA-core kernel (P > 2^21 particles)
    double *wsum = reinterpret_cast<double *>(w + L.wsum);

    cudaError_t e = launch_weight_sum(weights, P, wsum, st);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->launches += 1;
    if (use_tc2(ctx)) {
        int n = 0;
        ProfScope prof(ctx, VOILA_K_ROLLOUT, st);
        e = launch_rollout_tc2(ctx->tc2, ctx->model, a, st, &ctx->last_rollout_kernel, &n);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
        ctx->launches += n;
    } else if (use_tc(ctx)) {
        int n = 0;
        ProfScope prof(ctx, VOILA_K_ROLLOUT, st);
        e = launch_rollout_tc(ctx->tc, ctx->model, a, st, &ctx->last_rollout_kernel, &n);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
        ctx->launches += n;
    } else {
        ProfScope prof(ctx, VOILA_K_ROLLOUT, st);
        e = launch_rollout_ffma(ctx->model, a, ctx->prec == VOILA_PREC_BF16, st);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
        ctx->launches += 1;
        ctx->last_rollout_kernel = ctx->prec == VOILA_PREC_BF16 ? "rollout_ffma_kernel<bf16>"
                                                                 : "rollout_ffma_kernel<fp32>";
    }
    e = launch_rollout_reduce(a, ctx->O, wsum, values_out, obs_witness_out, st);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->launches += 1;
    return VOILA_OK;
}

static voila_status run_resample(voila_ctx *ctx, const ScanBuffers &sb, int N, const void *proposals,
                                 void *particles_out, float *weights_out, int32_t *ancestors_out,
                                 cudaStream_t st, const float *w_in, bool from_logits) {
    const int esize = ctx->prec == VOILA_PREC_BF16 ? 2 : 4;
    ProfScope prof(ctx, VOILA_K_RESAMPLE, st);
    cudaError_t e = launch_resample_gather(sb, N, proposals, ctx->S * esize, particles_out,
                                           weights_out, ancestors_out, st, w_in, from_logits);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->launches += 1;
    return VOILA_OK;
}

voila_status voila_belief_update(voila_ctx *ctx, const void *particles, int N, int32_t action,
                                 const float *observation, const float *weights, uint64_t seed,
                                 void *particles_out, float *weights_out, int32_t *ancestors_out,
                                 float *post_weights_out, void *proposals_out,
                                 float *log_evidence_out, int32_t *dev_status_out, void *cuda_stream) {
    return voila_belief_update_ess(ctx, particles, N, action, observation, weights, seed, INFINITY, particles_out,
                                   weights_out, ancestors_out, post_weights_out, proposals_out, log_evidence_out,
                                   nullptr, nullptr, dev_status_out, cuda_stream);
}

voila_status voila_belief_update_ess(voila_ctx *ctx, const void *particles, int N, int32_t action,
                                     const float *observation, const float *weights, uint64_t seed,
                                     float ess_threshold, void *particles_out, float *weights_out,
                                     int32_t *ancestors_out, float *post_weights_out, void *proposals_out,
                                     float *log_evidence_out, float *ess_out, int32_t *resampled_out,
                                     int32_t *dev_status_out, void *cuda_stream) {
    if (!ctx || !particles || !observation || !particles_out || N < 1) return VOILA_ERR_INVALID_ARG;
    if (!(ess_threshold > 0.0f)) return VOILA_ERR_INVALID_ARG;  // also rejects NaN
    if (misaligned(ess_out) || misaligned(resampled_out)) return VOILA_ERR_INVALID_ARG;
    if (action < 0 || action >= ctx->A) return VOILA_ERR_INVALID_ARG;
    if (particles_out == particles || proposals_out == particles || particles_out == proposals_out)
        return VOILA_ERR_INVALID_ARG;  // the gather reads proposal rows while other CTAs write particles_out
    if (((uintptr_t)log_evidence_out & 3u) || ((uintptr_t)dev_status_out & 3u)) return VOILA_ERR_INVALID_ARG;
    if (misaligned(particles) || misaligned(observation) || misaligned(weights) ||
        misaligned(particles_out) || misaligned(weights_out) || misaligned(ancestors_out) ||
        misaligned(post_weights_out) || misaligned(proposals_out))
        return VOILA_ERR_INVALID_ARG;
    if (!ctx->ws || N > ctx->res_N) return VOILA_ERR_WORKSPACE;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const Layout L = make_layout(ctx, ctx->res_P, ctx->res_Q, ctx->res_N);
    uint8_t *w = reinterpret_cast<uint8_t *>(ctx->ws);
    const ScanBuffers sb = scan_buffers(ctx, L);
    const bool bf16 = ctx->prec == VOILA_PREC_BF16;
    float *e_dev = reinterpret_cast<float *>(w + L.e);

    // scan bookkeeping reset + e = f(o): the observation tower, once
    cudaError_t e;
    if (obs_tower_fits(ctx->model.mlp[2])) {
        e = launch_bu_init_obs(sb, N, ctx->model.mlp[2], observation, e_dev, bf16, st);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
        ctx->launches += 1;
    } else {
        e = launch_bu_init(sb, N, st);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
        e = launch_mlp_forward_ffma(ctx->model, 2, observation, 1, e_dev, bf16, st);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
        ctx->launches += 2;
    }

    BeliefArgs a{};
    a.particles = particles;
    a.weights = weights;
    a.N = N;
    a.action = action;
    a.seed = seed;
    a.e = e_dev;
    a.proposals = proposals_out ? proposals_out : (void *)(w + L.proposals);
    a.logits = reinterpret_cast<float *>(w + L.logits);
    a.max_ordered = sb.max_ordered;
    a.part_wsum = sb.part_wsum;
    int n_parts = (N + kTileRows - 1) / kTileRows;
    if (use_tc2(ctx) && tc2_has_belief(ctx->tc2)) {
        int n = 0;
        ProfScope prof(ctx, VOILA_K_PROPOSE, st);
        e = launch_bu_propose_score_tc2(ctx->tc2, ctx->model, a, st, &n, &ctx->last_belief_kernel);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
        ctx->launches += n;
        n_parts = (N + 31) / 32;
    } else if (use_tc(ctx) && tc_has_belief(ctx->tc)) {
        int n = 0;
        ProfScope prof(ctx, VOILA_K_PROPOSE, st);
        e = launch_bu_propose_score_tc(ctx->tc, ctx->model, a, st, &n);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
        ctx->launches += n;
        n_parts = (N + 127) / 128;
    } else {
        ProfScope prof(ctx, VOILA_K_PROPOSE, st);
        e = launch_bu_propose_score_ffma(ctx->model, a, bf16, st);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
        ctx->launches += 1;
        ctx->last_belief_kernel = bf16 ? "bu_propose_score_ffma_kernel<bf16>" : "bu_propose_score_ffma_kernel<fp32>";
    }
    {
        // scan; its last CTA finalises (W, comb offset, evidence, status, ESS decision)
        FinalizeArgs fin{};
        fin.enabled = 1;
        fin.n_wsum_parts = n_parts;
        fin.has_prior = weights != nullptr;
        fin.from_logits = 1;
        fin.seed = seed;
        fin.ess_threshold = ess_threshold;
        fin.log_evidence_out = log_evidence_out; fin.ess_out = ess_out;
        fin.dev_status_out = dev_status_out; fin.resampled_out = resampled_out;
        ProfScope prof(ctx, VOILA_K_SCAN, st);
        e = launch_weight_scan(sb, a.logits, N, true, post_weights_out, st, &fin);
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->launches += 1;
    return run_resample(ctx, sb, N, a.proposals, particles_out, weights_out, ancestors_out, st, a.logits, true);
}

voila_status voila_resample_systematic(voila_ctx *ctx, const float *v, int N, uint64_t seed,
                                       int32_t *ancestors_out, int32_t *dev_status_out,
                                       void *cuda_stream) {
    if (!ctx || !v || !ancestors_out || N < 1) return VOILA_ERR_INVALID_ARG;
    if (misaligned(v) || misaligned(ancestors_out)) return VOILA_ERR_INVALID_ARG;
    if (!ctx->ws || N > ctx->res_N) return VOILA_ERR_WORKSPACE;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const Layout L = make_layout(ctx, ctx->res_P, ctx->res_Q, ctx->res_N);
    const ScanBuffers sb = scan_buffers(ctx, L);
    cudaError_t e = launch_bu_init(sb, N, st);
    if (e == cudaSuccess) {
        FinalizeArgs fin{};
        fin.enabled = 1;
        fin.seed = seed;
        fin.ess_threshold = INFINITY;
        fin.dev_status_out = dev_status_out;
        e = launch_weight_scan(sb, v, N, false, nullptr, st, &fin);
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->launches += 2;
    return run_resample(ctx, sb, N, nullptr, nullptr, nullptr, ancestors_out, st, v, false);
}

// ---- the no-allocation resampler (scratch: a static device array in belief.cu) ----
namespace {
thread_local char g_static_err[160] = "";
void static_err(const char *fmt, long a = 0, long b = 0) { snprintf(g_static_err, sizeof(g_static_err), fmt, a, b); }
}  // namespace

const char *voila_static_last_error(void) { return g_static_err; }

voila_status voila_resample_systematic_static(const float *v, int N, uint64_t seed, int32_t *ancestors_out,
                                              int32_t *dev_status_out, void *cuda_stream) {
    g_static_err[0] = 0;
    if (!v || !ancestors_out || N < 1) {
        static_err("voila_resample_systematic_static: NULL pointer or N < 1 (N = %ld)", (long)N);
        return VOILA_ERR_INVALID_ARG;
    }
    if (misaligned(v) || misaligned(ancestors_out)) {
        static_err("voila_resample_systematic_static: v and ancestors_out must be 16-byte aligned");
        return VOILA_ERR_INVALID_ARG;
    }
    if (N > static_resample_max_n()) {
        static_err("voila_resample_systematic_static: N = %ld exceeds VOILA_STATIC_MAX_N = %ld (the static scratch "
                   "array); use voila_resample_systematic with a reserved workspace", (long)N,
                   (long)static_resample_max_n());
        return VOILA_ERR_WORKSPACE;
    }
    const char *why = nullptr;
    const cudaError_t e = launch_resample_systematic_static(v, N, seed, ancestors_out, dev_status_out,
                                                            reinterpret_cast<cudaStream_t>(cuda_stream), &why);
    if (e != cudaSuccess) {
        snprintf(g_static_err, sizeof(g_static_err), "voila_resample_systematic_static: %s%s%s",
                 why ? why : "", why ? ": " : "", cudaGetErrorString(e));
        cudaGetLastError();
        return VOILA_ERR_CUDA;
    }
    return VOILA_OK;
}

// ---- progressive widening ----
namespace {
struct PwLayout {
    size_t sim_group, sim_branch, sim_rank, perm, seg_of_pos, sim_action, sim_seg, seg_count, seg_off, new_src,
        seg_max, E, logits, v_sorted, proposals, total;
};
PwLayout make_pw_layout(const voila_ctx *ctx, int N, int G, int M) {
    PwLayout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) {
        const size_t o = off;
        off += align_up(bytes > 0 ? bytes : 1);
        return o;
    };
    const size_t esize = ctx->prec == VOILA_PREC_BF16 ? 2 : 4;
    const size_t gm = (size_t)G * M;
    L.sim_group = take((size_t)N * 4);
    L.sim_branch = take((size_t)N * 4);
    L.sim_rank = take((size_t)N * 4);
    L.perm = take((size_t)N * 4);
    L.seg_of_pos = take((size_t)N * 4);
    L.sim_action = take((size_t)N * 4);
    L.sim_seg = take((size_t)N * 4);
    L.seg_count = take(gm * 4);
    L.seg_off = take((gm + 1) * 4);
    L.new_src = take(gm * 4);
    L.seg_max = take(gm * 4);
    L.E = take(gm * ctx->d * sizeof(float));
    L.logits = take((size_t)N * 4);
    L.v_sorted = take((size_t)N * 4);
    L.proposals = take((size_t)N * ctx->S * esize);
    L.total = off;
    return L;
}
}  // namespace

size_t voila_pw_workspace_bytes(const voila_ctx *ctx, int N, int G, int M_max) {
    if (!ctx || N < 0 || G < 0 || M_max < 0) return 0;
    return make_pw_layout(ctx, N, G, M_max).total;
}

voila_status voila_pw_reserve(voila_ctx *ctx, int N, int G, int M_max) {
    if (!ctx || N < 1 || G < 1 || M_max < 1 || M_max > kPwMaxBranches) return VOILA_ERR_INVALID_ARG;
    if ((long long)G * M_max >= (1ll << 30)) return VOILA_ERR_INVALID_ARG;
    // the uint64 scan of the sorted weights uses the belief update's scan buffers
    if (!ctx->ws || N > ctx->res_N) {
        const voila_status s = voila_reserve(ctx, ctx->res_P, ctx->res_Q, ctx->res_H, N > ctx->res_N ? N : ctx->res_N);
        if (s != VOILA_OK) return s;
    }
    DeviceGuard guard(ctx->device);
    cudaDeviceSynchronize();
    if (ctx->pw_ws) cudaFree(ctx->pw_ws);
    ctx->pw_ws = nullptr;
    ctx->pw_N = ctx->pw_G = ctx->pw_M = 0;
    const cudaError_t e = cudaMalloc(&ctx->pw_ws, make_pw_layout(ctx, N, G, M_max).total);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->pw_N = N; ctx->pw_G = G; ctx->pw_M = M_max;
    return VOILA_OK;
}

voila_status voila_pw_update(voila_ctx *ctx, const void *particles, int N, const int32_t *group_off, int G,
                             const int32_t *group_action, int32_t *visit_count, int32_t *branch_count,
                             float *branch_obs, int M_max, double k_o, double alpha_o, const float *weights,
                             uint64_t seed, void *particles_out, float *weights_out, int32_t *ancestors_out,
                             int32_t *sim_branch_out, int32_t *opened_out, float *post_weights_out,
                             void *proposals_out, int32_t *seg_status_out, void *cuda_stream) {
    if (!ctx || !particles || !group_off || !group_action || !visit_count || !branch_count || !branch_obs)
        return VOILA_ERR_INVALID_ARG;
    if (N < 1 || G < 1 || M_max < 1 || M_max > kPwMaxBranches || !(k_o > 0.0) || !(alpha_o > 0.0))
        return VOILA_ERR_INVALID_ARG;
    if (particles_out == particles || proposals_out == particles || (particles_out && particles_out == proposals_out))
        return VOILA_ERR_INVALID_ARG;
    if (misaligned(particles) || misaligned(weights) || misaligned(particles_out) || misaligned(proposals_out) ||
        misaligned(branch_obs))
        return VOILA_ERR_INVALID_ARG;
    if (!ctx->pw_ws || !ctx->ws || N > ctx->pw_N || N > ctx->res_N ||
        (long long)G * M_max > (long long)ctx->pw_G * ctx->pw_M)
        return VOILA_ERR_WORKSPACE;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const bool bf16 = ctx->prec == VOILA_PREC_BF16;
    const size_t esize = bf16 ? 2 : 4;
    // carve for the reserved maxima (G * M_max slots may be split differently than reserved)
    const PwLayout L = make_pw_layout(ctx, ctx->pw_N, ctx->pw_G, ctx->pw_M);
    uint8_t *w = reinterpret_cast<uint8_t *>(ctx->pw_ws);
    PwArgs a{};
    a.particles = particles; a.weights = weights;
    a.N = N; a.G = G; a.M_max = M_max;
    a.group_off = group_off; a.group_action = group_action;
    a.visit_count = visit_count; a.branch_count = branch_count; a.branch_obs = branch_obs;
    a.k_o = k_o; a.alpha_o = alpha_o; a.seed = seed;
    a.sim_group = reinterpret_cast<int32_t *>(w + L.sim_group);
    a.sim_branch = reinterpret_cast<int32_t *>(w + L.sim_branch);
    a.sim_rank = reinterpret_cast<int32_t *>(w + L.sim_rank);
    a.perm = reinterpret_cast<int32_t *>(w + L.perm);
    a.seg_of_pos = reinterpret_cast<int32_t *>(w + L.seg_of_pos);
    a.sim_action = reinterpret_cast<int32_t *>(w + L.sim_action);
    a.sim_seg = reinterpret_cast<int32_t *>(w + L.sim_seg);
    a.seg_count = reinterpret_cast<int32_t *>(w + L.seg_count);
    a.seg_off = reinterpret_cast<int32_t *>(w + L.seg_off);
    a.new_src = reinterpret_cast<int32_t *>(w + L.new_src);
    a.seg_max = reinterpret_cast<int *>(w + L.seg_max);
    a.E = reinterpret_cast<float *>(w + L.E);
    a.logits = reinterpret_cast<float *>(w + L.logits);
    a.v_sorted = reinterpret_cast<float *>(w + L.v_sorted);
    a.proposals = proposals_out ? proposals_out : (void *)(w + L.proposals);
    a.particles_out = particles_out; a.weights_out = weights_out; a.post_weights_out = post_weights_out;
    a.ancestors_out = ancestors_out; a.sim_branch_out = sim_branch_out; a.opened_out = opened_out;
    a.seg_status_out = seg_status_out;

    const Layout SL = make_layout(ctx, ctx->res_P, ctx->res_Q, ctx->res_N);
    const ScanBuffers sb = scan_buffers(ctx, SL);
    // tensor-core path: one fused propose+score pass over all simulations (per-row actions and tower
    // embeddings); the few rows that open a branch get their s' -> o on the CUDA cores first
    const bool tc_path = use_tc2(ctx) && tc2_has_pw(ctx->tc2) && ctx->d % 16 == 0;
    a.obs_from_particles = tc_path ? 1 : 0;
    cudaError_t e = launch_pw_widen(a, st);                                  // branches, children, sorted order
    if (e == cudaSuccess && !tc_path) e = launch_pw_propose_ffma(ctx->model, a, bf16, st);  // s' of every simulation
    if (tc_path && tc2_has_pw_slots(ctx->tc2)) {
        // o of the opened branches, then e = f(o) of every stored branch: two small tcgen05 passes over the slots
        if (e == cudaSuccess) e = launch_pw_slots_tc2(ctx->tc2, ctx->model, a, st);
    } else {
        if (e == cudaSuccess) e = launch_pw_obs_ffma(ctx->model, a, bf16, st);      // o of the opened branches
        if (e == cudaSuccess)                                                     // e = f(o) of every stored branch: one batch
            e = launch_mlp_forward_ffma(ctx->model, 2, branch_obs, G * M_max, a.E, bf16, st);
    }
    if (e == cudaSuccess) {                                                   // L_i, child maxima
        ProfScope prof(ctx, VOILA_K_PROPOSE, st);
        if (tc_path) {
            e = launch_pw_propose_score_tc2(ctx->tc2, ctx->model, a, a.sim_action, a.sim_seg, st, &ctx->last_belief_kernel);
        } else {
            e = launch_pw_score_ffma(ctx->model, a, bf16, st);
            ctx->last_belief_kernel = bf16 ? "pw_propose/score_ffma_kernel<bf16>" : "pw_propose/score_ffma_kernel<fp32>";
        }
    }
    if (e == cudaSuccess) e = launch_pw_weights(a, st);                       // v in sorted order
    if (e == cudaSuccess) e = launch_bu_init(sb, N, st);
    if (e == cudaSuccess) e = launch_weight_scan(sb, a.v_sorted, N, false, nullptr, st);  // uint64 CDF over the sorted order
    if (e == cudaSuccess) e = launch_pw_resample(a, sb.cdf, ctx->S * (int)esize, st);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->launches += (tc_path ? 10 : 11) + (seg_status_out ? 1 : 0);
    return VOILA_OK;
}

voila_status voila_porpp_backup_level(voila_ctx *ctx, const float *R, const float *logpi0,
                                      const int32_t *child_off, const int32_t *child_idx, const float *child_w,
                                      const float *v_next, int n_belief, int n_actions, float eta, float gamma,
                                      float *psi_out, float *v_out, void *cuda_stream) {
    if (!ctx || !R || !logpi0 || !child_off || !psi_out || !v_out || n_belief < 1 || n_actions < 1)
        return VOILA_ERR_INVALID_ARG;
    if (!(eta > 0.0f) || !(gamma >= 0.0f)) return VOILA_ERR_INVALID_ARG;
    if ((long long)n_belief * n_actions >= (1ll << 31)) return VOILA_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    const cudaError_t e = launch_porpp_backup_level(R, logpi0, child_off, child_idx, child_w, v_next, n_belief,
                                                    n_actions, eta, gamma, psi_out, v_out,
                                                    reinterpret_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->launches += 1;
    return VOILA_OK;
}

voila_status voila_diffusion_sample(voila_ctx *ctx, int which, const void *cond, const int32_t *actions, int N,
                                    int K, uint64_t seed, float *out, void *cuda_stream) {
    if (!ctx || which < 0 || which > 1 || !cond || !actions || !out || N < 1 || K < 1 || K > 256)
        return VOILA_ERR_INVALID_ARG;
    if (misaligned(cond) || misaligned(out)) return VOILA_ERR_INVALID_ARG;
    if (ctx->model.mlp[4 + which].n_layers < 1) return VOILA_ERR_UNSUPPORTED;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const bool bf16 = ctx->prec == VOILA_PREC_BF16;
    DiffusionArgs a{};
    a.cond = cond; a.actions = actions; a.N = N; a.which = which;
    a.D = which == 0 ? ctx->S : ctx->O;
    a.seed = seed; a.x = out;
    const double half_pi = 1.5707963267948966, pi = 3.141592653589793;
    for (int k = 0; k < K; ++k) {  // one denoiser call per step (why the teacher is expensive)
        const double tau = 1.0 - (double)k / (double)K, tau_n = 1.0 - (double)(k + 1) / (double)K;
        for (int e = 0; e < kTemb / 2; ++e) {
            a.temb[2 * e] = (float)std::sin(pi * (double)(1 << e) * tau);
            a.temb[2 * e + 1] = (float)std::cos(pi * (double)(1 << e) * tau);
        }
        a.al = (float)std::cos(half_pi * tau); a.si = (float)std::sin(half_pi * tau);
        a.al_n = (float)std::cos(half_pi * tau_n); a.si_n = (float)std::sin(half_pi * tau_n);
        a.first = k == 0;
        cudaError_t e;
        if (use_tc2(ctx) && tc2_has_diffusion(ctx->tc2, which)) {
            e = launch_diffusion_step_tc2(ctx->tc2, ctx->model, a, k, st, &ctx->last_belief_kernel);
            ctx->launches += 2;
        } else {
            e = launch_diffusion_step_ffma(ctx->model, a, bf16, st);
            ctx->last_belief_kernel = bf16 ? "diffusion_step_ffma_kernel<bf16>" : "diffusion_step_ffma_kernel<fp32>";
            ctx->launches += 1;
        }
        if (e != cudaSuccess) return cuda_fail(ctx, e);
    }
    return VOILA_OK;
}

voila_status voila_porpp_backup(voila_ctx *ctx, const voila_porpp_level *levels, int n_levels, int n_actions,
                                const float *leaf_values, float eta, float gamma, int32_t *root_action_out,
                                void *cuda_stream) {
    if (!ctx || !levels || n_levels < 1 || n_actions < 1) return VOILA_ERR_INVALID_ARG;
    if (!(eta > 0.0f) || !(gamma >= 0.0f)) return VOILA_ERR_INVALID_ARG;
    for (int d = 0; d < n_levels; ++d) {
        const voila_porpp_level &lv = levels[d];
        if (!lv.R || !lv.logpi0 || !lv.child_off || !lv.psi_out || !lv.v_out || lv.n_belief < 1)
            return VOILA_ERR_INVALID_ARG;
        if ((long long)lv.n_belief * n_actions >= (1ll << 31)) return VOILA_ERR_INVALID_ARG;
    }
    DeviceGuard guard(ctx->device);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const float *v_next = leaf_values;
    for (int d = n_levels - 1; d >= 0; --d) {
        const voila_porpp_level &lv = levels[d];
        const cudaError_t e = launch_porpp_backup_level(lv.R, lv.logpi0, lv.child_off, lv.child_idx, lv.child_w, v_next,
                                                        lv.n_belief, n_actions, eta, gamma, lv.psi_out, lv.v_out, st,
                                                        d == 0 ? root_action_out : nullptr);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
        ctx->launches += 1;
        v_next = lv.v_out;
    }
    return VOILA_OK;
}

voila_status voila_mlp_forward(voila_ctx *ctx, int which, const float *x, int rows, float *y,
                               void *cuda_stream) {
    if (!ctx || which < 0 || which > 3 || !x || !y || rows < 1) return VOILA_ERR_INVALID_ARG;
    if (misaligned(x) || misaligned(y)) return VOILA_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    cudaError_t e = launch_mlp_forward_ffma(ctx->model, which, x, rows, y, ctx->prec == VOILA_PREC_BF16,
                                            reinterpret_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->launches += 1;
    return VOILA_OK;
}

voila_status voila_best_action(voila_ctx *ctx, const float *values, const int32_t *action_seqs, int Q,
                               int H, int32_t *best_q_out, int32_t *best_action_out, void *cuda_stream) {
    if (!ctx || !values || !action_seqs || !best_action_out || Q < 1 || H < 1) return VOILA_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    cudaError_t e = launch_best_action(values, action_seqs, Q, H, best_q_out, best_action_out,
                                       reinterpret_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    ctx->launches += 1;
    return VOILA_OK;
}

voila_status voila_rollout_values_host(voila_ctx *ctx, const void *particles, int P,
                                       const int32_t *action_seqs, int Q, int H, const float *weights,
                                       uint64_t seed, float *values_out, float *obs_witness_out,
                                       void *cuda_stream) {
    return voila_plan_host(ctx, particles, P, action_seqs, Q, H, weights, seed, values_out, obs_witness_out,
                           nullptr, nullptr, cuda_stream);
}

voila_status voila_plan_host(voila_ctx *ctx, const void *particles, int P, const int32_t *action_seqs, int Q,
                             int H, const float *weights, uint64_t seed, float *values_out,
                             float *obs_witness_out, int32_t *best_q_out, int32_t *best_action_out,
                             void *cuda_stream) {
    if (!ctx || !particles || !action_seqs || !values_out || P < 1 || Q < 1 || H < 1)
        return VOILA_ERR_INVALID_ARG;
    if (!ctx->stage || P > ctx->res_P || Q > ctx->res_Q || H > ctx->res_H) return VOILA_ERR_WORKSPACE;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const Stage s = make_stage(ctx, ctx->res_P, ctx->res_Q, ctx->res_H, ctx->res_N);
    uint8_t *g = reinterpret_cast<uint8_t *>(ctx->stage);
    const size_t esize = ctx->prec == VOILA_PREC_BF16 ? 2 : 4;
    cudaError_t e = cudaMemcpyAsync(g + s.particles, particles, (size_t)P * ctx->S * esize,
                                    cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(g + s.actions, action_seqs, (size_t)Q * H * sizeof(int32_t),
                            cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && weights)
        e = cudaMemcpyAsync(g + s.weights, weights, (size_t)P * sizeof(float), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    voila_status vs = voila_rollout_values(
        ctx, g + s.particles, P, reinterpret_cast<const int32_t *>(g + s.actions), Q, H,
        weights ? reinterpret_cast<const float *>(g + s.weights) : nullptr, seed,
        reinterpret_cast<float *>(g + s.values),
        obs_witness_out ? reinterpret_cast<float *>(g + s.witness) : nullptr, nullptr, nullptr, cuda_stream);
    if (vs != VOILA_OK) return vs;
    int32_t *best = reinterpret_cast<int32_t *>(g + s.scalars + 32);  // best q, best action
    if (best_q_out || best_action_out) {
        vs = voila_best_action(ctx, reinterpret_cast<const float *>(g + s.values),
                               reinterpret_cast<const int32_t *>(g + s.actions), Q, H, best, best + 1, cuda_stream);
        if (vs != VOILA_OK) return vs;
        if (best_q_out) e = cudaMemcpyAsync(best_q_out, best, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && best_action_out)
            e = cudaMemcpyAsync(best_action_out, best + 1, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
    }
    e = cudaMemcpyAsync(values_out, g + s.values, (size_t)Q * sizeof(float), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && obs_witness_out)
        e = cudaMemcpyAsync(obs_witness_out, g + s.witness, (size_t)Q * ctx->O * sizeof(float),
                            cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return VOILA_OK;
}

voila_status voila_belief_update_host(voila_ctx *ctx, const void *particles, int N, int32_t action,
                                      const float *observation, const float *weights, uint64_t seed,
                                      void *particles_out, float *weights_out, int32_t *ancestors_out,
                                      float *log_evidence_out, int32_t *status_out, void *cuda_stream) {
    if (!ctx || !particles || !observation || !particles_out || N < 1) return VOILA_ERR_INVALID_ARG;
    if (!ctx->stage || N > ctx->res_N) return VOILA_ERR_WORKSPACE;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const Stage s = make_stage(ctx, ctx->res_P, ctx->res_Q, ctx->res_H, ctx->res_N);
    uint8_t *g = reinterpret_cast<uint8_t *>(ctx->stage);
    const size_t esize = ctx->prec == VOILA_PREC_BF16 ? 2 : 4;
    const size_t pbytes = (size_t)N * ctx->S * esize;
    cudaError_t e = cudaMemcpyAsync(g + s.particles, particles, pbytes, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(g + s.obs, observation, (size_t)ctx->O * sizeof(float), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && weights)
        e = cudaMemcpyAsync(g + s.weights, weights, (size_t)N * sizeof(float), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    float *le = reinterpret_cast<float *>(g + s.scalars);
    int32_t *stat = reinterpret_cast<int32_t *>(g + s.scalars + 16);
    voila_status vs = voila_belief_update(
        ctx, g + s.particles, N, action, reinterpret_cast<const float *>(g + s.obs),
        weights ? reinterpret_cast<const float *>(g + s.weights) : nullptr, seed, g + s.particles_out,
        weights_out ? reinterpret_cast<float *>(g + s.weights_out) : nullptr,
        ancestors_out ? reinterpret_cast<int32_t *>(g + s.ancestors) : nullptr, nullptr, nullptr, le, stat,
        cuda_stream);
    if (vs != VOILA_OK) return vs;
    e = cudaMemcpyAsync(particles_out, g + s.particles_out, pbytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && weights_out)
        e = cudaMemcpyAsync(weights_out, g + s.weights_out, (size_t)N * sizeof(float), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && ancestors_out)
        e = cudaMemcpyAsync(ancestors_out, g + s.ancestors, (size_t)N * sizeof(int32_t), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && log_evidence_out)
        e = cudaMemcpyAsync(log_evidence_out, le, sizeof(float), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && status_out)
        e = cudaMemcpyAsync(status_out, stat, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return VOILA_OK;
}

}  // extern "C"
