// voila_internal.h -- host-side context and kernel parameter blocks of libvoila.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/voila.h"

namespace voila {

constexpr int kMaxLayers = 8;
constexpr int kTileRows = 32;  // rows (particles) per CTA in the CUDA-core kernels

// One MLP as the CUDA-core kernels see it: per layer a TRANSPOSED fp32 weight matrix
// Wt[l] = [dims[l]][dims[l+1]] (k-major so that lanes read consecutive output neurons) and bias.
struct MlpDev {
    int n_layers;
    int act;
    int dims[kMaxLayers + 1];
    const float *Wt[kMaxLayers];
    const float *b[kMaxLayers];
};

struct RewardDev {
    int kind;
    const float *param;        // goal[S] | M[S][S] | c[S+1]
    const float *action_cost;  // [A] or nullptr
};

// Terminal regions (voila_terminal): everything by value except the centres.
struct TerminalDev {
    int n;
    int dim[VOILA_MAX_TERMINAL_REGIONS], off[VOILA_MAX_TERMINAL_REGIONS], stop[VOILA_MAX_TERMINAL_REGIONS];
    float r2[VOILA_MAX_TERMINAL_REGIONS], reward[VOILA_MAX_TERMINAL_REGIONS];
    const float *centers;  // device, concatenated
};

struct ModelDev {
    int S, O, A, Nz;
    int lik_action_cond;
    float lambda, gamma;
    MlpDev mlp[6];  // 0 f_T, 1 f_Z, 2 f (obs tower), 3 g (state tower), 4 / 5 denoisers v_T / v_Z (n_layers 0: none)
    RewardDev reward;
    TerminalDev term;
    int max_width;  // widest activation vector over all four networks (incl. inputs)
};

struct RolloutArgs {
    const void *particles;  // [P][S] fp32 | bf16
    const int32_t *action_seqs;
    const float *weights;  // or nullptr
    int P, Q, H;
    uint64_t seed;
    double *part_value;    // [Q][tiles]
    double *part_witness;  // [Q][tiles][O] or nullptr
    float *returns_out;
    float *final_states_out;
    int tiles;
};

struct BeliefArgs {
    const void *particles;
    const float *weights;
    int N;
    int action;
    uint64_t seed;
    const float *e;        // f(o), [d]
    void *proposals;       // [N][S] fp32 | bf16
    float *logits;         // [N]
    int *max_ordered;      // [1]
    double *part_wsum;     // [tiles]
};

// voila_pw_update (progressive widening, pw.cu): arguments, outputs and workspace of one call.
constexpr int kPwMaxBranches = 64;  // M_max limit (per-warp counters in shared memory)
struct PwArgs {
    const void *particles;  // [N][S]
    const float *weights;   // [N] or nullptr
    int N, G, M_max;
    const int32_t *group_off, *group_action;
    int32_t *visit_count, *branch_count;
    float *branch_obs;      // [G][M_max][O]
    double k_o, alpha_o;
    uint64_t seed;
    // workspace
    int32_t *sim_group, *sim_branch, *sim_rank, *perm, *seg_of_pos;  // [N]
    int32_t *sim_action, *sim_seg;                                  // [N] action / child index of every simulation
    int obs_from_particles;  // 1: the sampled observations of opened branches recompute s' (no stored proposals yet)
    int32_t *seg_count, *seg_off, *new_src;                         // [G*M_max] (+1 for seg_off)
    int *seg_max;                                                   // [G*M_max] ordered-int maxima
    float *E;                                                       // [G*M_max][d] tower embeddings
    float *logits, *v_sorted;                                       // [N]
    void *proposals;                                                // [N][S]
    // outputs (any may be null)
    void *particles_out;
    float *weights_out, *post_weights_out;
    int32_t *ancestors_out, *sim_branch_out, *opened_out, *seg_status_out;
};

// voila_diffusion_sample: one DDIM-ODE step (one denoiser call) over all samples.
constexpr int kTemb = 8;  // width of the diffusion-time embedding (reading R31)
struct DiffusionArgs {
    const void *cond;        // [N][S]
    const int32_t *actions;  // [N]
    int N, which, D;         // D = S (transition teacher) | O (observation teacher)
    int first;               // 1: x = omega (Philox stream 7) instead of the stored state
    uint64_t seed;
    float temb[kTemb];       // temb(tau_k)
    float al, si, al_n, si_n;  // alpha, sigma at tau_k and at tau_{k+1}
    float *x;                // [N][D] fp32 state, updated in place (the caller's output buffer)
};

// Bookkeeping block of the scan / resample kernels (device memory, zeroed per call by a kernel).
struct ScanState {
    unsigned long long total_q;  // W
    unsigned long long offset_u; // U
    double sum_v;
    double sum_w;
    float max_logit;
    int status;
    unsigned int tile_counter;   // ticket: scan CTAs take their tile index in start order (look-back never waits on a later start)
    unsigned int done_counter;   // scan CTAs that have published everything: the last one finalises
    int resample;        // 1: resample (always, unless adaptive resampling found ESS >= threshold * N)
    double ess;          // effective sample size (sum v)^2 / sum v^2 of the posterior weights
    double inv_sum_v;    // 1 / sum v (normalised weights without resampling)
};

}  // namespace voila

struct voila_ctx {
    int device = 0;
    int sm_count = 0;
    int prec = 0;
    int kernel = 0;
    voila::ModelDev model{};      // pointers into dev_blob
    std::vector<void *> dev_allocs;
    // workspace
    void *ws = nullptr;
    size_t ws_bytes = 0;
    int res_P = 0, res_Q = 0, res_H = 0, res_N = 0;
    // workspace of voila_pw_update (voila_pw_reserve)
    void *pw_ws = nullptr;
    int pw_N = 0, pw_G = 0, pw_M = 0;
    // staging for *_host entry points
    void *stage = nullptr;
    size_t stage_bytes = 0;
    // tcgen05 path (opaque here; owned by rollout_tc.cu)
    void *tc = nullptr;
    // CTA-pair tcgen05 path (owned by rollout_tc2.cu)
    void *tc2 = nullptr;
    // profiling rings (voila_set_profiling): event pairs per kernel kind
    bool profiling = false;
    static constexpr int kProfRing = 256;
    cudaEvent_t prof_ev[4][kProfRing][2] = {};
    int prof_n[4] = {0, 0, 0, 0};
    uint64_t launches = 0;
    std::string last_rollout_kernel;
    std::string last_belief_kernel;
    std::string last_cuda_error;
    // host copies needed for validation
    int S = 0, O = 0, A = 0, Nz = 0, d = 0;
};
