// voila_kernels.h -- launchers implemented by the .cu files of libvoila (host-callable).
#pragma once
#include "voila_internal.h"

namespace voila {

// ---- mlp_ffma.cu : CUDA-core (FFMA) path, any dims; bf16 mode rounds operands to bf16 ----
size_t ffma_smem_bytes(const ModelDev &m);
cudaError_t launch_weight_sum(const float *weights, int n, double *wsum_out, cudaStream_t st);
cudaError_t launch_rollout_ffma(const ModelDev &m, const RolloutArgs &a, bool bf16, cudaStream_t st);
cudaError_t launch_rollout_reduce(const RolloutArgs &a, int O, const double *wsum, float *values,
                                  float *witness, cudaStream_t st);
cudaError_t launch_best_action(const float *values, const int32_t *seqs, int Q, int H, int32_t *best_q,
                               int32_t *best_action, cudaStream_t st);
cudaError_t launch_mlp_forward_ffma(const ModelDev &m, int which, const float *x, int rows, float *y,
                                    bool bf16, cudaStream_t st);
cudaError_t launch_bu_propose_score_ffma(const ModelDev &m, const BeliefArgs &a, bool bf16,
                                         cudaStream_t st);

// ---- belief.cu : normalise, uint64 decoupled-lookback scan, systematic resample + gather ----
constexpr int kScanTile = 4096;
struct ScanBuffers {
    ScanState *state;
    unsigned int *tile_flag;           // [tiles]
    unsigned long long *tile_agg;      // [tiles]
    unsigned long long *tile_incl;     // [tiles]
    double *tile_sumv;                 // [tiles]
    unsigned long long *cdf;           // [N]
    int *max_ordered;                  // [1]
    double *part_wsum;                 // [bu tiles]
};
inline int scan_tiles(int N) { return (N + kScanTile - 1) / kScanTile; }
cudaError_t launch_bu_init(const ScanBuffers &sb, int N, cudaStream_t st);
// bu_init fused with the observation tower e = f(o) (one observation): one launch, one CTA
bool obs_tower_fits(const MlpDev &f);
cudaError_t launch_bu_init_obs(const ScanBuffers &sb, int N, const MlpDev &f, const float *obs, float *e_out,
                               bool bf16, cudaStream_t st);
// What the scan's last CTA does once every tile is published (the former bu_finalize launch): W, the
// comb offset U, log evidence, status, the ESS decision.  enabled = 0: scan only (progressive widening).
struct FinalizeArgs {
    int enabled, n_wsum_parts, has_prior, from_logits;
    uint64_t seed;
    float ess_threshold;
    float *log_evidence_out, *ess_out;
    int32_t *dev_status_out, *resampled_out;
};
// from_logits: v_i = exp(L_i - max) (belief update) ; else v_i = in[i] (stage-level resampler)
cudaError_t launch_weight_scan(const ScanBuffers &sb, const float *in, int N, bool from_logits,
                               float *post_weights_out, cudaStream_t st, const FinalizeArgs *fin = nullptr);
// ess_threshold: resample iff ESS < ess_threshold * N (INFINITY: always); ess_out / resampled_out may be null
cudaError_t launch_bu_finalize(const ScanBuffers &sb, int N, int n_wsum_parts, bool has_prior,
                               uint64_t seed, float *log_evidence_out, int32_t *dev_status_out,
                               cudaStream_t st, float ess_threshold, float *ess_out, int32_t *resampled_out);
// w_in: the array the scan read (logits or weights): without resampling weights_out = v_k / sum v
cudaError_t launch_resample_gather(const ScanBuffers &sb, int N, const void *proposals,
                                   int row_bytes, void *particles_out, float *weights_out,
                                   int32_t *ancestors_out, cudaStream_t st, const float *w_in,
                                   bool from_logits);

// voila_resample_systematic_static: scratch in a file-scope device array of belief.cu (no allocation)
int static_resample_max_n();
size_t static_scratch_bytes();
cudaError_t launch_resample_systematic_static(const float *v, int N, uint64_t seed, int32_t *ancestors_out,
                                              int32_t *dev_status_out, cudaStream_t st, const char **why);

// ---- pw.cu / mlp_ffma.cu : vectorised progressive widening with batched likelihood (voila_pw_update) ----
cudaError_t launch_pw_widen(const PwArgs &a, cudaStream_t st);          // widen + child offsets + sorted order (3 launches)
cudaError_t launch_pw_propose_ffma(const ModelDev &m, const PwArgs &a, bool bf16, cudaStream_t st);
cudaError_t launch_pw_obs_ffma(const ModelDev &m, const PwArgs &a, bool bf16, cudaStream_t st);
cudaError_t launch_pw_score_ffma(const ModelDev &m, const PwArgs &a, bool bf16, cudaStream_t st);
cudaError_t launch_pw_weights(const PwArgs &a, cudaStream_t st);
bool tc2_has_diffusion(const void *tc2, int which);  // the denoiser program of that teacher was built
cudaError_t launch_diffusion_step_tc2(void *tc2, const ModelDev &m, const DiffusionArgs &a, int k, cudaStream_t st,
                                      std::string *kernel_name);
bool tc2_has_pw(const void *tc2);  // the per-row-action propose+score program was built
bool tc2_has_pw_slots(const void *tc2);  // ... and the two slot passes (opened branches, tower f)
cudaError_t launch_pw_slots_tc2(void *tc2, const ModelDev &m, const PwArgs &a, cudaStream_t st);
cudaError_t launch_pw_propose_score_tc2(void *tc2, const ModelDev &m, const PwArgs &a, const int32_t *sim_action,
                                        const int32_t *sim_seg, cudaStream_t st, std::string *kernel_name);
cudaError_t launch_pw_resample(const PwArgs &a, const unsigned long long *cdf, int row_bytes, cudaStream_t st);  // 1-2 launches

// ---- mlp_ffma.cu : one DDIM-ODE step of the diffusion teacher's sampler (voila_diffusion_sample) ----
cudaError_t launch_diffusion_step_ffma(const ModelDev &m, const DiffusionArgs &a, bool bf16, cudaStream_t st);

// ---- porpp.cu : one level of the PORPP preference backup (Eq. 1) ----
cudaError_t launch_porpp_backup_level(const float *R, const float *logpi0, const int32_t *child_off,
                                      const int32_t *child_idx, const float *child_w, const float *v_next,
                                      int n_belief, int A, float eta, float gamma, float *psi_out, float *v_out,
                                      cudaStream_t st, int32_t *argmax_out = nullptr);

// ---- rollout_tc.cu : tcgen05 / TMEM / bulk-copy path (bf16 mode) ----
bool tc_supported(const voila_model_desc *desc, std::string *why);
void *tc_create(const voila_model_desc *desc, int sm_count, std::vector<void *> *allocs,
                std::string *err);
void tc_destroy(void *tc);
bool tc_has_belief(const void *tc);  // the belief-update propose+score program was built too
cudaError_t launch_rollout_tc(void *tc, const ModelDev &m, const RolloutArgs &a, cudaStream_t st,
                              std::string *kernel_name, int *n_launches);
cudaError_t launch_bu_propose_score_tc(void *tc, const ModelDev &m, const BeliefArgs &a,
                                       cudaStream_t st, int *n_launches);

// ---- rollout_tc2.cu : CTA-pair (cta_group::2) tcgen05 path (bf16 mode) ----
bool tc2_supported(const voila_model_desc *desc, std::string *why);
void *tc2_create(const voila_model_desc *desc, int sm_count, std::vector<void *> *allocs,
                 std::string *err);
void tc2_destroy(void *tc2);
bool tc2_has_belief(const void *tc2);  // the belief-update propose+score program was built too
cudaError_t launch_rollout_tc2(void *tc2, const ModelDev &m, const RolloutArgs &a, cudaStream_t st,
                               std::string *kernel_name, int *n_launches);
// writes one prior-weight partial sum per 32 particles into a.part_wsum
cudaError_t launch_bu_propose_score_tc2(void *tc2, const ModelDev &m, const BeliefArgs &a,
                                        cudaStream_t st, int *n_launches, std::string *kernel_name);

}  // namespace voila
