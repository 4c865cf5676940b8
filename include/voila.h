/*
 * voila.h -- C ABI of libvoila: the data-parallel hot path of VOiLA's online planner on one B200.
 *
 * Paper: "VOiLA: Vectorized Online Planning with Learned Diffusion Models for POMDP Agents"
 * (arxiv/paper_2606_19729; citations are lines of /root/reference/PAPER.md).  The two hot calls:
 *
 *   voila_rollout_values  -- Monte-Carlo evaluation of candidate action sequences: every belief
 *       particle x every sequence is rolled forward through the distilled generators
 *       s' = f_T(s, a, w_T) (Eq.2) and o = f_Z(s', a, w_Z) (Eq.5, PAPER.md:124;
 *       "given batched states and actions"), the discounted return
 *       sum_t gamma^t R(s_t, a_t) is accumulated and averaged over the belief
 *       (Monte-Carlo estimate of R(b,a)).
 *   voila_belief_update   -- one step of the SIR particle filter that tracks the belief
 *       b'(s') ~ Z(s',a,o) sum_s T(s,a,s') b(s): propose with f_T, weight with
 *       exp(l(s',a,o)/lambda), normalise, resample.
 *
 * Everything the paper leaves open (two-tower l, Philox keying, exact-integer systematic
 * resampling, reward forms, bf16 mode) is fixed in DESIGN.md "Readings of the paper".
 *
 * Conventions
 *   - No torch / CUDA types in any signature: device pointers are plain pointers, the stream is a
 *     `void*` holding a cudaStream_t (NULL = legacy default stream).
 *   - "dev" = pointer to device memory on the ctx's GPU, "host" = pointer to host memory.
 *   - The caller owns every buffer it passes; the library owns only the ctx (packed weights and
 *     the workspace reserved with voila_reserve).  Hot calls never allocate.
 *   - Device entry points are asynchronous and stream-ordered; *_host entry points copy in, run,
 *     copy out and synchronise the stream before returning.
 *   - Particle state buffers are fp32 when the ctx was created with VOILA_PREC_FP32 and bf16
 *     (16-bit patterns) with VOILA_PREC_BF16; weights, values, observations are always fp32;
 *     indices are int32.  All dev pointers must be 16-byte aligned.
 *   - Results are a pure function of (inputs, seed): no hidden RNG state, no float atomics;
 *     repeated calls are bit-identical.
 *   - Errors found on the host return a status and enqueue nothing.  Conditions only the device can
 *     see (all weights zero, non-finite scores) set *dev_status_out != 0.
 *   - There is no CPU fallback: without a usable sm_100 device voila_create fails.
 *   - A ctx owns ONE workspace (voila_reserve): its calls must be issued on one stream at a time; two
 *     calls of the same ctx running concurrently on different streams race on it.  Use one ctx per stream.
 *   - If the rollout's weights sum to zero (or are not finite) values_out / obs_witness_out are NaN.
 *   - particles_out must alias neither particles nor proposals_out.
 *   - Tuning knobs read once by voila_create from the environment (A/B measurements only; the defaults are
 *     what the tests and bench.py run): VOILA_T2_BLOCK_POLICY (0..4: accumulator block shapes of the
 *     tcgen05 pair kernels), VOILA_T2_ROLLOUT_WARPS (8 | 16 epilogue warps of the rollout kernel),
 *     VOILA_T2_STAGES (2..8 weight-ring stages), VOILA_T2_STAGE_ROWS (128 | 256: 16 KB | 32 KB ring stages
 *     for every program), VOILA_T2_BELIEF_1SLOT / VOILA_T2_ROLLOUT_1SLOT (disable the two-slot belief /
 *     rollout programs), VOILA_T2_NO_PINGPONG (narrow one-slot rollouts: one TMEM accumulator region),
 *     VOILA_T2_DUAL_SPLIT (both epilogue sets share every hidden layer of a two-slot program).
 */
#ifndef VOILA_H_
#define VOILA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default) /* the library is built with -fvisibility=hidden */
#endif

typedef struct voila_ctx voila_ctx; /* opaque */

typedef enum {
    VOILA_OK = 0,
    VOILA_ERR_INVALID_ARG = 1, /* NULL / non-positive size / action out of range / misaligned pointer */
    VOILA_ERR_UNSUPPORTED = 2, /* no sm_100 device, or model dims over the kernels' limits */
    VOILA_ERR_CUDA = 3,        /* a CUDA runtime call failed; see voila_last_cuda_error */
    VOILA_ERR_WORKSPACE = 4    /* sizes exceed what voila_reserve was given (or VOILA_STATIC_MAX_N) */
} voila_status;

typedef enum { VOILA_ACT_NONE = 0, VOILA_ACT_RELU = 1, VOILA_ACT_SILU = 2 } voila_act;
typedef enum { VOILA_PREC_FP32 = 0, VOILA_PREC_BF16 = 1 } voila_prec;

/* A feed-forward network y = W_L act(... act(W_1 x + b_1) ...) + b_L (hidden activation `act`,
 * output layer linear).  Used for f_T, f_Z and the likelihood towers. */
typedef struct {
    int n_layers;            /* 1..8 affine layers */
    const int *dims;         /* host [n_layers+1]: dims[0] input width ... dims[n_layers] output */
    const float *const *W;   /* host [n_layers] pointers; W[l] is [dims[l+1]][dims[l]] row-major */
    const float *const *b;   /* host [n_layers] pointers; b[l] is [dims[l+1]] */
    int act;                 /* voila_act */
} voila_mlp;

/* R(s,a) (bounded reward on the current state-action).  DESIGN.md reading R14. */
typedef enum {
    VOILA_R_NEG_L2_GOAL = 0,   /* -||s - goal||_2        param = goal[S]            */
    VOILA_R_NEG_QUADRATIC = 1, /* -s^T M s               param = M[S][S] row-major  */
    VOILA_R_LINEAR = 2         /* c^T s + c0             param = c[S+1] (c0 last)   */
} voila_reward_kind;

typedef struct {
    int kind;                  /* voila_reward_kind */
    const float *param;        /* host, see above */
    const float *action_cost;  /* host [n_actions], added to R; or NULL */
} voila_reward;

/* Terminal regions of the rollout.  The paper's domains pay terminal rewards and end
 * the episode when the state reaches a region: FloorPositioning +100 at the correct goal (terminates),
 * -100 at the incorrect goal (does not), -1 per non-terminal action; LeggedNavigation
 * +500 in a goal disc of radius 2 m / -500 on collision, both terminate; TargetFinding
 * +100 / -500.  DESIGN.md reading R25: region k is the ball
 * || s[0:dims[k]] - center_k ||_2 <= radii[k] over the LEADING dims[k] state coordinates.  At a step t
 * of a trajectory that is still alive, every region containing s_t pays rewards[k]; if one of them
 * has stops[k] != 0 the episode ends there: R(s_t, a_t) (action cost included) is not paid, the state
 * is frozen (final_states_out returns it), no observation is drawn and nothing accrues afterwards;
 * otherwise R(s_t, a_t) is paid as usual.  Membership is decided in fp32 (on the bf16 state in bf16
 * mode): d2 = fma chain over j = 0 .. dims[k]-1 of (s_j - c_j)^2, inside iff d2 <= r*r. */
#define VOILA_MAX_TERMINAL_REGIONS 8
typedef struct {
    int n_regions;          /* 0 .. VOILA_MAX_TERMINAL_REGIONS */
    const int *dims;        /* host [n_regions]: 1 .. state_dim (1 .. 8 on the tensor-core path) */
    const float *centers;   /* host: the centres concatenated, sum(dims) floats */
    const float *radii;     /* host [n_regions], >= 0 */
    const float *rewards;   /* host [n_regions] */
    const int *stops;       /* host [n_regions]: != 0 ends the episode */
} voila_terminal;

typedef struct {
    int state_dim;   /* S */
    int obs_dim;     /* O */
    int n_actions;   /* A: discrete actions, one-hot encoded */
    int noise_dim;   /* Nz: w_T, w_Z ~ N(0, I_Nz) */
    voila_mlp f_T;        /* [S + A + Nz] -> ... -> S ; input order [s ; onehot(a) ; w] */
    voila_mlp f_Z;        /* [S + A + Nz] -> ... -> O ; evaluated on the successor state */
    voila_mlp lik_obs;    /* f : O -> ... -> d   (observation tower of l = <f(o), g(s')>) */
    voila_mlp lik_state;  /* g : S (+A if lik_action_cond) -> ... -> d */
    int lik_action_cond;  /* 0 | 1: append onehot(a) to g's input (PAPER.md:128 writes l(s',a,o)) */
    float lik_temperature; /* lambda > 0: weights are exp(l / lambda) */
    float discount;        /* gamma in (0, 1] */
    voila_reward reward;
    int prec;              /* voila_prec */
    const voila_terminal *terminal; /* terminal regions of the rollout, or NULL (none) */
    /* Denoisers of the diffusion teachers, n_layers = 0: none.
     * v_T : [S + A + S + 8] -> ... -> S, v_Z : [S + A + O + 8] -> ... -> O, input order
     * [c ; onehot(a) ; x_tau ; temb(tau)], temb = (sin(pi 2^k tau), cos(pi 2^k tau)) for k = 0..3 (reading R31). */
    voila_mlp denoise_T, denoise_Z;
} voila_model_desc;

/* Which kernel family runs the generator MLPs (for tests and benchmarks; default AUTO). */
typedef enum {
    VOILA_KERNEL_AUTO = 0,   /* tcgen05 path when prec == BF16 and the dims fit it, else FFMA */
    VOILA_KERNEL_FFMA = 1,   /* CUDA-core path (fp32 mode; in bf16 mode rounds operands to bf16) */
    VOILA_KERNEL_TCGEN05 = 2, /* single-CTA tensor-core path (M = 128 per SM); UNSUPPORTED if the dims do not
                                 fit or the model has terminal regions */
    VOILA_KERNEL_TCGEN05_PAIR = 3 /* CTA-pair tensor-core path (cta_group::2, M = 256 per SM pair): what AUTO picks */
} voila_kernel;

/* Copies and packs the host weights onto `device`.  Fails with VOILA_ERR_UNSUPPORTED when the
 * device is not compute capability 10.x or a layer is wider than the kernels handle.  *out is set
 * only on VOILA_OK. */
voila_status voila_create(const voila_model_desc *desc, int device, voila_ctx **out);
void voila_destroy(voila_ctx *ctx);

/* Bytes of device workspace needed for rollouts of P particles x Q sequences x H steps and belief
 * updates of N particles (any of them may be 0). */
size_t voila_workspace_bytes(const voila_ctx *ctx, int P, int Q, int H, int N);
/* (Re)allocates the ctx-owned workspace (and, for the *_host entry points, staging buffers) for
 * those maximum sizes.  Not a hot call: synchronises the device. */
voila_status voila_reserve(voila_ctx *ctx, int P, int Q, int H, int N);

voila_status voila_set_kernel(voila_ctx *ctx, int kernel /* voila_kernel */);
/* 1 if the tcgen05 rollout / belief kernels support this ctx's dims, else 0. */
int voila_tcgen05_supported(const voila_ctx *ctx);

/*
 * V_q = sum_p wbar_p sum_{t<H} gamma^t R(s_t, a_{q,t}),  s_0 = particles[p],
 * s_{t+1} = f_T(s_t, a_{q,t}, w_T(p,q,t)),  o_{t+1} = f_Z(s_{t+1}, a_{q,t}, w_Z(p,q,t)),
 * wbar_p = weights[p] / sum weights   (O4).
 *   particles        dev [P][S]   fp32 | bf16 (see prec)
 *   action_seqs      dev [Q][H]   int32 in [0, A)   (an out-of-range entry is clamped into [0, A) by the kernels)
 *   weights          dev [P] fp32 >= 0, unnormalised; NULL = uniform
 *   seed             keys the Philox4x32-10 noise: counter (p, q, t, stream<<16 | block)
 *   values_out       dev [Q] fp32
 *   obs_witness_out  dev [Q][O] fp32 or NULL: sum_p wbar_p sum_t gamma^t o_{t+1} (R10)
 *   returns_out      dev [Q][P] fp32 or NULL: per-(q,p) discounted return (tests)
 *   final_states_out dev [Q][P][S] fp32 or NULL: s_H of every trajectory, or the state at which it
 *                    terminated (voila_terminal) (tests)
 * With terminal regions (voila_model_desc.terminal) the sums stop at the step a trajectory ends.
 */
voila_status voila_rollout_values(voila_ctx *ctx, const void *particles, int P,
                                  const int32_t *action_seqs, int Q, int H, const float *weights,
                                  uint64_t seed, float *values_out, float *obs_witness_out,
                                  float *returns_out, float *final_states_out, void *cuda_stream);

/*
 * SIR step (O5):
 *   s'_i = f_T(s_i, a, w(i)),  L_i = log w_i + <f(o), g(s'_i)> / lambda,  m = max L,
 *   v_i = exp(L_i - m),  ancestors = systematic resample of v (exact integer definition, O7),
 *   particles_out[k] = s'_{ancestors[k]},  weights_out[k] = 1/N.
 *   particles         dev [N][S] fp32 | bf16
 *   observation       dev [O] fp32
 *   weights           dev [N] fp32 >= 0 or NULL (uniform)
 *   particles_out     dev [N][S] same type as particles; must not alias particles
 *   weights_out       dev [N] fp32 or NULL
 *   ancestors_out     dev [N] int32 or NULL (non-decreasing)
 *   post_weights_out  dev [N] fp32 or NULL: v_i (max = 1)
 *   proposals_out     dev [N][S] same type as particles, or NULL: s'_i before resampling
 *   log_evidence_out  dev [1] fp32 or NULL: m + log sum v - log sum w
 *   dev_status_out    dev [1] int32 or NULL: 0 ok; 1 all weights zero or non-finite scores
 *                     (then ancestors = identity and particles_out = proposals)
 */
voila_status voila_belief_update(voila_ctx *ctx, const void *particles, int N, int32_t action,
                                 const float *observation, const float *weights, uint64_t seed,
                                 void *particles_out, float *weights_out, int32_t *ancestors_out,
                                 float *post_weights_out, void *proposals_out,
                                 float *log_evidence_out, int32_t *dev_status_out,
                                 void *cuda_stream);

/* Stage-level entry points (so that "indices bit-exact given identical weights" is testable). */

/* ancestors_out[k] = min{ i : N*C_i > k*W + U }, q_i = floor(v_i 2^32), C = inclusive scan of q,
 * W = C_{N-1}, U = (x0*W) >> 32 with x0 the Philox word of (seed, stream 4).  v dev [N] in [0,1].
 * dev_status_out as above (1 when every q_i is 0). */
voila_status voila_resample_systematic(voila_ctx *ctx, const float *v, int N, uint64_t seed,
                                       int32_t *ancestors_out, int32_t *dev_status_out,
                                       void *cuda_stream);

/* The same resampler for callers that may not allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): no ctx, no workspace, NO cudaMalloc / cudaFree or allocating
 * library call inside; three kernel launches on `cuda_stream` of the CURRENT device.  Its scratch (the
 * uint64 CDF, the look-back tile records, the scan bookkeeping) is one static device array of
 * 8 MiB + 16 KiB that every GPU loading libvoila holds until exit, hence the limit
 * N <= VOILA_STATIC_MAX_N (2^20).  Arguments and results exactly as voila_resample_systematic
 * (v, ancestors_out, dev_status_out are device pointers, 16-byte aligned; dev_status_out may be NULL).
 * All calls share that one array: calls that may overlap on the GPU (different streams, different host
 * threads) race on it -- issue them on one stream, or order them with events.  The array keeps the last
 * call's contents; every call clears what must start at zero itself.
 * Errors: VOILA_ERR_INVALID_ARG for NULL / N < 1 / misaligned pointers; VOILA_ERR_WORKSPACE for
 * N > VOILA_STATIC_MAX_N (nothing is launched); VOILA_ERR_CUDA when a runtime call fails.
 * voila_static_last_error() returns the calling thread's last message of this entry point ("" if none). */
#define VOILA_STATIC_MAX_N (1 << 20)
voila_status voila_resample_systematic_static(const float *v, int N, uint64_t seed, int32_t *ancestors_out,
                                              int32_t *dev_status_out, void *cuda_stream);
const char *voila_static_last_error(void);

/* y = MLP_which(x): which = 0 f_T, 1 f_Z, 2 f (obs tower), 3 g (state tower).
 * x dev [rows][dims[0]] fp32 (the full input, one-hot block included), y dev [rows][dims[L]] fp32.
 * Arithmetic follows the ctx precision (bf16 mode rounds weights and layer inputs to bf16). */
voila_status voila_mlp_forward(voila_ctx *ctx, int which, const float *x, int rows, float *y,
                               void *cuda_stream);

/* One level of the PORPP preference backup (Eq. 1) on a belief tree
 * stored as tensors: the level has n_belief belief nodes with n_actions action nodes each (action
 * node j = b * n_actions + a); action node j owns the observation branches
 * child_idx[child_off[j] .. child_off[j+1]) (belief nodes of the NEXT level) with weights
 * child_w = Z(b,a,o):
 *   Psi(b,a) = logpi0[j] / eta + R[j] + gamma * sum_c child_w[c] * v_next[child_idx[c]]
 *   V(b)     = (1/eta) log sum_a exp(eta * Psi(b,a))           (max-shifted)
 * Call once per level, deepest level first, feeding v_out of a level as v_next of the one above.
 *   R, logpi0 dev [n_belief * n_actions] fp32; child_off dev [n_belief * n_actions + 1] int32;
 *   child_idx dev int32 / child_w dev fp32 [child_off[last]] (may be NULL when there are no
 *   branches); v_next dev fp32 (may be NULL when there are no branches);
 *   psi_out dev [n_belief * n_actions] fp32, v_out dev [n_belief] fp32.
 * Errors: VOILA_ERR_INVALID_ARG for NULL / non-positive sizes, eta <= 0, gamma < 0. */
voila_status voila_porpp_backup_level(voila_ctx *ctx, const float *R, const float *logpi0,
                                      const int32_t *child_off, const int32_t *child_idx, const float *child_w,
                                      const float *v_next, int n_belief, int n_actions, float eta, float gamma,
                                      float *psi_out, float *v_out, void *cuda_stream);

/* The preference backup of a WHOLE belief tree in one call, and the root action (VOPP
 * stores the tree as "a collection of tensors storing belief nodes, action nodes, and action
 * preferences" and interleaves forward search with "fully vectorized preference backup"; the planner
 * then acts on the root preferences).  levels is a HOST array of n_levels records holding DEVICE
 * pointers, level 0 = the root level; level d's observation branches index the belief nodes of level
 * d + 1 (the last level's index leaf_values).  Levels are backed up deepest first on the stream, each
 * level's v_out feeding the level above; psi_out / v_out of every level are written.
 *   root_action_out dev [levels[0].n_belief] int32 or NULL: argmax_a Psi(b0, a), ties -> lowest a,
 *                   a NaN preference never wins.
 * Errors as voila_porpp_backup_level, plus n_levels < 1. */
typedef struct {
    const float *R, *logpi0;     /* dev [n_belief * n_actions] */
    const int32_t *child_off;    /* dev [n_belief * n_actions + 1] */
    const int32_t *child_idx;    /* dev [child_off[last]] or NULL */
    const float *child_w;        /* dev [child_off[last]] or NULL */
    int n_belief;
    float *psi_out;              /* dev [n_belief * n_actions] */
    float *v_out;                /* dev [n_belief] */
} voila_porpp_level;
voila_status voila_porpp_backup(voila_ctx *ctx, const voila_porpp_level *levels, int n_levels, int n_actions,
                                const float *leaf_values, float eta, float gamma, int32_t *root_action_out,
                                void *cuda_stream);

/* Root action selection for an open-loop sequence sweep: q* = argmax_q values[q] (ties -> lowest q,
 * NaN never wins), best_action_out[0] = action_seqs[q*][0], best_q_out[0] = q* (the
 * planner returns an action for the current belief; DESIGN.md input recipe, config 5).
 *   values dev [Q] fp32, action_seqs dev [Q][H] int32, best_q_out / best_action_out dev [1] int32
 *   (best_q_out may be NULL). */
voila_status voila_best_action(voila_ctx *ctx, const float *values, const int32_t *action_seqs, int Q,
                               int H, int32_t *best_q_out, int32_t *best_action_out,
                               void *cuda_stream);

/* Belief update with ADAPTIVE resampling (the SIR filter of PAPER.md:77 with the
 * usual effective-sample-size criterion): ESS = (sum_i v_i)^2 / sum_i v_i^2 of the posterior weights
 * v_i = exp(L_i - max L).  The filter resamples iff ESS < ess_threshold * N; otherwise
 * particles_out = proposals, ancestors_out[k] = k and weights_out[k] = v_k / sum v (the normalised
 * weights are carried to the next update).  ess_threshold > 0; INFINITY = always resample, which is
 * exactly voila_belief_update.  Every other argument as in voila_belief_update, plus
 *   ess_out dev [1] fp32 or NULL, resampled_out dev [1] int32 (1 | 0) or NULL.
 * Errors: VOILA_ERR_INVALID_ARG for ess_threshold <= 0 or NaN. */
voila_status voila_belief_update_ess(voila_ctx *ctx, const void *particles, int N, int32_t action,
                                     const float *observation, const float *weights, uint64_t seed,
                                     float ess_threshold, void *particles_out, float *weights_out,
                                     int32_t *ancestors_out, float *post_weights_out, void *proposals_out,
                                     float *log_evidence_out, float *ess_out, int32_t *resampled_out,
                                     int32_t *dev_status_out, void *cuda_stream);

/* Vectorised progressive widening with batched likelihood (section 4.3:
 * "an action node a is expanded with a sampled observation whenever |C(a)| < k_o N(a)^alpha_o ...
 * Otherwise, the sampled successor state is associated with a previously existing observation branch
 * of the same action node.  The likelihood model l(s', a, o) is then used to weight successor states
 * according to the observation stored at the selected branch, followed by resampling ... parallel
 * simulations are grouped by their parent action nodes, after which the above PW operations are
 * performed for all action-node groups in parallel").  DESIGN.md readings R26-R29 fix what the paper
 * leaves open.  N simulations, grouped: action node g owns the simulations
 * [group_off[g], group_off[g+1]) and has the action group_action[g], the visit count visit_count[g] =
 * N(a), branch_count[g] = |C(a)| stored observation branches branch_obs[g][0 .. |C(a)|) (M_max rows of O
 * floats reserved per node).  For every simulation i of node g, in index order:
 *   s'_i = f_T(s_i, a_g, w_T(i)) (Philox stream 3, counter (i,0,0)),
 *   N(a) += 1; if |C(a)| < min(M_max, ceil(k_o N(a)^alpha_o (1 - 1e-9))) the simulation opens branch |C(a)|,
 *   storing o_i = f_Z(s'_i, a_g, w_Z(i)) (stream 5), and is attached to it; otherwise it is attached to
 *   the existing branch (x_i |C(a)|) >> 32, x_i one Philox word (stream 6);
 *   L_i = log w_i + <f(obs_{g,b(i)}), g(s'_i)> / lambda  (every stored observation goes through the tower f
 *   as one batch).
 * Every (node, branch) pair that received simulations is a child belief: its members (in index order)
 * are resampled among themselves with the exact-integer systematic resampler (v = exp(L - max over the
 * child), offset word keyed by g*M_max+b); the r-th member receives the r-th draw.
 *   particles      dev [N][S] fp32 | bf16        group_off dev [G+1] int32 (group_off[0] = 0, [G] = N)
 *   group_action   dev [G] int32 in [0, A)       visit_count, branch_count dev [G] int32, updated in place
 *   branch_obs     dev [G][M_max][O] fp32, rows of opened branches are written      1 <= M_max <= 64
 *   weights        dev [N] fp32 >= 0 or NULL     k_o > 0, alpha_o > 0
 *   particles_out  dev [N][S] or NULL: s' of the simulation's draw;  weights_out dev [N] or NULL: 1 / members
 *   ancestors_out  dev [N] int32 or NULL: simulation index of the draw (a member of the same child)
 *   sim_branch_out dev [N] int32 or NULL;  opened_out dev [N] int32 or NULL (1: opened its branch)
 *   post_weights_out dev [N] fp32 or NULL: v_i;  proposals_out dev [N][S] or NULL: s'_i
 *   seg_status_out dev [G*M_max] int32 or NULL: 1 for a child whose weights are all zero / not finite
 *                  (its members keep themselves), else 0
 * The group arrays are not validated on the device (offsets must be non-decreasing, actions in range,
 * 0 <= branch_count <= M_max).  Needs voila_pw_reserve(N, G, M_max) first (VOILA_ERR_WORKSPACE otherwise).
 * Errors: VOILA_ERR_INVALID_ARG for NULL / non-positive sizes, M_max > 64, k_o <= 0, alpha_o <= 0. */
size_t voila_pw_workspace_bytes(const voila_ctx *ctx, int N, int G, int M_max);
voila_status voila_pw_reserve(voila_ctx *ctx, int N, int G, int M_max);
voila_status voila_pw_update(voila_ctx *ctx, const void *particles, int N, const int32_t *group_off, int G,
                             const int32_t *group_action, int32_t *visit_count, int32_t *branch_count,
                             float *branch_obs, int M_max, double k_o, double alpha_o, const float *weights,
                             uint64_t seed, void *particles_out, float *weights_out, int32_t *ancestors_out,
                             int32_t *sim_branch_out, int32_t *opened_out, float *post_weights_out,
                             void *proposals_out, int32_t *seg_status_out, void *cuda_stream);

/* The diffusion teacher's sampler.  The paper distils "an ODE-based diffusion sampler
 * [27]" of a conditional denoiser trained with the v-prediction objective and a cosine schedule
 * into f_T / f_Z, and reports the sampling cost of both; this call is
 * that teacher (readings R30-R32): abar_tau = cos^2(pi tau / 2); uniform grid tau_k = 1 - k/K;
 * x at tau = 1 is omega ~ N(0, I_D) (Philox stream 7, counter (i, 0, 0)); for k = 0 .. K-1
 *   v = v_theta(c_i, a_i, x, tau_k);  x0 = alpha x - sigma v;  eps = sigma x + alpha v;
 *   x <- alpha' x0 + sigma' eps            (DDIM, eta = 0; K denoiser calls per sample)
 * and x at tau = 0 is the sample.  which = 0: transition teacher (c = s, D = S), 1: observation teacher
 * (c = s', D = O).
 *   cond    dev [N][S] fp32 | bf16 (see prec)      actions dev [N] int32 in [0, A) (not range-checked)
 *   out     dev [N][D] fp32: the samples (also the state of the recursion between the K launches)
 * Errors: VOILA_ERR_INVALID_ARG for NULL / N < 1 / K < 1 / K > 256, VOILA_ERR_UNSUPPORTED when the model
 * has no such denoiser. */
voila_status voila_diffusion_sample(voila_ctx *ctx, int which, const void *cond, const int32_t *actions, int N,
                                    int K, uint64_t seed, float *out, void *cuda_stream);

/* Host-buffer variants: every pointer is HOST memory (pinned for best speed); inputs are copied to
 * ctx-owned device staging buffers, the device entry point runs, outputs are copied back and the
 * stream is synchronised.  Optional outputs as above (NULL to skip). */
voila_status voila_rollout_values_host(voila_ctx *ctx, const void *particles, int P,
                                       const int32_t *action_seqs, int Q, int H,
                                       const float *weights, uint64_t seed, float *values_out,
                                       float *obs_witness_out, void *cuda_stream);
/* The whole planning half through host buffers: the rollout, then the executed action (the first action
 * of argmax_q V_q, voila_best_action) on the device; best_q_out / best_action_out host [1] int32 or NULL. */
voila_status voila_plan_host(voila_ctx *ctx, const void *particles, int P, const int32_t *action_seqs, int Q,
                             int H, const float *weights, uint64_t seed, float *values_out,
                             float *obs_witness_out, int32_t *best_q_out, int32_t *best_action_out,
                             void *cuda_stream);
voila_status voila_belief_update_host(voila_ctx *ctx, const void *particles, int N, int32_t action,
                                      const float *observation, const float *weights,
                                      uint64_t seed, void *particles_out, float *weights_out,
                                      int32_t *ancestors_out, float *log_evidence_out,
                                      int32_t *status_out, void *cuda_stream);

/* Introspection used by bench.py: number of kernel launches the library has enqueued on this ctx
 * since creation, and the name / launch geometry of the last rollout kernel. */
uint64_t voila_launch_count(const voila_ctx *ctx);
const char *voila_last_rollout_kernel(const voila_ctx *ctx);
/* Name of the propose+score kernel the last voila_belief_update launched. */
const char *voila_last_belief_kernel(const voila_ctx *ctx);

/* Kernel timing for bench.py's roofline line.  When profiling is on, the library brackets each
 * launch of its main kernels with CUDA events on the caller's stream (a ring of 256 pairs per
 * kernel kind).  voila_profile_read waits for the recorded events of `which`, writes up to max_n
 * durations in milliseconds (oldest first) to the HOST array ms_out, clears the ring for that
 * kind and returns how many it wrote.  which: 0 rollout kernel, 1 belief propose+score kernel,
 * 2 weight scan kernel, 3 resample+gather kernel. */
typedef enum { VOILA_K_ROLLOUT = 0, VOILA_K_PROPOSE = 1, VOILA_K_SCAN = 2, VOILA_K_RESAMPLE = 3 } voila_kernel_kind;
voila_status voila_set_profiling(voila_ctx *ctx, int on);
int voila_profile_read(voila_ctx *ctx, int which, float *ms_out, int max_n);

const char *voila_status_string(voila_status s);
const char *voila_last_cuda_error(const voila_ctx *ctx);
int voila_version(void);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif /* VOILA_H_ */
