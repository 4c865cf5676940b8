/*
 * voila_oracle.c -- plain CPU oracle for the VOiLA planner hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path under paper_2606_19729_b200/csrc/.
 *
 * What it computes (all citations are /root/reference/PAPER.md:<line>):
 *   - the vectorised Monte-Carlo evaluation of (particle x action-sequence) rollouts through
 *     the distilled generators  s' = f_T(s,a,w_T)  (Eq.2),
 *     o = f_Z(s',a,w_Z) (Eq.5; "given batched states and actions"),
 *     with the discounted return  sum_t gamma^t R(s_t,a_t) and the Monte-Carlo
 *     belief average of R;
 *   - the SIR particle-filter belief update: propose with f_T, weight with
 *     exp(l(s',a,o)/lambda), resample.
 * Everything the paper leaves open (two-tower likelihood, Philox keying, Box-Muller, integer
 * systematic resampling, reward forms) follows DESIGN.md "Readings of the paper" R1..R20,
 * which restate SURVEY.md section 8(c).
 *
 * Arithmetic: `real` is float (the north_star fixes the oracle to fp32).  The same source
 * compiled with -DVO_REAL=double gives an fp64 build used only to *derive* tolerances
 * (how far fp32 itself is from the exact value); noise normals are always produced in fp32
 * (reading R4) so both builds and the GPU see the same random numbers.
 * Cross-particle sums (value, witness, evidence) are accumulated in double in both builds.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   vo_philox4x32_10   : Random123 known-answer vectors (tests/golden/philox4x32_10_kat.txt)
 *   vo_normals         : sample moments, |z| bound, counter layout brute force
 *   vo_mlp_forward     : torch.nn.functional.linear chain (library special case), hand 2x2
 *   vo_rollout_values  : linear generators (closed form), identity-ReLU generator, constant
 *                        reward geometric series, depth-2 brute-force enumeration, stochastic
 *                        linear moments
 *   vo_belief_update   : exponential-tilt closed form (Gaussian proposals, linear towers),
 *                        shift invariance, lambda->inf, scipy.special.logsumexp
 *   vo_resample_*      : count invariants, uniform->identity, one-hot, dyadic weights vs
 *                        numpy.searchsorted, brute force over all offsets for N<=4
 * No function here is "parity unpinned".
 *
 * No blocking, fusion or reordering: every loop is the textbook loop.  OpenMP is used only
 * over independent (sequence) / (particle) units and never changes any result.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef VO_REAL
#define VO_REAL float
#endif
typedef VO_REAL real;

#define VO_MAX_LAYERS 8
#define VO_MAX_TERM 8
#define VO_ACT_NONE 0
#define VO_ACT_RELU 1
#define VO_ACT_SILU 2
#define VO_R_NEG_L2_GOAL 0
#define VO_R_NEG_QUADRATIC 1
#define VO_R_LINEAR 2

/* Noise streams (reading R3): which Philox stream feeds which random input. */
#define VO_STREAM_ROLLOUT_T 1u
#define VO_STREAM_ROLLOUT_Z 2u
#define VO_STREAM_BELIEF_T 3u
#define VO_STREAM_RESAMPLE 4u
#define VO_STREAM_PW_OBS 5u    /* progressive widening: noise of the sampled observation o_i */
#define VO_STREAM_PW_ATTACH 6u /* progressive widening: word that picks an existing branch */
#define VO_STREAM_DIFFUSION 7u /* diffusion teacher: the initial noise x_1 = omega */
#define VO_TEMB 8              /* width of the diffusion-time embedding (reading R31) */

typedef struct {
    int n_layers;                 /* number of affine layers */
    int dims[VO_MAX_LAYERS + 1];  /* dims[0] = input width ... dims[n_layers] = output width */
    int act;                      /* hidden activation; the output layer is linear */
    real *W[VO_MAX_LAYERS];       /* W[l] is [dims[l+1]][dims[l]] row-major: y = W x + b */
    real *b[VO_MAX_LAYERS];
} vo_mlp;

typedef struct {
    int S, O, A, Nz;
    vo_mlp mlp[6]; /* 0: f_T, 1: f_Z, 2: obs tower f, 3: state tower g, 4 / 5: diffusion teachers' denoisers v_T / v_Z */
    int lik_action_cond;
    float lambda, gamma;
    int reward_kind;
    real *reward_param; /* goal[S] | M[S][S] | c[S+1] */
    real *action_cost;  /* [A] or NULL */
    int emulate_bf16;   /* debugging hook, see vo_model_set_emulate_bf16 */
    /* terminal regions, see vo_model_set_terminal */
    int n_term;
    int term_dim[VO_MAX_TERM];
    float *term_center[VO_MAX_TERM];
    float term_radius[VO_MAX_TERM], term_reward[VO_MAX_TERM];
    int term_stop[VO_MAX_TERM];
} vo_model;

/* ------------------------------------------------------------------------------------------
 * bf16 emulation hook (reading R18): round-to-nearest-even to 8 significant bits.  Used only
 * to separate "bf16 rounding" from "kernel bug" in tests; the oracle proper is fp32.
 * ---------------------------------------------------------------------------------------- */
static float bf16_round(float x) {
    uint32_t u;
    memcpy(&u, &x, 4);
    if ((u & 0x7f800000u) == 0x7f800000u) return x; /* inf / nan unchanged */
    u += 0x7fffu + ((u >> 16) & 1u);
    u &= 0xffff0000u;
    memcpy(&x, &u, 4);
    return x;
}

/* ------------------------------------------------------------------------------------------
 * O1. Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  ctr/key/out are 32-bit words.
 * ---------------------------------------------------------------------------------------- */
void vo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        if (round < 9) { k0 += W0; k1 += W1; }
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* O2. uniform in (0,1] from one 32-bit word, then Box-Muller on word pairs (reading R4). */
static float u01(uint32_t x) { return fmaf((float)x, 0x1p-32f, 0x1p-33f); }

static void box_muller(uint32_t xa, uint32_t xb, float *z0, float *z1) {
    float ua = u01(xa), ub = u01(xb);
    float r = sqrtf(-2.0f * logf(ua));
    float ang = 6.283185307179586f * ub;
    *z0 = r * cosf(ang);
    *z1 = r * sinf(ang);
}

/* n standard normals for the random input keyed by (seed; p, q, t, stream) (reading R3):
 * key = (seed lo, seed hi), counter = (p, q, t, stream<<16 | blk), component j uses block
 * blk = j/4 and output word j%4. */
void vo_normals(uint64_t seed, uint32_t p, uint32_t q, uint32_t t, uint32_t stream, int n,
                float *out) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    for (int blk = 0; 4 * blk < n; ++blk) {
        uint32_t ctr[4] = {p, q, t, (stream << 16) | (uint32_t)blk}, x[4];
        float z[4];
        vo_philox4x32_10(ctr, key, x);
        box_muller(x[0], x[1], &z[0], &z[1]);
        box_muller(x[2], x[3], &z[2], &z[3]);
        for (int j = 0; j < 4 && 4 * blk + j < n; ++j) out[4 * blk + j] = z[j];
    }
}

/* The single word that places the systematic-resampling comb (stream 4, reading R3). */
uint32_t vo_resample_word(uint64_t seed) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t ctr[4] = {0, 0, 0, VO_STREAM_RESAMPLE << 16}, x[4];
    vo_philox4x32_10(ctr, key, x);
    return x[0];
}

/* ------------------------------------------------------------------------------------------
 * Model handle
 * ---------------------------------------------------------------------------------------- */
vo_model *vo_model_create(int S, int O, int A, int Nz, int lik_action_cond, float lambda,
                          float gamma) {
    vo_model *m = (vo_model *)calloc(1, sizeof(vo_model));
    m->S = S; m->O = O; m->A = A; m->Nz = Nz;
    m->lik_action_cond = lik_action_cond;
    m->lambda = lambda; m->gamma = gamma;
    return m;
}

/* which: 0 f_T, 1 f_Z, 2 f (obs tower), 3 g (state tower).  W_flat / b_flat are the layers'
 * fp32 parameters concatenated in layer order (W[l] is [out][in] row-major). */
int vo_model_set_mlp(vo_model *m, int which, int n_layers, const int *dims, int act,
                     const float *W_flat, const float *b_flat) {
    if (which < 0 || which > 5 || n_layers < 1 || n_layers > VO_MAX_LAYERS) return -1;
    vo_mlp *f = &m->mlp[which];
    f->n_layers = n_layers; f->act = act;
    for (int l = 0; l <= n_layers; ++l) f->dims[l] = dims[l];
    size_t wo = 0, bo = 0;
    for (int l = 0; l < n_layers; ++l) {
        size_t nw = (size_t)dims[l] * dims[l + 1], nb = (size_t)dims[l + 1];
        free(f->W[l]); free(f->b[l]);
        f->W[l] = (real *)malloc(nw * sizeof(real));
        f->b[l] = (real *)malloc(nb * sizeof(real));
        for (size_t i = 0; i < nw; ++i) f->W[l][i] = (real)W_flat[wo + i];
        for (size_t i = 0; i < nb; ++i) f->b[l][i] = (real)b_flat[bo + i];
        wo += nw; bo += nb;
    }
    return 0;
}

int vo_model_set_reward(vo_model *m, int kind, const float *param, const float *action_cost) {
    int n = kind == VO_R_NEG_L2_GOAL ? m->S : kind == VO_R_NEG_QUADRATIC ? m->S * m->S : m->S + 1;
    if (kind < 0 || kind > 2) return -1;
    m->reward_kind = kind;
    free(m->reward_param); free(m->action_cost);
    m->reward_param = (real *)malloc((size_t)n * sizeof(real));
    for (int i = 0; i < n; ++i) m->reward_param[i] = (real)param[i];
    m->action_cost = NULL;
    if (action_cost) {
        m->action_cost = (real *)malloc((size_t)m->A * sizeof(real));
        for (int i = 0; i < m->A; ++i) m->action_cost[i] = (real)action_cost[i];
    }
    return 0;
}

/* Terminal regions.  The paper's three domains pay terminal rewards and end the
 * episode when the state reaches a region of the state space: FloorPositioning +100 at the correct
 * goal (terminates) and -100 at the incorrect goal (does not), -1 per non-terminal action
 * (PAPER.md:161); LeggedNavigation +500 in a goal disc of radius 2 m, -500 on collision, both
 * terminate; TargetFinding +100 / -500.  Reading (R25):
 * region k is a ball over the LEADING dim_k state coordinates, || s[0:dim_k] - c_k ||_2 <= r_k;
 * at a step t that is still alive, every region containing s_t pays reward_k; if one of them has
 * stop_k the episode ends there: the step reward R(s_t, a_t) (incl. the action cost) is NOT paid,
 * the state is frozen, nothing accrues afterwards; otherwise R(s_t, a_t) is paid as usual.
 * Membership is decided in fp32: d2 = fma chain over j = 0..dim_k-1 of (s_j - c_j)^2, inside iff
 * d2 <= r_k * r_k (both sides take the decision in this precision and order). */
int vo_model_set_terminal(vo_model *m, int n, const int *dims, const float *centers, const float *radii,
                          const float *rewards, const int *stops) {
    if (n < 0 || n > VO_MAX_TERM) return -1;
    for (int k = 0; k < VO_MAX_TERM; ++k) { free(m->term_center[k]); m->term_center[k] = NULL; }
    m->n_term = n;
    size_t off = 0;
    for (int k = 0; k < n; ++k) {
        if (dims[k] < 1 || dims[k] > m->S) return -1;
        m->term_dim[k] = dims[k];
        m->term_center[k] = (float *)malloc(sizeof(float) * (size_t)dims[k]);
        for (int j = 0; j < dims[k]; ++j) m->term_center[k][j] = centers[off + j];
        off += (size_t)dims[k];
        m->term_radius[k] = radii[k];
        m->term_reward[k] = rewards[k];
        m->term_stop[k] = stops[k] ? 1 : 0;
    }
    return 0;
}

/* bf16-emulation hook: when on, weights (already stored) are rounded once to bf16 and every
 * layer's INPUT vector is rounded to bf16 before the affine map; accumulation, bias, activation
 * stay in `real`.  Call after all vo_model_set_mlp calls.  Not part of the oracle proper. */
void vo_model_set_emulate_bf16(vo_model *m, int on) {
    m->emulate_bf16 = on;
    if (!on) return;
    for (int w = 0; w < 6; ++w)
        for (int l = 0; l < m->mlp[w].n_layers; ++l) {
            size_t nw = (size_t)m->mlp[w].dims[l] * m->mlp[w].dims[l + 1];
            for (size_t i = 0; i < nw; ++i) m->mlp[w].W[l][i] = (real)bf16_round((float)m->mlp[w].W[l][i]);
        }
}

void vo_model_destroy(vo_model *m) {
    if (!m) return;
    for (int w = 0; w < 6; ++w)
        for (int l = 0; l < VO_MAX_LAYERS; ++l) { free(m->mlp[w].W[l]); free(m->mlp[w].b[l]); }
    for (int k = 0; k < VO_MAX_TERM; ++k) free(m->term_center[k]);
    free(m->reward_param); free(m->action_cost); free(m);
}

/* ------------------------------------------------------------------------------------------
 * O3. MLP forward: x_{l+1} = act(W_l x_l + b_l), last layer linear.
 * ---------------------------------------------------------------------------------------- */
static int mlp_max_width(const vo_mlp *f) {
    int w = 0;
    for (int l = 0; l <= f->n_layers; ++l) if (f->dims[l] > w) w = f->dims[l];
    return w;
}

static void mlp_forward_one(const vo_mlp *f, int emulate_bf16, const real *x, real *y,
                            real *buf0, real *buf1) {
    const real *in = x;
    for (int l = 0; l < f->n_layers; ++l) {
        int K = f->dims[l], N = f->dims[l + 1];
        int last = (l == f->n_layers - 1);
        real *out = last ? y : ((l & 1) ? buf1 : buf0);
        for (int j = 0; j < N; ++j) {
            real acc = 0;
            for (int k = 0; k < K; ++k) {
                real xv = emulate_bf16 ? (real)bf16_round((float)in[k]) : in[k];
                acc += f->W[l][(size_t)j * K + k] * xv;
            }
            acc += f->b[l][j];
            if (!last) {
                if (f->act == VO_ACT_RELU) acc = acc > 0 ? acc : 0;
                else if (f->act == VO_ACT_SILU) {
#if defined(VO_REAL_IS_DOUBLE)
                    acc = acc / (1.0 + exp(-acc));
#else
                    acc = acc / (1.0f + expf(-acc));
#endif
                }
            }
            out[j] = acc;
        }
        in = out;
    }
}

/* rows of x ([rows][dims[0]]) -> rows of y ([rows][dims[n_layers]]), fp32 in/out. */
int vo_mlp_forward(const vo_model *m, int which, const float *x, int rows, float *y) {
    if (which < 0 || which > 5 || m->mlp[which].n_layers < 1) return -1;
    const vo_mlp *f = &m->mlp[which];
    int w = mlp_max_width(f), K0 = f->dims[0], NL = f->dims[f->n_layers];
    real *b0 = (real *)malloc(sizeof(real) * w * 4), *b1 = b0 + w, *xi = b1 + w, *yo = xi + w;
    for (int r = 0; r < rows; ++r) {
        for (int k = 0; k < K0; ++k) xi[k] = (real)x[(size_t)r * K0 + k];
        mlp_forward_one(f, m->emulate_bf16, xi, yo, b0, b1);
        for (int j = 0; j < NL; ++j) y[(size_t)r * NL + j] = (float)yo[j];
    }
    free(b0);
    return 0;
}

/* generator input x0 = [s ; onehot(a) ; omega]  (reading R12: this order) */
static void build_gen_input(const vo_model *m, const real *s, int a, const float *omega, real *x) {
    int S = m->S, A = m->A, Nz = m->Nz;
    for (int i = 0; i < S; ++i) x[i] = s[i];
    for (int i = 0; i < A; ++i) x[S + i] = (i == a) ? (real)1 : (real)0;
    for (int i = 0; i < Nz; ++i) x[S + A + i] = (real)omega[i];
}

/* R(s,a): bounded reward on the CURRENT state-action (readings R7, R14). */
static real reward(const vo_model *m, const real *s, int a) {
    int S = m->S;
    real r = 0;
    if (m->reward_kind == VO_R_NEG_L2_GOAL) {
        real d2 = 0;
        for (int i = 0; i < S; ++i) { real d = s[i] - m->reward_param[i]; d2 += d * d; }
#if defined(VO_REAL_IS_DOUBLE)
        r = -sqrt(d2);
#else
        r = -sqrtf(d2);
#endif
    } else if (m->reward_kind == VO_R_NEG_QUADRATIC) {
        real acc = 0;
        for (int i = 0; i < S; ++i) {
            real row = 0;
            for (int j = 0; j < S; ++j) row += m->reward_param[(size_t)i * S + j] * s[j];
            acc += s[i] * row;
        }
        r = -acc;
    } else {
        real acc = 0;
        for (int i = 0; i < S; ++i) acc += m->reward_param[i] * s[i];
        r = acc + m->reward_param[S];
    }
    if (m->action_cost) r += m->action_cost[a];
    return r;
}

/* One alive step's reward with the terminal regions (see vo_model_set_terminal): returns the reward
 * paid at this step and sets *stop when the episode ends here.  *margin (optional) is lowered to the
 * smallest | ||s - c_k|| - r_k | seen: how close the membership decisions were to flipping. */
static real step_reward_term(const vo_model *m, const real *s, int a, int *stop, float *margin) {
    real bonus = 0;
    *stop = 0;
    for (int k = 0; k < m->n_term; ++k) {
        float d2 = 0.0f;
        for (int j = 0; j < m->term_dim[k]; ++j) {
            float sj = (float)s[j];
            if (m->emulate_bf16) sj = bf16_round(sj); /* bf16 mode stores particle states in bf16 (R18) */
            const float d = sj - m->term_center[k][j];
            d2 = fmaf(d, d, d2);
        }
        const float r = m->term_radius[k];
        if (margin) {
            const float mg = fabsf(sqrtf(d2) - r);
            if (mg < *margin) *margin = mg;
        }
        if (d2 <= r * r) {
            bonus += (real)m->term_reward[k];
            if (m->term_stop[k]) *stop = 1;
        }
    }
    if (*stop) return bonus;
    return bonus + reward(m, s, a);
}

typedef struct { real *x, *b0, *b1, *s, *sn, *o; float *omega; } scratch;

static scratch scratch_alloc(const vo_model *m) {
    scratch z;
    int w = 1;
    for (int i = 0; i < 6; ++i) { int v = mlp_max_width(&m->mlp[i]); if (v > w) w = v; }
    if (m->S + m->A + m->Nz > w) w = m->S + m->A + m->Nz;
    z.x = (real *)malloc(sizeof(real) * w * 6);
    z.b0 = z.x + w; z.b1 = z.b0 + w; z.s = z.b1 + w; z.sn = z.s + w; z.o = z.sn + w;
    z.omega = (float *)malloc(sizeof(float) * (m->Nz + 4));
    return z;
}
static void scratch_free(scratch *z) { free(z->x); free(z->omega); }

/* one generator call: y = f(s, a, omega(seed; p,q,t,stream)) */
static void gen_step(const vo_model *m, int which, const real *s, int a, uint64_t seed, uint32_t p,
                     uint32_t q, uint32_t t, uint32_t stream, scratch *z, real *y) {
    vo_normals(seed, p, q, t, stream, m->Nz, z->omega);
    build_gen_input(m, s, a, z->omega, z->x);
    mlp_forward_one(&m->mlp[which], m->emulate_bf16, z->x, y, z->b0, z->b1);
}

/* ------------------------------------------------------------------------------------------
 * Single (p,q) trajectory, for pins and debugging: states_out [H+1][S], obs_out [H][O],
 * returns the discounted return G = sum_t gamma^t R(s_t, a_t).
 * ---------------------------------------------------------------------------------------- */
double vo_rollout_trajectory(const vo_model *m, const float *s0, const int32_t *actions, int H,
                             uint32_t p, uint32_t q, uint64_t seed, float *states_out,
                             float *obs_out) {
    scratch z = scratch_alloc(m);
    int S = m->S, O = m->O;
    for (int i = 0; i < S; ++i) z.s[i] = (real)s0[i];
    real G = 0, disc = 1;
    for (int i = 0; i < S; ++i) if (states_out) states_out[i] = (float)z.s[i];
    int alive = 1;
    for (int t = 0; t < H; ++t) {
        int a = actions[t];
        if (alive) {
            int stop = 0;
            G += disc * step_reward_term(m, z.s, a, &stop, NULL);
            if (stop) alive = 0;
        }
        if (!alive) { /* terminated: the state stays frozen, no observation, nothing accrues */
            if (states_out) for (int i = 0; i < S; ++i) states_out[(size_t)(t + 1) * S + i] = (float)z.s[i];
            if (obs_out) for (int i = 0; i < O; ++i) obs_out[(size_t)t * O + i] = 0.0f;
            continue;
        }
        gen_step(m, 0, z.s, a, seed, p, q, (uint32_t)t, VO_STREAM_ROLLOUT_T, &z, z.sn);
        gen_step(m, 1, z.sn, a, seed, p, q, (uint32_t)t, VO_STREAM_ROLLOUT_Z, &z, z.o);
        disc *= (real)m->gamma;
        for (int i = 0; i < S; ++i) z.s[i] = z.sn[i];
        if (states_out) for (int i = 0; i < S; ++i) states_out[(size_t)(t + 1) * S + i] = (float)z.s[i];
        if (obs_out) for (int i = 0; i < O; ++i) obs_out[(size_t)t * O + i] = (float)z.o[i];
    }
    scratch_free(&z);
    return (double)G;
}

/* ------------------------------------------------------------------------------------------
 * O4. Rollout values.  particles [P][S], action_seqs [Q][H] (this call's sequences; their
 * absolute indices for the noise keying are q_offset .. q_offset+Q-1), weights [P] or NULL.
 * values_out [Q]; witness_out [Q][O] or NULL (reading R10); returns_out [Q][P] or NULL
 * (per-(p,q) discounted returns, for pins).
 * ---------------------------------------------------------------------------------------- */
int vo_rollout_values_term(const vo_model *m, const float *particles, int P, const int32_t *action_seqs,
                           int Q, int H, const float *weights, uint64_t seed, int q_offset,
                           float *values_out, float *witness_out, float *returns_out,
                           float *final_states_out, int32_t *t_term_out, float *margin_out);

int vo_rollout_values(const vo_model *m, const float *particles, int P, const int32_t *action_seqs,
                      int Q, int H, const float *weights, uint64_t seed, int q_offset,
                      float *values_out, float *witness_out, float *returns_out) {
    return vo_rollout_values_term(m, particles, P, action_seqs, Q, H, weights, seed, q_offset, values_out,
                                  witness_out, returns_out, NULL, NULL, NULL);
}

/* The same with the per-trajectory detail the termination tests need: final_states_out [Q][P][S]
 * (s_H, or the frozen state of a terminated trajectory), t_term_out [Q][P] (step at which the
 * episode ended, H if it did not), margin_out [Q][P] (see step_reward_term).  Any may be NULL. */
int vo_rollout_values_term(const vo_model *m, const float *particles, int P, const int32_t *action_seqs,
                           int Q, int H, const float *weights, uint64_t seed, int q_offset,
                           float *values_out, float *witness_out, float *returns_out,
                           float *final_states_out, int32_t *t_term_out, float *margin_out) {
    int S = m->S, O = m->O;
    double wsum = 0;
    for (int p = 0; p < P; ++p) wsum += weights ? (double)weights[p] : 1.0;
    if (!(wsum > 0)) return -2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int q = 0; q < Q; ++q) {
        scratch z = scratch_alloc(m);
        double V = 0;
        double *Wit = (double *)calloc((size_t)O, sizeof(double));
        real *wit = (real *)malloc(sizeof(real) * O);
        for (int p = 0; p < P; ++p) {
            double wbar = (weights ? (double)weights[p] : 1.0) / wsum;
            for (int i = 0; i < S; ++i) z.s[i] = (real)particles[(size_t)p * S + i];
            for (int i = 0; i < O; ++i) wit[i] = 0;
            real G = 0, disc = 1;
            int t_term = H;
            float margin = INFINITY;
            for (int t = 0; t < H; ++t) {
                int a = action_seqs[(size_t)q * H + t];
                int stop = 0;
                /* reward on CURRENT state, gamma^t, t from 0; terminal regions: vo_model_set_terminal */
                G += disc * step_reward_term(m, z.s, a, &stop, &margin);
                if (stop) { t_term = t; break; } /* state frozen, nothing accrues afterwards */
                gen_step(m, 0, z.s, a, seed, (uint32_t)p, (uint32_t)(q + q_offset), (uint32_t)t,
                         VO_STREAM_ROLLOUT_T, &z, z.sn);
                gen_step(m, 1, z.sn, a, seed, (uint32_t)p, (uint32_t)(q + q_offset), (uint32_t)t,
                         VO_STREAM_ROLLOUT_Z, &z, z.o);
                for (int i = 0; i < O; ++i) wit[i] += disc * z.o[i];
                disc *= (real)m->gamma;
                for (int i = 0; i < S; ++i) z.s[i] = z.sn[i];
            }
            V += wbar * (double)G;
            for (int i = 0; i < O; ++i) Wit[i] += wbar * (double)wit[i];
            if (returns_out) returns_out[(size_t)q * P + p] = (float)G;
            if (final_states_out)
                for (int i = 0; i < S; ++i) final_states_out[((size_t)q * P + p) * S + i] = (float)z.s[i];
            if (t_term_out) t_term_out[(size_t)q * P + p] = t_term;
            if (margin_out) margin_out[(size_t)q * P + p] = margin;
        }
        values_out[q] = (float)V;
        if (witness_out) for (int i = 0; i < O; ++i) witness_out[(size_t)q * O + i] = (float)Wit[i];
        free(Wit); free(wit);
        scratch_free(&z);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O7. Systematic resampling, exact integer definition (reading R6).
 *   q_i = floor(v_i * 2^32) (v_i in [0,1], exact), C_i = sum_{j<=i} q_j, W = C_{N-1},
 *   U = (x0 * W) >> 32,  i_k = min{ i : N*C_i > k*W + U }  (128-bit integers).
 * Returns 0, or -2 when every weight quantises to zero (ancestors := identity).
 * ---------------------------------------------------------------------------------------- */
int vo_resample_systematic_x0(const float *v, int N, uint32_t x0, int32_t *ancestors) {
    uint64_t *C = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)N);
    uint64_t run = 0;
    for (int i = 0; i < N; ++i) {
        double s = (double)v[i] * 4294967296.0;
        uint64_t qi = 0;
        if (s > 0) qi = (s >= 4294967296.0) ? 4294967296ull : (uint64_t)s; /* v>1 or NaN clamp */
        run += qi;
        C[i] = run;
    }
    uint64_t W = run;
    if (W == 0) {
        for (int k = 0; k < N; ++k) ancestors[k] = k;
        free(C);
        return -2;
    }
    uint64_t U = (uint64_t)(((unsigned __int128)x0 * W) >> 32);
    int i = 0;
    for (int k = 0; k < N; ++k) {
        unsigned __int128 rhs = (unsigned __int128)(uint64_t)k * W + U;
        while (!((unsigned __int128)(uint64_t)N * C[i] > rhs)) ++i; /* exists: rhs < N*W */
        ancestors[k] = i;
    }
    free(C);
    return 0;
}

int vo_resample_systematic(const float *v, int N, uint64_t seed, int32_t *ancestors) {
    return vo_resample_systematic_x0(v, N, vo_resample_word(seed), ancestors);
}

/* ------------------------------------------------------------------------------------------
 * O5. Belief update.
 *   proposals_out [N][S] (s'_i), logits_out [N] (L_i), post_weights_out [N] (v_i),
 *   log_evidence_out [1], ancestors_out [N], particles_out [N][S], weights_out [N] (=1/N).
 *   Any output pointer may be NULL.  Returns 0, or -2 if all weights are zero / m is not finite
 *   (then particles_out := proposals, ancestors := identity).
 * ---------------------------------------------------------------------------------------- */
/* Effective sample size of unnormalised weights (Kong, Liu & Wong 1994; the criterion of adaptive
 * resampling in SIR filters): ESS = (sum v)^2 / sum v^2, in [1, N]; 0 if all v = 0. */
double vo_effective_sample_size(const float *v, int N) {
    double s1 = 0, s2 = 0;
    for (int i = 0; i < N; ++i) {
        s1 += (double)v[i];
        s2 += (double)v[i] * (double)v[i];
    }
    return s2 > 0 ? s1 * s1 / s2 : 0.0;
}

/* Belief update with ADAPTIVE resampling: the filter resamples only when
 * ESS(v) < ess_threshold * N (ess_threshold = +inf: always, the plain update below).  Otherwise the
 * proposals are kept (ancestors = identity) and the normalised weights v_i / sum v are carried
 * forward in weights_out.  ess_out / resampled_out may be NULL. */
int vo_belief_update_ess(const vo_model *m, const float *particles, int N, int action,
                         const float *observation, const float *weights, uint64_t seed,
                         float ess_threshold, float *proposals_out, float *logits_out,
                         float *post_weights_out, double *log_evidence_out, int32_t *ancestors_out,
                         float *particles_out, float *weights_out, double *ess_out,
                         int32_t *resampled_out) {
    int S = m->S, O = m->O, A = m->A;
    const vo_mlp *tf = &m->mlp[2], *tg = &m->mlp[3];
    int d = tf->dims[tf->n_layers];
    float *prop = (float *)malloc(sizeof(float) * (size_t)N * S);
    float *L = (float *)malloc(sizeof(float) * (size_t)N);
    float *v = (float *)malloc(sizeof(float) * (size_t)N);
    int32_t *anc = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    /* e = f(o), once */
    real *e = (real *)malloc(sizeof(real) * d);
    {
        scratch z = scratch_alloc(m);
        for (int i = 0; i < O; ++i) z.x[i] = (real)observation[i];
        mlp_forward_one(tf, m->emulate_bf16, z.x, e, z.b0, z.b1);
        scratch_free(&z);
    }
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        scratch z = scratch_alloc(m);
        real *gout = (real *)malloc(sizeof(real) * d);
        for (int k = 0; k < S; ++k) z.s[k] = (real)particles[(size_t)i * S + k];
        gen_step(m, 0, z.s, action, seed, (uint32_t)i, 0, 0, VO_STREAM_BELIEF_T, &z, z.sn);
        for (int k = 0; k < S; ++k) prop[(size_t)i * S + k] = (float)z.sn[k];
        /* g(s' [; onehot(a)]) */
        for (int k = 0; k < S; ++k) z.x[k] = z.sn[k];
        if (m->lik_action_cond)
            for (int k = 0; k < A; ++k) z.x[S + k] = (k == action) ? (real)1 : (real)0;
        mlp_forward_one(tg, m->emulate_bf16, z.x, gout, z.b0, z.b1);
        real ell = 0;
        for (int k = 0; k < d; ++k) ell += e[k] * gout[k]; /* raw dot product (reading R1) */
        float lw = 0.0f;
        if (weights) lw = weights[i] > 0 ? logf(weights[i]) : -INFINITY;
        L[i] = lw + (float)ell / m->lambda;
        free(gout);
        scratch_free(&z);
    }
    free(e);
    float mx = -INFINITY;
    int has_nan = 0;
    for (int i = 0; i < N; ++i) {
        if (L[i] > mx) mx = L[i];
        if (L[i] != L[i]) has_nan = 1;
    }
    int status = 0;
    /* reading R20: all weights zero, or ANY non-finite score (a NaN never wins a comparison) */
    if (!(mx > -INFINITY) || !(mx < INFINITY) || has_nan) status = -2;
    double sv = 0, sw = 0;
    for (int i = 0; i < N; ++i) {
        v[i] = status ? 0.0f : expf(L[i] - mx);
        sv += (double)v[i];
        sw += weights ? (double)weights[i] : 1.0;
    }
    const double ess = status ? 0.0 : vo_effective_sample_size(v, N);
    const int resample = status == 0 && (isinf(ess_threshold) || ess < (double)ess_threshold * (double)N);
    if (resample) status = vo_resample_systematic(v, N, seed, anc);
    if (status || !resample) for (int k = 0; k < N; ++k) anc[k] = k;
    if (ess_out) *ess_out = ess;
    if (resampled_out) *resampled_out = (resample && status == 0) ? 1 : 0;
    if (log_evidence_out) *log_evidence_out = status ? -INFINITY : (double)mx + log(sv) - log(sw);
    for (int k = 0; k < N; ++k) {
        if (particles_out)
            for (int j = 0; j < S; ++j) particles_out[(size_t)k * S + j] = prop[(size_t)anc[k] * S + j];
        if (weights_out) weights_out[k] = (resample || status) ? 1.0f / (float)N : (float)((double)v[k] / sv);
        if (ancestors_out) ancestors_out[k] = anc[k];
    }
    if (proposals_out) memcpy(proposals_out, prop, sizeof(float) * (size_t)N * S);
    if (logits_out) memcpy(logits_out, L, sizeof(float) * (size_t)N);
    if (post_weights_out) memcpy(post_weights_out, v, sizeof(float) * (size_t)N);
    free(prop); free(L); free(v); free(anc);
    return status;
}

/* The plain SIR update: always resample. */
int vo_belief_update(const vo_model *m, const float *particles, int N, int action,
                     const float *observation, const float *weights, uint64_t seed,
                     float *proposals_out, float *logits_out, float *post_weights_out,
                     double *log_evidence_out, int32_t *ancestors_out, float *particles_out,
                     float *weights_out) {
    return vo_belief_update_ess(m, particles, N, action, observation, weights, seed, INFINITY, proposals_out,
                                logits_out, post_weights_out, log_evidence_out, ancestors_out, particles_out,
                                weights_out, NULL, NULL);
}

/* ------------------------------------------------------------------------------------------
 * f1. Vectorised progressive widening with batched likelihood (section 4.3;
 * SURVEY 8f f1).  "Parallel simulations are grouped by their parent action nodes, after which the
 * PW operations are performed for all action-node groups in parallel".
 *
 * Inputs: N simulations (particles [N][S]) grouped by parent action node: group g owns the
 * simulations [group_off[g], group_off[g+1]) and has action group_action[g], visit count
 * visit_count[g] = N(a), branch count branch_count[g] = |C(a)| and stored branch observations
 * branch_obs[g][0 .. |C(a)|) (rows of O floats, M_max rows reserved per group).
 * For every simulation i of group g, in index order (readings R26-R29 of DESIGN.md):
 *   s'_i = f_T(s_i, a_g, w_T(i))                       (stream 3, counter (i,0,0), as the belief update)
 *   o_i  = f_Z(s'_i, a_g, w_Z(i))                      (stream 5)
 *   N(a) += 1;  if |C(a)| < min(M_max, T(N(a))) the simulation opens branch |C(a)| with the
 *   observation o_i and is attached to it; otherwise it is attached to an existing branch picked
 *   uniformly, b = (x_i * |C(a)|) >> 32 with x_i one Philox word (stream 6)
 *   T(n) = ceil(k_o * n^alpha_o * (1 - 1e-9)) in fp64: the criterion |C(a)| < k_o N(a)^alpha_o with a
 *   relative tolerance, so that exact powers do not depend on the last bit of pow().
 * Then "the likelihood model is used to weight successor states according to the observation
 * stored at the selected branch, followed by resampling": with e_{g,m} = f(obs_{g,m})
 * (all branch observations go through the tower as one batch),
 *   L_i = log w_i + <e_{g,b(i)}, g(s'_i)> / lambda,
 * and every (action node, branch) pair that received simulations is one child belief: its members
 * (in index order) are resampled among themselves with the exact-integer systematic resampler (O7),
 * v = exp(L - max over the members), offset word = Philox word of (seed, stream 4, counter (g*M_max+m,0,0)).
 * The r-th member receives the r-th draw: particles_out[i_r] = s'_{ancestor}, ancestors_out[i_r] = the
 * ancestor's simulation index.  A child whose weights are all zero / not finite keeps its members
 * (identity) and sets seg_status_out[g*M_max+m] = 1.
 * Outputs (any may be NULL): proposals_out [N][S], obs_out [N][O], sim_branch_out [N], opened_out [N]
 * (1 if the simulation opened its branch), logits_out [N], post_weights_out [N] (v_i),
 * ancestors_out [N], particles_out [N][S], weights_out [N] (1 / members), seg_status_out [G*M_max].
 * visit_count, branch_count and branch_obs are updated in place.  Returns 0 or -1 (bad arguments).
 * ---------------------------------------------------------------------------------------- */
static int pw_threshold(double k_o, double alpha_o, int n) {
    const double x = k_o * pow((double)n, alpha_o) * (1.0 - 1e-9);
    if (!(x < 2147483647.0)) return 2147483647;
    const int t = (int)ceil(x);
    return t < 0 ? 0 : t;
}

int vo_pw_update(const vo_model *m, const float *particles, int N, const int32_t *group_off, int G,
                 const int32_t *group_action, int32_t *visit_count, int32_t *branch_count,
                 float *branch_obs, int M_max, double k_o, double alpha_o, const float *weights,
                 uint64_t seed, float *proposals_out, float *obs_out, int32_t *sim_branch_out,
                 int32_t *opened_out, float *logits_out, float *post_weights_out, int32_t *ancestors_out,
                 float *particles_out, float *weights_out, int32_t *seg_status_out) {
    int S = m->S, O = m->O, A = m->A;
    const vo_mlp *tf = &m->mlp[2], *tg = &m->mlp[3];
    int d = tf->dims[tf->n_layers];
    if (N < 1 || G < 1 || M_max < 1 || !(k_o > 0) || !(alpha_o > 0)) return -1;
    if (group_off[0] != 0 || group_off[G] != N) return -1;
    for (int g = 0; g < G; ++g)
        if (group_off[g + 1] < group_off[g] || group_action[g] < 0 || group_action[g] >= A ||
            branch_count[g] < 0 || branch_count[g] > M_max || visit_count[g] < 0) return -1;
    float *prop = (float *)malloc(sizeof(float) * (size_t)N * S);
    float *obs = (float *)malloc(sizeof(float) * (size_t)N * O);
    float *L = (float *)malloc(sizeof(float) * (size_t)N);
    float *v = (float *)calloc((size_t)N, sizeof(float));
    int32_t *br = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    int32_t *anc = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    int32_t *gid = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    for (int g = 0; g < G; ++g)
        for (int i = group_off[g]; i < group_off[g + 1]; ++i) gid[i] = g;
    /* 1. successor states and sampled observations of every simulation */
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        scratch z = scratch_alloc(m);
        const int a = group_action[gid[i]];
        for (int k = 0; k < S; ++k) z.s[k] = (real)particles[(size_t)i * S + k];
        gen_step(m, 0, z.s, a, seed, (uint32_t)i, 0, 0, VO_STREAM_BELIEF_T, &z, z.sn);
        for (int k = 0; k < S; ++k) prop[(size_t)i * S + k] = (float)z.sn[k];
        gen_step(m, 1, z.sn, a, seed, (uint32_t)i, 0, 0, VO_STREAM_PW_OBS, &z, z.o);
        for (int k = 0; k < O; ++k) obs[(size_t)i * O + k] = (float)z.o[k];
        scratch_free(&z);
    }
    /* 2. progressive widening, simulation by simulation within each action node */
    for (int g = 0; g < G; ++g) {
        int C = branch_count[g], n = visit_count[g];
        for (int i = group_off[g]; i < group_off[g + 1]; ++i) {
            ++n;
            int T = pw_threshold(k_o, alpha_o, n);
            if (T > M_max) T = M_max;
            int opened = 0;
            if (C < T) {
                memcpy(branch_obs + ((size_t)g * M_max + C) * O, obs + (size_t)i * O, sizeof(float) * (size_t)O);
                br[i] = C;
                ++C;
                opened = 1;
            } else {
                const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
                const uint32_t ctr[4] = {(uint32_t)i, 0, 0, VO_STREAM_PW_ATTACH << 16};
                uint32_t x[4];
                vo_philox4x32_10(ctr, key, x);
                br[i] = (int32_t)(((uint64_t)x[0] * (uint64_t)C) >> 32); /* C >= 1 here: T(n) >= 1 */
            }
            if (opened_out) opened_out[i] = opened;
        }
        branch_count[g] = C;
        visit_count[g] = n;
    }
    /* 3. batched likelihood: every stored branch observation through the tower f, then the scores */
    real *E = (real *)calloc((size_t)G * M_max * d, sizeof(real));
#pragma omp parallel for schedule(static)
    for (int gm = 0; gm < G * M_max; ++gm) {
        if (gm % M_max >= branch_count[gm / M_max]) continue;
        scratch z = scratch_alloc(m);
        for (int k = 0; k < O; ++k) z.x[k] = (real)branch_obs[(size_t)gm * O + k];
        mlp_forward_one(tf, m->emulate_bf16, z.x, E + (size_t)gm * d, z.b0, z.b1);
        scratch_free(&z);
    }
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        scratch z = scratch_alloc(m);
        real *gout = (real *)malloc(sizeof(real) * d);
        const int g = gid[i], a = group_action[g];
        for (int k = 0; k < S; ++k) z.x[k] = (real)prop[(size_t)i * S + k];
        if (m->lik_action_cond)
            for (int k = 0; k < A; ++k) z.x[S + k] = (k == a) ? (real)1 : (real)0;
        mlp_forward_one(tg, m->emulate_bf16, z.x, gout, z.b0, z.b1);
        const real *e = E + ((size_t)g * M_max + br[i]) * d;
        real ell = 0;
        for (int k = 0; k < d; ++k) ell += e[k] * gout[k];
        float lw = 0.0f;
        if (weights) lw = weights[i] > 0 ? logf(weights[i]) : -INFINITY;
        L[i] = lw + (float)ell / m->lambda;
        free(gout);
        scratch_free(&z);
    }
    free(E);
    /* 4. every (action node, branch) child belief: normalise, resample among its members */
    for (int i = 0; i < N; ++i) anc[i] = i;
    if (seg_status_out) for (int gm = 0; gm < G * M_max; ++gm) seg_status_out[gm] = 0;
    int32_t *mem = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    float *vm = (float *)malloc(sizeof(float) * (size_t)N);
    int32_t *am = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    for (int g = 0; g < G; ++g)
        for (int b = 0; b < branch_count[g]; ++b) {
            int n = 0;
            for (int i = group_off[g]; i < group_off[g + 1]; ++i) if (br[i] == b) mem[n++] = i;
            if (n == 0) continue;
            float mx = -INFINITY;
            int bad = 0;
            for (int r = 0; r < n; ++r) {
                if (L[mem[r]] > mx) mx = L[mem[r]];
                if (L[mem[r]] != L[mem[r]]) bad = 1;
            }
            if (!(mx > -INFINITY) || !(mx < INFINITY)) bad = 1;
            int st = bad ? -2 : 0;
            if (!bad) {
                for (int r = 0; r < n; ++r) vm[r] = expf(L[mem[r]] - mx);
                const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
                const uint32_t ctr[4] = {(uint32_t)(g * M_max + b), 0, 0, VO_STREAM_RESAMPLE << 16};
                uint32_t x[4];
                vo_philox4x32_10(ctr, key, x);
                st = vo_resample_systematic_x0(vm, n, x[0], am);
                for (int r = 0; r < n; ++r) v[mem[r]] = vm[r];
            }
            if (weights_out) for (int r = 0; r < n; ++r) weights_out[mem[r]] = 1.0f / (float)n;
            if (st) {
                if (seg_status_out) seg_status_out[g * M_max + b] = 1;
                continue; /* members keep themselves */
            }
            for (int r = 0; r < n; ++r) anc[mem[r]] = mem[am[r]];
        }
    free(mem); free(vm); free(am);
    for (int i = 0; i < N; ++i) {
        if (particles_out)
            for (int j = 0; j < S; ++j) particles_out[(size_t)i * S + j] = prop[(size_t)anc[i] * S + j];
        if (ancestors_out) ancestors_out[i] = anc[i];
        if (sim_branch_out) sim_branch_out[i] = br[i];
    }
    if (proposals_out) memcpy(proposals_out, prop, sizeof(float) * (size_t)N * S);
    if (obs_out) memcpy(obs_out, obs, sizeof(float) * (size_t)N * O);
    if (logits_out) memcpy(logits_out, L, sizeof(float) * (size_t)N);
    if (post_weights_out) memcpy(post_weights_out, v, sizeof(float) * (size_t)N);
    free(prop); free(obs); free(L); free(v); free(br); free(anc); free(gid);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * f4. The diffusion teacher's sampler: the conditional denoiser
 * v(c, a, x_tau, tau) is trained with the v-prediction objective on x_tau = sqrt(abar) x_0 +
 * sqrt(1 - abar) eps with a cosine schedule, and samples are drawn with an
 * "ODE-based diffusion sampler [27]" (DDIM) from the latent noise omega.
 * Readings R30-R32: abar_tau = cos^2(pi tau / 2), i.e. alpha = cos(pi tau / 2), sigma = sin(pi tau / 2);
 * denoiser input [c ; onehot(a) ; x_tau ; temb(tau)] with temb = (sin(pi 2^k tau), cos(pi 2^k tau))_{k<4};
 * uniform grid tau_k = 1 - k / K, x at tau_0 = 1 is omega ~ N(0, I_D) (Philox stream 7, counter (i,0,0));
 * for k = 0 .. K-1 (one denoiser call each):
 *     v = v_theta(c, a, x, tau_k);  x0_hat = alpha x - sigma v;  eps_hat = sigma x + alpha v   (v-prediction)
 *     x <- alpha' x0_hat + sigma' eps_hat                                   (DDIM, eta = 0; ' = at tau_{k+1})
 * and x at tau_K = 0 is the sample.  which = 0: transition teacher (c = s, D = S), 1: observation
 * teacher (c = s', D = O).  cond [N][S], actions [N], out [N][D]; traj_out [K+1][D] or NULL: the path
 * of sample `traj_row`.  Returns 0, -1 bad arguments / no such denoiser.
 * ---------------------------------------------------------------------------------------- */
int vo_diffusion_sample(const vo_model *m, int which, const float *cond, const int32_t *actions, int N, int K,
                        uint64_t seed, float *out, int traj_row, float *traj_out) {
    if (which < 0 || which > 1 || N < 1 || K < 1) return -1;
    const vo_mlp *f = &m->mlp[4 + which];
    const int S = m->S, A = m->A, D = which == 0 ? m->S : m->O;
    if (f->n_layers < 1 || f->dims[0] != S + A + D + VO_TEMB || f->dims[f->n_layers] != D) return -1;
    const double half_pi = 1.5707963267948966;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        scratch z = scratch_alloc(m);
        float *omega = (float *)malloc(sizeof(float) * (size_t)(D + 4));
        real *x = (real *)malloc(sizeof(real) * (size_t)D), *v = (real *)malloc(sizeof(real) * (size_t)D);
        vo_normals(seed, (uint32_t)i, 0, 0, VO_STREAM_DIFFUSION, D, omega);
        for (int j = 0; j < D; ++j) x[j] = (real)omega[j];
        if (traj_out && i == traj_row) for (int j = 0; j < D; ++j) traj_out[j] = (float)x[j];
        for (int k = 0; k < K; ++k) {
            const double tau = 1.0 - (double)k / (double)K, tau_n = 1.0 - (double)(k + 1) / (double)K;
            for (int j = 0; j < S; ++j) z.x[j] = (real)cond[(size_t)i * S + j];
            for (int j = 0; j < A; ++j) z.x[S + j] = (j == actions[i]) ? (real)1 : (real)0;
            for (int j = 0; j < D; ++j) z.x[S + A + j] = x[j];
            for (int e = 0; e < VO_TEMB / 2; ++e) {
                const double arg = 3.141592653589793 * (double)(1 << e) * tau;
                z.x[S + A + D + 2 * e] = (real)sin(arg);
                z.x[S + A + D + 2 * e + 1] = (real)cos(arg);
            }
            mlp_forward_one(f, m->emulate_bf16, z.x, v, z.b0, z.b1);
            const real al = (real)cos(half_pi * tau), si = (real)sin(half_pi * tau);
            const real al_n = (real)cos(half_pi * tau_n), si_n = (real)sin(half_pi * tau_n);
            for (int j = 0; j < D; ++j) {
                const real x0_hat = al * x[j] - si * v[j];
                const real eps_hat = si * x[j] + al * v[j];
                x[j] = al_n * x0_hat + si_n * eps_hat;
            }
            if (traj_out && i == traj_row) for (int j = 0; j < D; ++j) traj_out[(size_t)(k + 1) * D + j] = (float)x[j];
        }
        for (int j = 0; j < D; ++j) out[(size_t)i * D + j] = (float)x[j];
        free(omega); free(x); free(v);
        scratch_free(&z);
    }
    return 0;
}

/* Normalised weights as the resampler sees them (O6): wbar_i = q_i / W in double. */
int vo_normalised_weights(const float *v, int N, double *wbar) {
    double W = 0;
    for (int i = 0; i < N; ++i) {
        double s = floor((double)v[i] * 4294967296.0);
        if (!(s > 0)) s = 0;
        if (s > 4294967296.0) s = 4294967296.0;
        wbar[i] = s; W += s;
    }
    if (!(W > 0)) return -2;
    for (int i = 0; i < N; ++i) wbar[i] /= W;
    return 0;
}

int vo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void vo_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int vo_real_bytes(void) { return (int)sizeof(real); }
