/*
 * econojax.h -- C ABI of the B200-native batched EconoJax environment step.
 *
 * What it computes: the environment transition of EconoJax (arXiv 2410.22165; "P:n" =
 * PAPER.md line n, "G#" = the readings listed in DESIGN.md section 3) for E independent
 * economies of N population agents + 1 government: gather, craft,
 * order placement with escrow, per-resource matching with price-time priority
 * at the price of the order placed last, order expiry (P:162,
 * P:275), bracketed tax collection and uniform redistribution at period ends (P:173,
 * P:190-195), isoelastic utility rewards (Eq.1-2), government welfare reward
 * (Eq.3-5), population observations and government statistics mean / std /
 * median (Fig.1).
 *
 * Conventions
 *  - Every function returns 0 (EJ_OK) or a negative EJ_ERR_* code; ej_last_error() gives a
 *    static/handle-owned string naming the offending field.  No exceptions, no errno.
 *  - "device pointer" = memory of the CUDA device that was current at ej_create; it is owned
 *    by the caller, must be 16-byte aligned (observation buffers and rings: checked, EJ_ERR_PARAM;
 *    int32 / float arrays: 4-byte aligned at least), is not retained after the call returns, but must
 *    stay alive until the handle's stream has executed the call (calls are asynchronous on
 *    the stream set by ej_set_stream, default stream 0).  "host pointer" = ordinary memory.
 *  - There is no CPU fallback: every step of the path runs in the sm_100a kernels of
 *    csrc/econojax.cu.  Without a CUDA device ej_create returns EJ_ERR_CUDA.
 *  - An out-of-range or currently invalid action is NOT an API error: it is a no-op for that
 *    agent (no labor) and bumps the env's `invalid` counter (G2).  Stepping a finished env
 *    (t == episode_length) changes nothing, returns rewards 0 and done = 1 (G28).
 */
#ifndef ECONOJAX_H
#define ECONOJAX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EJ_OK 0
#define EJ_ERR_PARAM (-1)  /* bad argument or parameter field; ej_last_error names it */
#define EJ_ERR_NOMEM (-2)  /* device or host allocation failed */
#define EJ_ERR_CUDA (-3)   /* CUDA runtime error (text in ej_last_error) */
#define EJ_ERR_STATE (-4)  /* call not valid in the handle's state (e.g. step before reset) */

#define EJ_MAX_PRICES 16
#define EJ_MAX_BRACKETS 16
#define EJ_MAX_RATE_LEVELS 32
#define EJ_MAX_RESOURCES 16
#define EJ_MAX_AGENTS 1024
#define EJ_MAX_ACTIVE_ORDERS 32

#define EJ_CRAFT_SINGLE 0        /* the paper's single craft action (30/86 actions P:350) */
#define EJ_CRAFT_PER_RESOURCE 1  /* "convert r" variant of BASELINE.json (G3) */
#define EJ_SKILL_UNIFORM01 0
#define EJ_SKILL_PARETO_CLIP 1   /* Pareto(alpha=4) clipped to [lo, hi] (G29) */
#define EJ_SKILL_NORMAL_CLIP 2   /* f3, section 5 ("a normal distribution around 1.0 with a standard deviation of
                                    1.0"): skill_mean + skill_std * z clipped to [lo, hi], z = sum of twelve 24-bit
                                    Philox uniforms - 6 (G42) */

/* Environment parameters (Table 2, unless noted).  POD, versioned by struct_size. */
typedef struct ej_params {
    uint32_t struct_size;                   /* = sizeof(ej_params) */
    int32_t num_prices;                     /* P, 1..16 */
    int32_t prices[EJ_MAX_PRICES];          /* strictly ascending positive integers (G4) */
    int32_t episode_length;                 /* T, 1..65535 */
    int32_t tax_period;                     /* >= 1 */
    int32_t num_brackets;                   /* B = thresholds + 1, 1..16 */
    float thresholds[EJ_MAX_BRACKETS];      /* B-1 used, strictly ascending, > 0 (G32) */
    int32_t num_rate_levels;                /* L, 1..32 (21) */
    float rate_table[EJ_MAX_RATE_LEVELS];   /* tax rate of government level k (G5) */
    int32_t allow_noop;
    float starting_coin;
    int32_t order_expiry;                   /* steps an order stays live, >= 1 (G14) */
    int32_t max_active_orders;              /* M per agent, 1..32, N*M < 65535 */
    int32_t book_cap;                       /* K per (resource, side); 0 = unbounded (G15) */
    int32_t craft_units;                    /* R_kappa */
    int32_t craft_distinct;                 /* R_d <= R */
    int32_t craft_mode;                     /* EJ_CRAFT_* (G3) */
    float labor_craft, labor_gather, labor_trade;
    float eta;                              /* != 1 */
    float omega;
    float craft_scale;                      /* "scaled by a constant" P:158 (G6) */
    int32_t taxes_enabled;
    int32_t skill_init;                     /* EJ_SKILL_* */
    float skill_clip_lo, skill_clip_hi;
    float obs_scale_coin, obs_scale_count, obs_scale_price, obs_scale_labor; /* G25 */
    uint32_t env_id_base;                   /* global id of local env 0: every random draw is keyed by
                                               the global env id, so results do not depend on E or on
                                               how envs are sharded over GPUs (multi-GPU: DESIGN.md 7) */
    float skill_growth_rate;                /* f3: 0 = skills fixed.  > 0: after a valid gather r (craft) the
                                               skill SG[r] (SC) becomes min(skill_max, s + s * (rate * (1 - s / skill_max))),
                                               one binary32 rounding per operation (G41); the action itself uses the old skill */
    float skill_max;                        /* > 0 when skill_growth_rate > 0 (5) */
    float skill_mean, skill_std;            /* EJ_SKILL_NORMAL_CLIP only (1.0, 1.0); skill_std >= 0 */
} ej_params;

typedef struct ej_env ej_env;

/* Sizes and offsets derived from (E, N, R, params).  All counts in elements unless "bytes". */
typedef struct ej_layout_info {
    int32_t E, N, R, P, B, L;
    int32_t A;                  /* number of discrete actions R + (1|R) + 2RP + noop */
    int32_t base_craft, base_buy, base_sell, noop_action; /* first index of each action group; noop = -1 if off */
    int32_t D_pop;              /* 6 + 8R + B floats per agent */
    int32_t D_gov;              /* 3(3+R) + B + 2 floats per env */
    int32_t D_gov_pad;          /* D_gov rounded up to a multiple of 4 */
    size_t gov_obs_offset;      /* floats: start of the government region in an obs buffer (multiple of 4) */
    size_t obs_floats;          /* total floats of one obs buffer: gov_obs_offset + E*D_gov_pad */
    size_t rew_floats;          /* E*(N+1) */
    size_t state_words;         /* int32 words per env of the canonical dump (ej_get_state) */
    size_t device_state_bytes;  /* library-owned device bytes per env */
    size_t smem_bytes;          /* dynamic shared memory per CTA of the step kernel */
    int32_t threads_per_env;    /* CTA size */
    int32_t D_priv;             /* f2: 3R + 4 agent-private columns of a population row */
    int32_t D_shared;           /* f2: 5R + B + 2 env-wide columns (market statistics, rates, timers: P:424) */
    int32_t D_shared_pad;       /* D_shared rounded up to a multiple of 4 (row stride of obs_shared_ring) */
} ej_layout_info;

/* Optional inputs/outputs of ej_rollout; all device pointers, any may be NULL. */
typedef struct ej_rollout_io {
    uint32_t struct_size;             /* = sizeof(ej_rollout_io) */
    int32_t ring_depth;               /* >= 1: step s of the call writes ring slot s % ring_depth */
    const int32_t* actions_in;        /* [T][E][N]; NULL = draw with the Philox/CDF generator (G30) */
    const int32_t* gov_actions_in;    /* [T][E][B] level indices; NULL = draw */
    float* obs_ring;                  /* [ring_depth][obs_floats] */
    float* rew_ring;                  /* [ring_depth][E][N+1] */
    uint8_t* done_ring;               /* [ring_depth][E] */
    int32_t* actions_ring;            /* [ring_depth][E][N] actions actually applied */
    int32_t* gov_actions_ring;        /* [ring_depth][E][B] */
    float* pop_logits_ring;           /* policy mode only: [ring_depth][E*N][A] logits the actions were sampled from */
    float* gov_logits_ring;           /* policy mode only: [ring_depth][E][B*L] */
    /* f2, factored observations: the last 5R + B + 2 entries of a population row (market statistics,
     * tax rates, timers: P:424) are the same for every agent of an env, so the observation of a step
     * can leave as an agent-private block and one env-wide block.  Column k < 3R + 4 of obs row
     * (e, i) = priv[e][i][k]; column 3R + 4 + k = shared[e][k].  Set priv and shared together and
     * leave obs_ring NULL; needs N * (3R + 4) to be a multiple of 4 and a shape whose full tile is
     * staged in shared memory (N <= 256 and state + scratch + N * D_pop * 4 bytes <= 100 KB per CTA), not available in policy mode:
     * EJ_ERR_PARAM otherwise. */
    float* obs_priv_ring;             /* [ring_depth][E][N][3R + 4] */
    float* obs_shared_ring;           /* [ring_depth][E][ceil4(5R + B + 2)] */
    float* obs_gov_ring;              /* [ring_depth][E][D_gov_pad] government rows (optional) */
    /* f4 (the rollout a PPO loop runs; G44).  auto_reset != 0: an env whose episode ends at a step
     * (done = 1 in done_ring) starts its next episode within the same step -- the state of ej_reset, every random draw
     * of the new episode keyed by (seed, global env, agent, t, stream | episode << 8), event counters kept -- and the
     * observation written for that step is the one of the fresh state (the one the policy acts on next; the terminal
     * observation is not written).  Rewards and done are the step's own, so with ring_depth = T the rings rew_ring
     * [T][E][N+1] and done_ring [T][E] are what a backward GAE scan reads.  An env already finished when the call begins
     * starts its next episode with the call's first step.  auto_reset == 0 (default): envs stay done (G28).  Not available
     * together with the factored observation rings (EJ_ERR_PARAM). */
    int32_t auto_reset;
    int32_t reserved0;
} ej_rollout_io;

/* One tanh MLP  in_dim -> 128 -> 128 -> out_dim  (Table 2; BASELINE.json
 * configs[4]).  HOST pointers, read during ej_set_policy only: bf16 bit patterns in the
 * row-major [out_features][in_features] layout of a linear layer, fp32 biases. */
typedef struct ej_mlp {
    uint32_t struct_size;             /* = sizeof(ej_mlp) */
    int32_t in_dim;                   /* D_pop (population) or D_gov (government) */
    int32_t hidden;                   /* must be 128 */
    int32_t out_dim;                  /* A (population) or B*L (government: B heads of L levels), <= 256 */
    const uint16_t* w1;               /* [128][in_dim] */
    const uint16_t* w2;               /* [128][128] */
    const uint16_t* w3;               /* [out_dim][128] */
    const float* b1;                  /* [128] */
    const float* b2;                  /* [128] */
    const float* b3;                  /* [out_dim] */
} ej_mlp;

/* Validate, allocate library-owned device state for E envs on the current CUDA device.
 * Errors: EJ_ERR_PARAM (field named), EJ_ERR_NOMEM, EJ_ERR_CUDA.  *out is NULL on failure;
 * a failed create leaves its message readable through ej_last_error(NULL). */
int ej_create(int32_t E, int32_t N, int32_t R, const ej_params* p, ej_env** out);
int ej_destroy(ej_env* h);
/* cudaStream_t (as void*) all later calls are enqueued on. */
int ej_set_stream(ej_env* h, void* cuda_stream);
int ej_layout(const ej_env* h, ej_layout_info* out);
const char* ej_last_error(const ej_env* h);

/* Full re-initialisation (G29, G30): coin = starting_coin, everything else 0, books
 * empty, rates 0, t = 0, skills drawn from Philox(seed; global env, agent).  Same (params,
 * seed) => bit-identical state. */
int ej_reset(ej_env* h, uint64_t seed);

/* Observation of the current state (e.g. right after reset) into obs_out (device, obs_floats). */
int ej_observe(ej_env* h, float* obs_out);

/* f1: action mask of the current state ("unavailable actions" get zero probability;
 * P:199; action preconditions P:145-168; order cap P:277) into mask_out, device, [E][N][A] bytes,
 * 1 = available, 4-byte aligned: gather and no-op always; craft iff #{r : inv[r] >= craft_units} >=
 * craft_distinct (PER_RESOURCE r: inv[r] >= craft_units); buy (r, p) iff coin >= prices[p] and live
 * orders < max_active_orders; sell (r, p) iff inv[r] >= 1 and live orders < max_active_orders.  With
 * book_cap == 0 an action is available exactly when submitting it would not bump the env's `invalid`
 * counter; the per-book cap depends on the step's arrival order and is not part of the mask (G15).
 * Errors: EJ_ERR_PARAM (NULL / misaligned pointer), EJ_ERR_STATE (before reset), EJ_ERR_CUDA. */
int ej_action_mask(ej_env* h, uint8_t* mask_out);

/* One step of all E envs (order of effects G1: actions -> match -> expire -> tax -> rewards ->
 * observations -> t++).
 *  actions      device [E][N] int32 action indices (layout ej_layout_info.base_*)
 *  gov_actions  device [E][B] int32 rate-level indices; read every step, applied at period ends (G18)
 *  obs_out      device, one buffer of obs_floats floats with two regions: population
 *               [E][N][D_pop] dense, then government [E][D_gov_pad] at gov_obs_offset; or NULL
 *  rew_out      device [E][N+1] float, last = government; or NULL
 *  done_out     device [E] uint8; or NULL */
int ej_step(ej_env* h, const int32_t* actions, const int32_t* gov_actions, float* obs_out, float* rew_out,
            uint8_t* done_out);

/* Same step with HOST buffers (pinned or pageable): copies actions host->device, steps, copies
 * observations / rewards / done device->host, and synchronises the stream before returning. */
int ej_step_host(ej_env* h, const int32_t* actions, const int32_t* gov_actions, float* obs_out, float* rew_out,
                 uint8_t* done_out);

/* f2: the same step with HOST buffers and FACTORED observations.  Every value of the dense
 * observation leaves once: the 3R + 4 agent-private columns per agent, the 5R + B + 2 env-wide columns (market
 * statistics, tax rates, timers: P:424) once per env instead of N times, so the device->host copy carries
 * 4 N (3R + 4) + 4 ceil4(5R + B + 2) instead of 4 N D_pop bytes per env (2.5x fewer at the headline shape).
 *  actions, gov_actions  host, as ej_step
 *  priv_out     host [E][N][3R + 4] float: columns 0 .. 3R + 3 of the dense population rows
 *  shared_out   host [E][ceil4(5R + B + 2)] float: columns 3R + 4 .. D_pop - 1 of every row of the env
 *  gov_obs_out  host [E][D_gov_pad] float, or NULL
 *  rew_out      host [E][N+1] float, or NULL;  done_out  host [E] uint8, or NULL
 * Shapes whose rows cannot be staged (see ej_rollout_io.obs_priv_ring) and policy mode: EJ_ERR_PARAM.
 * Synchronises the stream before returning; staging buffers are library-owned. */
int ej_step_host_factored(ej_env* h, const int32_t* actions, const int32_t* gov_actions, float* priv_out,
                          float* shared_out, float* gov_obs_out, float* rew_out, uint8_t* done_out);

/* T steps in ONE persistent launch: each env's state stays in shared memory for the whole
 * call.  Actions come from io->actions_in / gov_actions_in or, when NULL, from the Philox/CDF
 * generator (ej_set_action_cdf; uniform over the A actions by default).  io may be NULL
 * (no outputs).  Envs that reach episode_length stay done (G28) unless io->auto_reset is set (f4).
 * Limits (EJ_ERR_PARAM): ring_depth * obs_floats < 2^32 and, with actions_in, T * E * N < 2^32
 * (the kernels index rings and action streams with 32-bit element offsets). */
int ej_rollout(ej_env* h, int32_t T, const ej_rollout_io* io);

/* Cumulative uint32 thresholds of the rollout's action generator: action = smallest a with
 * x < cdf[a], x = Philox word 0; the last entry is read as 2^32.  cdf is a HOST pointer [A]. */
int ej_set_action_cdf(ej_env* h, const uint32_t* cdf, int32_t A);

/* Canonical, representation-free state dump of envs [env_begin, env_begin+env_count) into /
 * from a HOST buffer of env_count*state_words int32 words (layout: DESIGN.md "Canonical state
 * dump").  Both synchronise the stream.  Cold path: used by tests and checkpointing.
 * The dump holds the state of the economies, not the Philox key: ej_set_state needs a handle that was
 * reset (EJ_ERR_STATE otherwise), and a restored run continues draw for draw only if that ej_reset used
 * the seed of the run the dump was taken from.  ej_set_state rejects (EJ_ERR_PARAM) dumps whose books are
 * crossed (best bid >= best ask: resting books are uncrossed after every step, G13), whose orders are off
 * the price grid or exceed max_active_orders per agent. */
int ej_get_state(ej_env* h, int32_t env_begin, int32_t env_count, int32_t* words, size_t n_words);
int ej_set_state(ej_env* h, int32_t env_begin, int32_t env_count, const int32_t* words, size_t n_words);

/* f1 masked sampling ("unavailable actions" get zero probability).  on != 0: whenever
 * ej_rollout / ej_policy_act draw population actions themselves, they draw among the actions that
 * ej_action_mask marks available in the state the step starts from:
 *  - table generator: integer weights w_a = cdf[a] - cdf[a-1] (last entry read as 2^32); S = sum of
 *    the available w_a; target = floor(x0 * S / 2^32), x0 = Philox stream 0 word 0; action = first
 *    available a whose running sum of available weights exceeds target (exact integer arithmetic);
 *  - policy: unavailable logits are excluded from the max, the sum and the running sum of the
 *    sampling rule of ej_set_policy.
 * Government levels and caller-supplied actions (actions_in) are never masked.  Default: off. */
int ej_set_action_masking(ej_env* h, int32_t on);

/* a12 (G33): install (or, with two NULLs, remove) the shared population policy and the
 * government policy.  While installed, ej_rollout draws its actions from them whenever
 * io->actions_in / gov_actions_in is NULL: logits = W3 tanh(W2 tanh(W1 bf16(obs) + b1) + b2) + b3
 * with bf16 operands, fp32 accumulation on the tensor cores and activations re-rounded to
 * bf16; action = first a with u * S < sum_{j<=a} exp(l_j - max l), u = (x >> 8) * 2^-24 from the
 * Philox word the CDF generator would have used (population: stream 0 word 0; government
 * head b: stream 1 + b/4, word b%4).  Errors: EJ_ERR_PARAM (dims), EJ_ERR_NOMEM, EJ_ERR_CUDA. */
int ej_set_policy(ej_env* h, const ej_mlp* pop, const ej_mlp* gov);

/* Sample actions for the current clock of every env from the installed policies.
 *  obs              device, obs_floats floats: observation of the current state (ej_observe / last ej_step)
 *  actions_out      device [E][N] int32
 *  gov_actions_out  device [E][B] int32
 *  pop_logits_out   device [E*N][A] float or NULL;  gov_logits_out  device [E][B*L] float or NULL */
int ej_policy_act(ej_env* h, const float* obs, int32_t* actions_out, int32_t* gov_actions_out, float* pop_logits_out,
                  float* gov_logits_out);

/* A rollout for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): E fresh economies (the state ej_reset(seed) gives) stepped T times with the caller's actions, in ONE call
 * that needs no handle and calls no cudaMalloc, cudaFree or other allocating routine.  The state blobs the kernels work
 * on live in a static device array of EJ_NOALLOC_SCRATCH_BYTES (4 MiB: 430 envs at N = 100, R = 2; 267 at R = 6; 34 at N = 1000),
 * which every GPU that loads the library holds until the process exits; E * device_state_bytes beyond it: EJ_ERR_PARAM
 * with the limit in ej_last_error(NULL).  Outputs are those of ej_rollout with ring_depth = T on a handle that was
 * just reset with the same seed:
 *  actions      device [T][E][N] int32;  gov_actions  device [T][E][B] int32  (both required)
 *  obs_ring     device [T][obs_floats] float, 16-byte aligned, or NULL
 *  rew_ring     device [T][E][N+1] float, or NULL;  done_ring  device [T][E] uint8, or NULL
 *  cuda_stream  cudaStream_t (as void*) the two kernels are enqueued on; the call does not synchronise
 * Every call shares the one scratch array and leaves its final state in it: calls that overlap on the GPU (different
 * streams, or graphs replayed concurrently) race; calls on one stream are ordered.  Each call starts by rewriting
 * every byte of the E blobs it uses, so nothing of an earlier call is read.  The first call on a device looks up
 * the array's device address (and raises the kernels' shared-memory limit): make it outside a graph capture, e.g.
 * with T = 0, which only does this set-up.  Errors: EJ_ERR_PARAM (field named), EJ_ERR_CUDA; text in
 * ej_last_error(NULL). */
#define EJ_NOALLOC_SCRATCH_BYTES (4u << 20)
int ej_rollout_noalloc(int32_t E, int32_t N, int32_t R, const ej_params* p, uint64_t seed, int32_t T, const int32_t* actions,
                       const int32_t* gov_actions, float* obs_ring, float* rew_ring, uint8_t* done_ring, void* cuda_stream);

/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
int64_t ej_launch_count(const ej_env* h);

#ifdef __cplusplus
}
#endif
#endif
