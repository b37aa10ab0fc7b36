/*
 * EconoJax CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded C restatement of the EconoJax environment step
 * (arXiv 2410.22165, /root/reference/PAPER.md = "P:n"; gap-filling readings from
 * SURVEY.md section 8(c) = "G1..G38", some after /root/reference/SPEC.md = "S:n").
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.  It shares no code, header, table or helper with the CUDA path
 * under paper_2410_22165_b200/csrc/, and neither side includes the other.
 *
 * Arithmetic contract (G31): agent state is IEEE-754 binary32; every state-changing
 * float operation below is ONE correctly rounded operation written as its own C
 * statement (compile with -ffp-contract=off, no -ffast-math).  Rewards and
 * statistics are evaluated in binary64 from the binary32 state.
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): tax worked example
 * P:195; utility closed forms (Eq.1); action counts 30/86; gather
 * worked values and the analytic probabilities of floor(SG+rho); craft
 * examples; matching examples and brute force on tiny books (P:162-164,
 * P:432-433); gini textbook values; mean/std/median against numpy; Philox4x32-10
 * known answers (Salmon et al. SC'11); conservation / escrow / telescoping
 * invariants on fuzzed episodes.
 * Parity unpinned (conventions of this build, fixed only by oracle == GPU): the
 * observation normalisation constants, the 7-bracket thresholds, craft_scale.
 */
#ifndef ECONOJAX_ORACLE_H
#define ECONOJAX_ORACLE_H

#include <stdint.h>
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_MAX_PRICES 16
#define ORC_MAX_BRACKETS 16
#define ORC_MAX_RATE_LEVELS 32
#define ORC_MAX_RESOURCES 16

#define ORC_CRAFT_SINGLE 0       /* the paper's single craft action (30/86 actions P:350) */
#define ORC_CRAFT_PER_RESOURCE 1 /* BASELINE.json's "convert r" variant (G3) */
#define ORC_SKILL_UNIFORM01 0
#define ORC_SKILL_PARETO_CLIP 1  /* Pareto(alpha=4) clipped, BASELINE.json configs 2-5 (G29) */
#define ORC_SKILL_NORMAL_CLIP 2  /* f3, section 5: "a normal distribution around 1.0 with a standard deviation of 1.0"
                                    (P:345), clipped to [lo, hi] (G42) */

/* Environment parameters; defaults are Table 2 unless BASELINE.json overrides. */
typedef struct orc_params {
    int32_t num_prices;                     /* P */
    int32_t prices[ORC_MAX_PRICES];         /* strictly ascending positive integers (G4) */
    int32_t episode_length;                 /* T */
    int32_t tax_period;
    int32_t num_brackets;                   /* B = number of thresholds + 1 */
    float thresholds[ORC_MAX_BRACKETS];     /* B-1 used, strictly ascending (G32) */
    int32_t num_rate_levels;                /* L (21) */
    float rate_table[ORC_MAX_RATE_LEVELS];  /* rate of level k, supplied by the caller (G5) */
    int32_t allow_noop;
    float starting_coin;
    int32_t order_expiry;
    int32_t max_active_orders;              /* M */
    int32_t book_cap;                       /* K per (resource, side); 0 = unbounded (G15) */
    int32_t craft_units;                    /* R_kappa */
    int32_t craft_distinct;                 /* R_d */
    int32_t craft_mode;                     /* ORC_CRAFT_* (G3) */
    float labor_craft, labor_gather, labor_trade;
    float eta;
    float omega;
    float craft_scale;                      /* "scaled by a constant" P:158; 10 after S:119 (G6) */
    int32_t taxes_enabled;
    int32_t skill_init;                     /* ORC_SKILL_* */
    float skill_clip_lo, skill_clip_hi;     /* PARETO_CLIP bounds */
    float obs_scale_coin, obs_scale_count, obs_scale_price, obs_scale_labor; /* G25 */
    uint32_t env_id_base;                   /* global id of local env 0 (Philox counter word 0) */
    float skill_growth_rate;                /* f3: 0 = skills fixed (default); section 5 uses 0.005 */
    float skill_max;                        /* f3: "maximum skill level of 5" */
    float skill_mean, skill_std;            /* f3: NORMAL_CLIP parameters (1.0 and 1.0) */
} orc_params;

/* f3, normal skill draw (G42).  The paper names the distribution, not a generator.  To stay a pure
 * function of the Philox words with no transcendental function in it, the standard normal is the classical
 * sum of twelve uniforms: z = sum_{k<12} u_k - 6 with u_k = (word_k >> 8) * 2^-24 (mean 0, variance 1 up to the
 * 2^-24 lattice, support [-6, 6)); the sum is an exact integer, z and std * z are exact in binary64, then
 *   skill = clip((float)(mean + std * z), lo, hi). */
float orc_normal_skill(const uint32_t words[12], float mean, float std, float lo, float hi);

/* f3, skill growth ("Whenever an agent gathers or crafts, the respective skill is increased
 * by 0.5%.  This 0.5% bonus shrinks as the agent approaches the maximum skill level of 5"; the
 * paper gives no formula: linear damping after S:101, G41):
 *   skill' = min(max, skill + skill * (rate * (1 - skill / max))), each operation rounded to binary32. */
float orc_progress_skill(float skill, float rate, float max);

typedef struct orc_sim orc_sim;

/* ---- rule-level functions (pinned one by one in tests/test_oracle_rules.py) ---- */

/* Philox4x32-10, Salmon et al. SC'11 (G30). */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* u = (x >> 8) * 2^-24 in [0,1). */
float orc_u01(uint32_t x);
/* floor(SG + rho), rho = u * 1.1 (G8). */
int32_t orc_gather_amount(float SG, float u);
/* Number of discrete actions: R + (1|R) + 2*R*P + noop (30/86 at P:350). */
int32_t orc_num_actions(int32_t R, int32_t P, int32_t craft_mode, int32_t allow_noop);
/* Craft on one inventory; r_named is used only in PER_RESOURCE mode.  Returns 1 and
 * consumes if valid, else returns 0 and leaves inv untouched (G7). */
int32_t orc_craft_consume(int32_t* inv, int32_t R, int32_t craft_units, int32_t craft_distinct,
                          int32_t craft_mode, int32_t r_named);
/* Bracketed marginal tax. B brackets, B-1 thresholds. */
float orc_marginal_tax(float income, const float* thresholds, const float* rates, int32_t B);
/* Eq.1. */
double orc_utility(double C, double L, double eta);
/* Gini index, mean-absolute-difference form (G23). */
double orc_gini(const float* c, int32_t n);
/* Eq.3-5 with Eq.4 read as omega*(1-gini) + (1-omega) (G22). */
void orc_social_welfare(const float* c, int32_t n, double omega, double* eq, double* prod, double* u_g);
/* mean, population std (binary64) and midpoint median (binary32 ops) of n values (G26). */
void orc_stats(const float* x, int32_t n, double* mean, double* std, float* median);

/* One order of a book. */
typedef struct orc_order {
    int32_t price;     /* coin */
    int32_t owner;     /* agent index */
    int32_t placed_at; /* step index */
    uint32_t key;      /* arrival tie key of its step (G11) */
} orc_order;
/* One executed trade. */
typedef struct orc_trade {
    int32_t buyer, seller, bid_price, ask_price, price;
} orc_trade;
/* One matching round on one resource's book (G11-G13): repeatedly
 * take the best bid and the best ask, trade while bid >= ask at the price of the later
 * arrival.  Matched orders are removed from the arrays (*nb, *na updated, remaining
 * orders keep their relative order).  Returns the number of trades written to `out`
 * (capacity max_out). */
int32_t orc_match_book(orc_order* bids, int32_t* nb, orc_order* asks, int32_t* na,
                       orc_trade* out, int32_t max_out);

/* ---- environment-level API ---- */
orc_sim* orc_create(int32_t E, int32_t N, int32_t R, const orc_params* p);
void orc_destroy(orc_sim* s);
const char* orc_last_error(void);
int32_t orc_obs_dim_pop(const orc_sim* s); /* 6 + 8R + B */
int32_t orc_obs_dim_gov(const orc_sim* s); /* 3(3+R) + B + 2 */
void orc_reset(orc_sim* s, uint64_t seed);
/* f4 (G44): envs [env_begin, +env_count) start episode `episode`: the state of a reset, every random draw of the
 * episode keyed by (seed, env, agent, t, stream | episode << 8).  orc_reset starts episode 0 everywhere. */
void orc_begin_episode(orc_sim* s, int32_t env_begin, int32_t env_count, int32_t episode);
/* f4: orc_step for an auto-resetting rollout: an env whose episode ends with this step starts its next episode at
 * once and returns the observation of the fresh state; rewards and done are the step's own. */
void orc_step_auto(orc_sim* s, int32_t env_begin, int32_t env_count, const int32_t* actions,
                   const int32_t* gov_actions, float* obs_pop, float* obs_gov, float* rew, uint8_t* done);
/* Observation of the current state of envs [env_begin, env_begin+env_count) (used after reset). */
void orc_observe(orc_sim* s, int32_t env_begin, int32_t env_count, float* obs_pop, float* obs_gov);
/* One step of envs [env_begin, env_begin+env_count).  actions [env_count][N], gov_actions
 * [env_count][B], obs_pop [env_count][N][D_pop], obs_gov [env_count][D_gov], rew
 * [env_count][N+1] (last = government), done [env_count]; output pointers may be NULL. */
void orc_step(orc_sim* s, int32_t env_begin, int32_t env_count, const int32_t* actions,
              const int32_t* gov_actions, float* obs_pop, float* obs_gov, float* rew, uint8_t* done);
/* Draw this step's actions for envs [env_begin, +env_count) from the Philox/CDF generator
 * (G30): population action = smallest a with x0 < cdf[a] (last entry read as 2^32),
 * government level = (x * L) >> 32 from streams 1.. . */
void orc_draw_actions(const orc_sim* s, int32_t env_begin, int32_t env_count, const uint32_t* cdf,
                      int32_t* actions, int32_t* gov_actions);
/* f1: availability of every action for every agent in the current state (rules in the .c file):
 * mask [env_count][N][A] bytes, 1 = available. */
void orc_action_mask(const orc_sim* s, int32_t env_begin, int32_t env_count, uint8_t* mask);

/* f1 masked sampling: orc_draw_actions restricted to the available actions of the
 * current state and renormalised with integer weights (exact); definition in the .c file. */
void orc_draw_actions_masked(const orc_sim* s, int32_t env_begin, int32_t env_count, const uint32_t* cdf,
                             int32_t* actions, int32_t* gov_actions);
/* Canonical, representation-free state dump (layout in DESIGN.md "Canonical state dump"). */
size_t orc_state_words(const orc_sim* s);
void orc_get_state(const orc_sim* s, int32_t env_begin, int32_t env_count, int32_t* words);
/* Scripted-test setters. */
void orc_set_agent(orc_sim* s, int32_t env, int32_t agent, float coin, const int32_t* inv,
                   const float* SG, float SC);
void orc_set_rates(orc_sim* s, int32_t env, const float* rates);
/* Per-agent scalar getters for tests: what = 0 coin, 1 labor, 2 income. */
float orc_get_agent_f(const orc_sim* s, int32_t env, int32_t agent, int32_t what);

#ifdef __cplusplus
}
#endif
#endif
