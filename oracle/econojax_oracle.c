/*
 * EconoJax CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see econojax_oracle.h).
 *
 * Plain sequential C.  One env at a time, one agent at a time, books as flat arrays
 * with linear scans.  No blocking, fusion or reordering beyond what the paper (P:n)
 * and the readings G1..G38 (restated in DESIGN.md) state.
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/__init__.py).
 */
#include "econojax_oracle.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------- */
/* Rule-level functions                                                       */
/* ------------------------------------------------------------------------- */

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), as restated in G30: ten rounds of
 * hi0:lo0 = M0*c0, hi1:lo1 = M1*c2, c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0), key bumped
 * by the Weyl constants between rounds. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Uniform float in [0,1) from the top 24 bits (G30). Exact in binary32. */
float orc_u01(uint32_t x) {
    return (float)(x >> 8) * (1.0f / 16777216.0f);
}

/* amount gathered = floor(SG + rho), rho uniform in [0, 1.1).  G8: rho = fl(u*1.1f),
 * then one add, then floor: two separately rounded binary32 operations. */
int32_t orc_gather_amount(float SG, float u) {
    float rho = u * 1.1f;
    float s = SG + rho;
    return (int32_t)floorf(s);
}

/* S:47, pinned by the paper's 30 and 86 actions at R=4 and R=12 with 3 prices. */
int32_t orc_num_actions(int32_t R, int32_t P, int32_t craft_mode, int32_t allow_noop) {
    int32_t n_craft = (craft_mode == ORC_CRAFT_PER_RESOURCE) ? R : 1;
    return R + n_craft + 2 * R * P + (allow_noop ? 1 : 0);
}

/* P:154-157.  SINGLE: valid iff at least R_d resources hold >= R_kappa units; consumes
 * R_kappa units of each of the R_d most-held resources, ties to the lowest index (G7).
 * PER_RESOURCE (G3): valid iff inv[r_named] >= R_kappa; consumes only that resource. */
int32_t orc_craft_consume(int32_t* inv, int32_t R, int32_t craft_units, int32_t craft_distinct,
                          int32_t craft_mode, int32_t r_named) {
    if (craft_mode == ORC_CRAFT_PER_RESOURCE) {
        if (r_named < 0 || r_named >= R) return 0;
        if (inv[r_named] < craft_units) return 0;
        inv[r_named] -= craft_units;
        return 1;
    }
    int32_t enough = 0;
    for (int32_t r = 0; r < R; ++r)
        if (inv[r] >= craft_units) ++enough;
    if (enough < craft_distinct) return 0;
    int32_t used[ORC_MAX_RESOURCES];
    for (int32_t r = 0; r < R; ++r) used[r] = 0;
    for (int32_t k = 0; k < craft_distinct; ++k) {
        int32_t best = -1;
        for (int32_t r = 0; r < R; ++r) {
            if (used[r]) continue;
            if (best < 0 || inv[r] > inv[best]) best = r; /* strict '>' keeps the lowest index on ties */
        }
        used[best] = 1;
        inv[best] -= craft_units;
    }
    return 1;
}

/* brackets [0,thr0), [thr0,thr1), ..., [thr_{B-2}, inf); tax is the sum over
 * brackets of rate * (part of the income inside the bracket).  Worked example P:195:
 * 130 at (10%,30%,50%) on [50;100] pays 0.10*50 + 0.30*50 + 0.50*30 = 35. */
float orc_marginal_tax(float income, const float* thresholds, const float* rates, int32_t B) {
    float tax = 0.0f;
    float lo = 0.0f;
    for (int32_t b = 0; b < B; ++b) {
        float hi = (b < B - 1) ? thresholds[b] : INFINITY;
        float top = (income < hi) ? income : hi;
        float por = top - lo;
        if (por < 0.0f) por = 0.0f;
        float part = rates[b] * por;
        tax = tax + part;
        lo = hi;
    }
    return tax;
}

/* Eq.1: u = (C^(1-eta) - 1)/(1-eta) - L. */
double orc_utility(double C, double L, double eta) {
    double a = 1.0 - eta;
    return (pow(C, a) - 1.0) / a - L;
}

/* Gini index in its defining mean-absolute-difference form (G23):
 * sum_i sum_j |c_i - c_j| / (2 n sum_k c_k); 0 when the total is 0 or n = 1. */
double orc_gini(const float* c, int32_t n) {
    double total = 0.0;
    for (int32_t i = 0; i < n; ++i) total += (double)c[i];
    if (n <= 1 || total == 0.0) return 0.0;
    double sad = 0.0;
    for (int32_t i = 0; i < n; ++i)
        for (int32_t j = 0; j < n; ++j) sad += fabs((double)c[i] - (double)c[j]);
    return sad / (2.0 * (double)n * total);
}

/* Eq.3 u_g = Eq * Prod; Eq.5 Prod = sum C; Eq.4 is garbled in the source
 * (P:180 prints "+ 1 + omega"); G22 reads it as omega*(1-gini) + (1-omega), which gives
 * the "Equality: (1 - gini)" of Fig.2 at omega = 1. */
void orc_social_welfare(const float* c, int32_t n, double omega, double* eq, double* prod, double* u_g) {
    double p = 0.0;
    for (int32_t i = 0; i < n; ++i) p += (double)c[i];
    double g = orc_gini(c, n);
    double e = omega * (1.0 - g) + (1.0 - omega);
    *eq = e;
    *prod = p;
    *u_g = e * p;
}

/* Mean, population standard deviation (two passes, binary64) and median (G26).
 * Median: middle order statistic for odd n, fl(0.5f * fl(a + b)) of the two middle ones
 * for even n, on the raw binary32 values. */
void orc_stats(const float* x, int32_t n, double* mean, double* std, float* median) {
    double sum = 0.0;
    for (int32_t i = 0; i < n; ++i) sum += (double)x[i];
    double m = sum / (double)n;
    double ss = 0.0;
    for (int32_t i = 0; i < n; ++i) {
        double d = (double)x[i] - m;
        ss += d * d;
    }
    *mean = m;
    *std = sqrt(ss / (double)n);
    float* tmp = (float*)malloc(sizeof(float) * (size_t)n);
    memcpy(tmp, x, sizeof(float) * (size_t)n);
    for (int32_t i = 1; i < n; ++i) { /* insertion sort */
        float v = tmp[i];
        int32_t j = i - 1;
        while (j >= 0 && tmp[j] > v) { tmp[j + 1] = tmp[j]; --j; }
        tmp[j + 1] = v;
    }
    if (n % 2 == 1) {
        *median = tmp[n / 2];
    } else {
        float s = tmp[n / 2 - 1] + tmp[n / 2];
        *median = 0.5f * s;
    }
    free(tmp);
}

/* Arrival order (G11): an older step precedes a newer one; inside a step the Philox tie
 * key, then the agent index.  Returns 1 iff a arrived strictly after b. */
static int arrived_after(const orc_order* a, const orc_order* b) {
    if (a->placed_at != b->placed_at) return a->placed_at > b->placed_at;
    if (a->key != b->key) return a->key > b->key;
    return a->owner > b->owner;
}

static void remove_order(orc_order* o, int32_t* n, int32_t idx) {
    for (int32_t i = idx; i + 1 < *n; ++i) o[i] = o[i + 1];
    --*n;
}

/* "high-value orders (high bids / low asks) are evaluated first. Ties are then
 * first broken by the age of the order and lastly at random"; the trade price
 * is that of the order placed last.  G12: owner-equal pairs trade like any other. */
int32_t orc_match_book(orc_order* bids, int32_t* nb, orc_order* asks, int32_t* na,
                       orc_trade* out, int32_t max_out) {
    int32_t n_tr = 0;
    for (;;) {
        if (*nb == 0 || *na == 0) break;
        int32_t ib = 0;
        for (int32_t i = 1; i < *nb; ++i) {
            if (bids[i].price > bids[ib].price ||
                (bids[i].price == bids[ib].price && arrived_after(&bids[ib], &bids[i])))
                ib = i;
        }
        int32_t ia = 0;
        for (int32_t i = 1; i < *na; ++i) {
            if (asks[i].price < asks[ia].price ||
                (asks[i].price == asks[ia].price && arrived_after(&asks[ia], &asks[i])))
                ia = i;
        }
        if (bids[ib].price < asks[ia].price) break;
        orc_trade tr;
        tr.buyer = bids[ib].owner;
        tr.seller = asks[ia].owner;
        tr.bid_price = bids[ib].price;
        tr.ask_price = asks[ia].price;
        tr.price = arrived_after(&bids[ib], &asks[ia]) ? bids[ib].price : asks[ia].price;
        if (n_tr < max_out) out[n_tr] = tr;
        ++n_tr;
        remove_order(bids, nb, ib);
        remove_order(asks, na, ia);
    }
    return n_tr;
}

/* ------------------------------------------------------------------------- */
/* Environment                                                                */
/* ------------------------------------------------------------------------- */

typedef struct orc_book {
    orc_order* o;
    int32_t n, cap;
} orc_book;

typedef struct orc_env {
    int32_t t;
    int32_t episode;   /* f4: index of the episode this env is in (0 after orc_reset); part of every Philox counter (G44) */
    float* coin;       /* [N] inventory coin C_i */
    float* labor;      /* [N] cumulative labor L_i */
    float* income;     /* [N] earnings since the last collection (G16) */
    float* SC;         /* [N] craft skill */
    float* SG;         /* [N][R] gather skills */
    int32_t* inv;      /* [N][R] */
    int32_t* esc_res;  /* [N][R] escrow units */
    int32_t* esc_coin; /* [N] escrow coin, integer sum of bid prices (G10) */
    int32_t* n_live;   /* [N] live orders */
    orc_book* book;    /* [R][2], side 0 = bids, 1 = asks */
    int32_t* last_price; /* [R], 0 = no trade yet */
    float rates[ORC_MAX_BRACKETS];
    double u_g_prev;
    int32_t n_trades, n_placed, n_invalid, n_expired, n_bad_gov;
} orc_env;

struct orc_sim {
    int32_t E, N, R;
    orc_params p;
    uint64_t seed;
    orc_env* env;
};

static char g_err[256];
const char* orc_last_error(void) { return g_err; }

static void book_push(orc_book* b, orc_order o) {
    if (b->n == b->cap) {
        b->cap = b->cap ? 2 * b->cap : 64;
        b->o = (orc_order*)realloc(b->o, sizeof(orc_order) * (size_t)b->cap);
    }
    b->o[b->n++] = o;
}

orc_sim* orc_create(int32_t E, int32_t N, int32_t R, const orc_params* p) {
    g_err[0] = 0;
    if (E < 1 || N < 1 || R < 1 || R > ORC_MAX_RESOURCES) { snprintf(g_err, sizeof g_err, "E/N/R"); return NULL; }
    if (p->num_prices < 1 || p->num_prices > ORC_MAX_PRICES) { snprintf(g_err, sizeof g_err, "num_prices"); return NULL; }
    for (int i = 0; i < p->num_prices; ++i)
        if (p->prices[i] < 1 || (i > 0 && p->prices[i] <= p->prices[i - 1])) { snprintf(g_err, sizeof g_err, "prices"); return NULL; }
    if (p->num_brackets < 1 || p->num_brackets > ORC_MAX_BRACKETS) { snprintf(g_err, sizeof g_err, "num_brackets"); return NULL; }
    for (int i = 0; i + 1 < p->num_brackets; ++i)
        if (!(p->thresholds[i] > (i ? p->thresholds[i - 1] : 0.0f))) { snprintf(g_err, sizeof g_err, "thresholds"); return NULL; }
    if (p->num_rate_levels < 1 || p->num_rate_levels > ORC_MAX_RATE_LEVELS) { snprintf(g_err, sizeof g_err, "num_rate_levels"); return NULL; }
    if (p->craft_mode == ORC_CRAFT_SINGLE && (p->craft_distinct < 1 || p->craft_distinct > R)) { snprintf(g_err, sizeof g_err, "craft_distinct"); return NULL; }
    if (p->eta == 1.0f) { snprintf(g_err, sizeof g_err, "eta"); return NULL; }
    if (p->episode_length < 1 || p->tax_period < 1) { snprintf(g_err, sizeof g_err, "episode_length/tax_period"); return NULL; }
    orc_sim* s = (orc_sim*)calloc(1, sizeof(orc_sim));
    s->E = E; s->N = N; s->R = R; s->p = *p;
    s->env = (orc_env*)calloc((size_t)E, sizeof(orc_env));
    for (int32_t e = 0; e < E; ++e) {
        orc_env* v = &s->env[e];
        v->coin = (float*)calloc((size_t)N, sizeof(float));
        v->labor = (float*)calloc((size_t)N, sizeof(float));
        v->income = (float*)calloc((size_t)N, sizeof(float));
        v->SC = (float*)calloc((size_t)N, sizeof(float));
        v->SG = (float*)calloc((size_t)N * R, sizeof(float));
        v->inv = (int32_t*)calloc((size_t)N * R, sizeof(int32_t));
        v->esc_res = (int32_t*)calloc((size_t)N * R, sizeof(int32_t));
        v->esc_coin = (int32_t*)calloc((size_t)N, sizeof(int32_t));
        v->n_live = (int32_t*)calloc((size_t)N, sizeof(int32_t));
        v->book = (orc_book*)calloc((size_t)R * 2, sizeof(orc_book));
        v->last_price = (int32_t*)calloc((size_t)R, sizeof(int32_t));
    }
    return s;
}

void orc_destroy(orc_sim* s) {
    if (!s) return;
    for (int32_t e = 0; e < s->E; ++e) {
        orc_env* v = &s->env[e];
        free(v->coin); free(v->labor); free(v->income); free(v->SC); free(v->SG);
        free(v->inv); free(v->esc_res); free(v->esc_coin); free(v->n_live);
        for (int32_t b = 0; b < 2 * s->R; ++b) free(v->book[b].o);
        free(v->book); free(v->last_price);
    }
    free(s->env);
    free(s);
}

int32_t orc_obs_dim_pop(const orc_sim* s) { return 6 + 8 * s->R + s->p.num_brackets; }
int32_t orc_obs_dim_gov(const orc_sim* s) { return 3 * (3 + s->R) + s->p.num_brackets + 2; }

/* Counter = (global env id, agent, t, stream | episode << 8) (G30; G44: the episode index rides in the upper bits of
 * the stream word, so episode 0 draws exactly what the counters of G30 draw). */
static void draw(const orc_sim* s, uint32_t episode, uint32_t env_gid, uint32_t agent, uint32_t t, uint32_t stream, uint32_t x[4]) {
    uint32_t ctr[4] = { env_gid, agent, t, stream | (episode << 8) };
    uint32_t key[2] = { (uint32_t)(s->seed & 0xFFFFFFFFu), (uint32_t)(s->seed >> 32) };
    orc_philox4x32_10(ctr, key, x);
}

/* Skill draw number d of an agent: Philox stream 16, "t" field = d/4, word d%4 (G30).
 * NORMAL_CLIP (f3, G42): stream 17, "t" fields 3d, 3d+1, 3d+2 give the twelve words of draw d. */
static float skill_draw(const orc_sim* s, uint32_t episode, uint32_t env_gid, uint32_t agent, int32_t d) {
    uint32_t x[4];
    if (s->p.skill_init == ORC_SKILL_NORMAL_CLIP) {
        uint32_t w[12];
        for (int32_t j = 0; j < 3; ++j) draw(s, episode, env_gid, agent, (uint32_t)(3 * d + j), 17u, &w[4 * j]);
        return orc_normal_skill(w, s->p.skill_mean, s->p.skill_std, s->p.skill_clip_lo, s->p.skill_clip_hi);
    }
    draw(s, episode, env_gid, agent, (uint32_t)(d / 4), 16u, x);
    float u = orc_u01(x[d % 4]);
    if (s->p.skill_init == ORC_SKILL_UNIFORM01) return u;
    /* Pareto(alpha=4, x_m=1) by inversion with correctly rounded ops only (G29, 8(c) "Skill init"). */
    float v = 1.0f - u;
    float r = sqrtf(v);
    r = sqrtf(r);
    float x1 = 1.0f / r;
    if (x1 < s->p.skill_clip_lo) x1 = s->p.skill_clip_lo;
    if (x1 > s->p.skill_clip_hi) x1 = s->p.skill_clip_hi;
    return x1;
}

static double env_welfare(const orc_sim* s, const orc_env* v) {
    double eq, prod, ug;
    orc_social_welfare(v->coin, s->N, (double)s->p.omega, &eq, &prod, &ug);
    return ug;
}

/* every agent holds starting_coin, nothing else; books empty; rates zero; t = 0.  Skills are drawn anew
 * from the counters of the given episode (f4, G44); the counters (trades, invalid actions, ...) keep running over
 * episodes. */
static void init_env(const orc_sim* s, orc_env* v, uint32_t gid, int32_t episode, int32_t clear_counters) {
    const int32_t N = s->N, R = s->R;
    v->t = 0;
    v->episode = episode;
    for (int32_t i = 0; i < N; ++i) {
        v->coin[i] = s->p.starting_coin;
        v->labor[i] = 0.0f;
        v->income[i] = 0.0f;
        v->esc_coin[i] = 0;
        v->n_live[i] = 0;
        for (int32_t r = 0; r < R; ++r) {
            v->inv[i * R + r] = 0;
            v->esc_res[i * R + r] = 0;
            v->SG[i * R + r] = skill_draw(s, (uint32_t)episode, gid, (uint32_t)i, r);
        }
        v->SC[i] = skill_draw(s, (uint32_t)episode, gid, (uint32_t)i, R);
    }
    for (int32_t b = 0; b < 2 * R; ++b) v->book[b].n = 0;
    for (int32_t r = 0; r < R; ++r) v->last_price[r] = 0;
    for (int32_t b = 0; b < ORC_MAX_BRACKETS; ++b) v->rates[b] = 0.0f;
    if (clear_counters) v->n_trades = v->n_placed = v->n_invalid = v->n_expired = v->n_bad_gov = 0;
    v->u_g_prev = env_welfare(s, v);
}

void orc_reset(orc_sim* s, uint64_t seed) {
    s->seed = seed;
    for (int32_t e = 0; e < s->E; ++e) init_env(s, &s->env[e], s->p.env_id_base + (uint32_t)e, 0, 1);
}

/* f4 (G44): start episode `episode` in envs [env_begin, +env_count): the state of a reset, with every random draw of
 * the episode keyed by its index.  orc_reset = episode 0 everywhere. */
void orc_begin_episode(orc_sim* s, int32_t env_begin, int32_t env_count, int32_t episode) {
    for (int32_t k = 0; k < env_count; ++k)
        init_env(s, &s->env[env_begin + k], s->p.env_id_base + (uint32_t)(env_begin + k), episode, 0);
}

/* Observation layouts: SURVEY 8(c) "Population observation layout" / "Government observation
 * layout" (Fig.1; G25-G27). tq = the clock the timers show. */
static void build_obs(const orc_sim* s, const orc_env* v, int32_t tq, float* obs_pop, float* obs_gov) {
    const int32_t N = s->N, R = s->R, B = s->p.num_brackets;
    const orc_params* p = &s->p;
    /* market statistics per resource: best bid, best ask, counts, last price */
    float mstat[ORC_MAX_RESOURCES][5];
    for (int32_t r = 0; r < R; ++r) {
        const orc_book* bb = &v->book[2 * r + 0];
        const orc_book* ab = &v->book[2 * r + 1];
        int32_t best_bid = 0, best_ask = 0;
        for (int32_t i = 0; i < bb->n; ++i)
            if (bb->o[i].price > best_bid) best_bid = bb->o[i].price;
        for (int32_t i = 0; i < ab->n; ++i)
            if (best_ask == 0 || ab->o[i].price < best_ask) best_ask = ab->o[i].price;
        mstat[r][0] = (float)best_bid * p->obs_scale_price;
        mstat[r][1] = (float)best_ask * p->obs_scale_price;
        mstat[r][2] = (float)bb->n * p->obs_scale_count;
        mstat[r][3] = (float)ab->n * p->obs_scale_count;
        mstat[r][4] = (float)v->last_price[r] * p->obs_scale_price;
    }
    float timer_period = (float)(tq % p->tax_period) / (float)p->tax_period;
    float timer_episode = (float)tq / (float)p->episode_length;
    if (obs_pop) {
        const int32_t D = orc_obs_dim_pop(s);
        for (int32_t i = 0; i < N; ++i) {
            float* o = obs_pop + (size_t)i * D;
            int32_t k = 0;
            o[k++] = v->coin[i] * p->obs_scale_coin;
            for (int32_t r = 0; r < R; ++r) o[k++] = (float)v->inv[i * R + r] * p->obs_scale_count;
            o[k++] = (float)v->esc_coin[i] * p->obs_scale_coin;
            for (int32_t r = 0; r < R; ++r) o[k++] = (float)v->esc_res[i * R + r] * p->obs_scale_count;
            for (int32_t r = 0; r < R; ++r) o[k++] = v->SG[i * R + r];
            o[k++] = v->SC[i];
            o[k++] = v->labor[i] * p->obs_scale_labor;
            for (int32_t r = 0; r < R; ++r)
                for (int32_t j = 0; j < 5; ++j) o[k++] = mstat[r][j];
            for (int32_t b = 0; b < B; ++b) o[k++] = v->rates[b];
            o[k++] = timer_period;
            o[k++] = timer_episode;
        }
    }
    if (obs_gov) {
        int32_t k = 0;
        float* x = (float*)malloc(sizeof(float) * (size_t)N);
        for (int32_t m = 0; m < 3 + R; ++m) {
            float scale;
            for (int32_t i = 0; i < N; ++i) {
                if (m == 0) x[i] = v->coin[i];
                else if (m == 1) x[i] = v->labor[i];
                else if (m == 2) x[i] = v->income[i];
                else x[i] = (float)v->inv[i * R + (m - 3)];
            }
            if (m == 0 || m == 2) scale = p->obs_scale_coin;
            else if (m == 1) scale = p->obs_scale_labor;
            else scale = p->obs_scale_count;
            double mean, std; float med;
            orc_stats(x, N, &mean, &std, &med);
            obs_gov[k++] = (float)(mean * (double)scale);
            obs_gov[k++] = (float)(std * (double)scale);
            obs_gov[k++] = med * scale;
        }
        free(x);
        for (int32_t b = 0; b < B; ++b) obs_gov[k++] = v->rates[b];
        obs_gov[k++] = timer_period;
        obs_gov[k++] = timer_episode;
    }
}

void orc_observe(orc_sim* s, int32_t env_begin, int32_t env_count, float* obs_pop, float* obs_gov) {
    const size_t Dp = (size_t)orc_obs_dim_pop(s), Dg = (size_t)orc_obs_dim_gov(s);
    for (int32_t k = 0; k < env_count; ++k) {
        const orc_env* v = &s->env[env_begin + k];
        build_obs(s, v, v->t, obs_pop ? obs_pop + (size_t)k * s->N * Dp : NULL, obs_gov ? obs_gov + (size_t)k * Dg : NULL);
    }
}

typedef struct cand {
    int32_t agent, r, side, price;
    uint32_t key;
} cand;

/* One env, one step, in the order actions -> match -> expire -> tax -> rewards -> obs -> t++ (G1). */
static void step_env(const orc_sim* s, orc_env* v, uint32_t gid, const int32_t* act, const int32_t* gov,
                     float* obs_pop, float* obs_gov, float* rew, uint8_t* done) {
    const orc_params* p = &s->p;
    const int32_t N = s->N, R = s->R, P = p->num_prices, B = p->num_brackets;
    const int32_t T = p->episode_length;

    if (v->t >= T) { /* G28: stepping a finished env is a no-op */
        if (rew) for (int32_t i = 0; i <= N; ++i) rew[i] = 0.0f;
        if (obs_pop || obs_gov) build_obs(s, v, v->t, obs_pop, obs_gov);
        if (done) *done = 1;
        return;
    }
    const int32_t t = v->t;

    double* u_pre = (double*)malloc(sizeof(double) * (size_t)N);
    for (int32_t i = 0; i < N; ++i) u_pre[i] = orc_utility((double)v->coin[i], (double)v->labor[i], (double)p->eta);

    /* ---- P1 actions (one action per agent per timestep) ---- */
    const int32_t n_craft = (p->craft_mode == ORC_CRAFT_PER_RESOURCE) ? R : 1;
    const int32_t base_buy = R + n_craft;
    const int32_t base_sell = base_buy + R * P;
    const int32_t A = orc_num_actions(R, P, p->craft_mode, p->allow_noop);
    cand* cands = (cand*)malloc(sizeof(cand) * (size_t)N);
    int32_t n_cand = 0;
    for (int32_t i = 0; i < N; ++i) {
        uint32_t x[4];
        draw(s, (uint32_t)v->episode, gid, (uint32_t)i, (uint32_t)t, 0u, x);
        const int32_t a = act[i];
        if (a < 0 || a >= A) { v->n_invalid++; continue; } /* G2 */
        if (a < R) { /* gather r */
            int32_t amt = orc_gather_amount(v->SG[i * R + a], orc_u01(x[1]));
            v->inv[i * R + a] += amt;
            v->labor[i] = v->labor[i] + p->labor_gather;
            if (p->skill_growth_rate > 0.0f) /* f3: the amount above used the skill before the increase */
                v->SG[i * R + a] = orc_progress_skill(v->SG[i * R + a], p->skill_growth_rate, p->skill_max);
        } else if (a < base_buy) { /* craft */
            if (orc_craft_consume(&v->inv[i * R], R, p->craft_units, p->craft_distinct, p->craft_mode, a - R)) {
                float pay = v->SC[i] * p->craft_scale;
                v->coin[i] = v->coin[i] + pay;
                v->income[i] = v->income[i] + pay;
                v->labor[i] = v->labor[i] + p->labor_craft;
                if (p->skill_growth_rate > 0.0f) /* f3: the payout above used the skill before the increase */
                    v->SC[i] = orc_progress_skill(v->SC[i], p->skill_growth_rate, p->skill_max);
            } else {
                v->n_invalid++;
            }
        } else if (a < base_sell + R * P) { /* market order */
            const int32_t side = (a >= base_sell) ? 1 : 0;
            const int32_t k = a - (side ? base_sell : base_buy);
            const int32_t r = k / P, price = p->prices[k % P];
            int32_t ok = v->n_live[i] < p->max_active_orders;
            if (side == 0) ok = ok && (v->coin[i] >= (float)price);
            else ok = ok && (v->inv[i * R + r] >= 1);
            if (!ok) { v->n_invalid++; continue; }
            cand c = { i, r, side, price, x[2] };
            cands[n_cand++] = c;
        } else {
            /* NO-OP: nothing, no labor */
        }
    }
    /* arrival order of this step's candidates: (key, agent) (G11); insertion sort */
    for (int32_t a = 1; a < n_cand; ++a) {
        cand c = cands[a];
        int32_t b = a - 1;
        while (b >= 0 && (cands[b].key > c.key || (cands[b].key == c.key && cands[b].agent > c.agent))) {
            cands[b + 1] = cands[b];
            --b;
        }
        cands[b + 1] = c;
    }
    /* acceptance against the book cap, counted from the book size at step start (G15) */
    {
        int32_t n_rest[2 * ORC_MAX_RESOURCES], seen[2 * ORC_MAX_RESOURCES];
        for (int32_t b = 0; b < 2 * R; ++b) { n_rest[b] = v->book[b].n; seen[b] = 0; }
        for (int32_t a = 0; a < n_cand; ++a) {
            const cand* c = &cands[a];
            const int32_t b = 2 * c->r + c->side;
            const int32_t j = seen[b]++;
            if (p->book_cap != 0 && !(n_rest[b] + j < p->book_cap)) { v->n_invalid++; continue; }
            const int32_t i = c->agent;
            if (c->side == 0) { /* escrow */
                v->coin[i] = v->coin[i] - (float)c->price;
                v->esc_coin[i] += c->price;
            } else {
                v->inv[i * R + c->r] -= 1;
                v->esc_res[i * R + c->r] += 1;
            }
            v->n_live[i] += 1;
            v->labor[i] = v->labor[i] + p->labor_trade;
            orc_order o = { c->price, i, t, c->key };
            book_push(&v->book[b], o);
            v->n_placed++;
        }
    }
    free(cands);

    /* ---- P2 match, per resource ---- */
    int32_t* credit = (int32_t*)calloc((size_t)N, sizeof(int32_t));
    int32_t* sale = (int32_t*)calloc((size_t)N, sizeof(int32_t));
    orc_trade* trades = (orc_trade*)malloc(sizeof(orc_trade) * (size_t)(N > 0 ? N : 1));
    for (int32_t r = 0; r < R; ++r) {
        orc_book* bb = &v->book[2 * r + 0];
        orc_book* ab = &v->book[2 * r + 1];
        /* every trade involves an order of this step (the resting book is uncrossed), so <= N */
        int32_t n_tr = orc_match_book(bb->o, &bb->n, ab->o, &ab->n, trades, N);
        for (int32_t k = 0; k < n_tr; ++k) {
            const orc_trade* tr = &trades[k];
            v->esc_coin[tr->buyer] -= tr->bid_price;
            credit[tr->buyer] += tr->bid_price - tr->price; /* refund of the escrowed excess */
            v->inv[tr->buyer * R + r] += 1;
            v->n_live[tr->buyer] -= 1;
            v->esc_res[tr->seller * R + r] -= 1;
            credit[tr->seller] += tr->price;
            sale[tr->seller] += tr->price;
            v->n_live[tr->seller] -= 1;
            v->last_price[r] = tr->price;
            v->n_trades++;
        }
    }
    free(trades);
    for (int32_t i = 0; i < N; ++i)
        if (sale[i] > 0) v->income[i] = v->income[i] + (float)sale[i]; /* G16 */

    /* ---- P3 expire (G14), then credit coin once ---- */
    for (int32_t b = 0; b < 2 * R; ++b) {
        orc_book* bk = &v->book[b];
        const int32_t r = b / 2, side = b % 2;
        int32_t w = 0;
        for (int32_t k = 0; k < bk->n; ++k) {
            const orc_order o = bk->o[k];
            if (t - o.placed_at >= p->order_expiry) {
                if (side == 0) { v->esc_coin[o.owner] -= o.price; credit[o.owner] += o.price; }
                else { v->esc_res[o.owner * R + r] -= 1; v->inv[o.owner * R + r] += 1; }
                v->n_live[o.owner] -= 1;
                v->n_expired++;
            } else {
                bk->o[w++] = o;
            }
        }
        bk->n = w;
    }
    for (int32_t i = 0; i < N; ++i)
        if (credit[i] > 0) v->coin[i] = v->coin[i] + (float)credit[i];
    free(credit);
    free(sale);

    /* ---- P4 tax at period end (G17-G20) ---- */
    if (p->taxes_enabled && (t + 1) % p->tax_period == 0) {
        int64_t pool_fx = 0; /* 2^-20 coin units, exact and order-free (G19) */
        for (int32_t i = 0; i < N; ++i) {
            float tax = orc_marginal_tax(v->income[i], p->thresholds, v->rates, B);
            if (tax > v->coin[i]) tax = v->coin[i]; /* G17 */
            v->coin[i] = v->coin[i] - tax;
            pool_fx += (int64_t)llrint((double)tax * 1048576.0);
        }
        float pool = (float)((double)pool_fx * (1.0 / 1048576.0));
        float share = pool / (float)N; /* P:195 "(1/n)" */
        for (int32_t i = 0; i < N; ++i) {
            v->coin[i] = v->coin[i] + share;
            v->income[i] = 0.0f;
        }
        for (int32_t b = 0; b < B; ++b) { /* new rates for the upcoming period */
            const int32_t lvl = gov[b];
            if (lvl < 0 || lvl >= p->num_rate_levels) { v->n_bad_gov++; continue; }
            v->rates[b] = p->rate_table[lvl];
        }
    }

    /* ---- P5 rewards (Eq.2) ---- */
    {
        double ug = env_welfare(s, v);
        if (rew) {
            for (int32_t i = 0; i < N; ++i) {
                double u_post = orc_utility((double)v->coin[i], (double)v->labor[i], (double)p->eta);
                rew[i] = (float)(u_post - u_pre[i]);
            }
            rew[N] = (float)(ug - v->u_g_prev);
        }
        v->u_g_prev = ug;
    }
    free(u_pre);

    /* ---- P6 observations of the post-step state, clock, done ---- */
    if (obs_pop || obs_gov) build_obs(s, v, t + 1, obs_pop, obs_gov);
    v->t = t + 1;
    if (done) *done = (uint8_t)(v->t == T);
}

void orc_step(orc_sim* s, int32_t env_begin, int32_t env_count, const int32_t* actions,
              const int32_t* gov_actions, float* obs_pop, float* obs_gov, float* rew, uint8_t* done) {
    const size_t N = (size_t)s->N, B = (size_t)s->p.num_brackets;
    const size_t Dp = (size_t)orc_obs_dim_pop(s), Dg = (size_t)orc_obs_dim_gov(s);
    for (int32_t k = 0; k < env_count; ++k) {
        const int32_t e = env_begin + k;
        step_env(s, &s->env[e], s->p.env_id_base + (uint32_t)e, actions + (size_t)k * N, gov_actions + (size_t)k * B,
                 obs_pop ? obs_pop + (size_t)k * N * Dp : NULL, obs_gov ? obs_gov + (size_t)k * Dg : NULL,
                 rew ? rew + (size_t)k * (N + 1) : NULL, done ? done + k : NULL);
    }
}

/* f4 (G44), the step of an auto-resetting rollout: the plain step; an env whose episode ends with it (done = 1)
 * then starts its next episode at once, and the observation returned for that step is the one of the fresh state
 * (the terminal observation is not returned: the caller's policy acts on what it is given next).  Rewards and done are
 * those of the step itself. */
void orc_step_auto(orc_sim* s, int32_t env_begin, int32_t env_count, const int32_t* actions,
                   const int32_t* gov_actions, float* obs_pop, float* obs_gov, float* rew, uint8_t* done) {
    const size_t N = (size_t)s->N, B = (size_t)s->p.num_brackets;
    const size_t Dp = (size_t)orc_obs_dim_pop(s), Dg = (size_t)orc_obs_dim_gov(s);
    for (int32_t k = 0; k < env_count; ++k) {
        const int32_t e = env_begin + k;
        orc_env* v = &s->env[e];
        uint8_t d = 0;
        float* op = obs_pop ? obs_pop + (size_t)k * N * Dp : NULL;
        float* og = obs_gov ? obs_gov + (size_t)k * Dg : NULL;
        step_env(s, v, s->p.env_id_base + (uint32_t)e, actions + (size_t)k * N, gov_actions + (size_t)k * B, op, og,
                 rew ? rew + (size_t)k * (N + 1) : NULL, &d);
        if (done) done[k] = d;
        if (d) {
            orc_begin_episode(s, e, 1, v->episode + 1);
            if (op || og) build_obs(s, v, 0, op, og);
        }
    }
}

/* f3 (G41): one correctly rounded binary32 operation per step of the formula. */
float orc_progress_skill(float skill, float rate, float max) {
    const float frac = skill / max;
    const float room = 1.0f - frac;
    const float g = rate * room;
    const float inc = skill * g;
    float out = skill + inc;
    if (out > max) out = max;
    return out;
}

/* f3 (G42): sum of twelve 24-bit uniforms minus 6 as the standard normal. */
float orc_normal_skill(const uint32_t words[12], float mean, float std, float lo, float hi) {
    int64_t sum = 0;
    for (int32_t k = 0; k < 12; ++k) sum += (int64_t)(words[k] >> 8);
    const double z = (double)sum * (1.0 / 16777216.0) - 6.0; /* exact: |sum - 6 * 2^24| < 2^27 */
    const double scaled = (double)std * z;                   /* exact: 24 x 27 significant bits */
    float x = (float)((double)mean + scaled);
    if (x < lo) x = lo;
    if (x > hi) x = hi;
    return x;
}

/* Rollout-mode action generator (G30): Philox stream 0 word 0 through the caller's CDF
 * table for the population; streams 1.. for the government's per-bracket levels. */
void orc_draw_actions(const orc_sim* s, int32_t env_begin, int32_t env_count, const uint32_t* cdf,
                      int32_t* actions, int32_t* gov_actions) {
    const int32_t N = s->N, B = s->p.num_brackets;
    const int32_t A = orc_num_actions(s->R, s->p.num_prices, s->p.craft_mode, s->p.allow_noop);
    for (int32_t k = 0; k < env_count; ++k) {
        const int32_t e = env_begin + k;
        const uint32_t gid = s->p.env_id_base + (uint32_t)e;
        const uint32_t t = (uint32_t)s->env[e].t;
        for (int32_t i = 0; i < N; ++i) {
            uint32_t x[4];
            draw(s, (uint32_t)s->env[e].episode, gid, (uint32_t)i, t, 0u, x);
            int32_t a = 0;
            while (a < A - 1 && !(x[0] < cdf[a])) ++a;
            actions[(size_t)k * N + i] = a;
        }
        for (int32_t b = 0; b < B; ++b) {
            uint32_t x[4];
            draw(s, (uint32_t)s->env[e].episode, gid, (uint32_t)N, t, (uint32_t)(1 + b / 4), x);
            gov_actions[(size_t)k * B + b] = (int32_t)(((uint64_t)x[b % 4] * (uint64_t)s->p.num_rate_levels) >> 32);
        }
    }
}

/* ---- canonical dump ---- */
static int32_t dump_cap(const orc_sim* s) { return s->N * s->p.max_active_orders; }

size_t orc_state_words(const orc_sim* s) {
    const size_t N = (size_t)s->N, R = (size_t)s->R, B = (size_t)s->p.num_brackets;
    return 13 + B + R + N * (6 + 3 * R) + 2 * R * (1 + 3 * (size_t)dump_cap(s)) + 1;  /* last word: episode (f4) */
}

static int32_t f2w(float f) { int32_t w; memcpy(&w, &f, 4); return w; }

void orc_get_state(const orc_sim* s, int32_t env_begin, int32_t env_count, int32_t* words) {
    const int32_t N = s->N, R = s->R, B = s->p.num_brackets, cap = dump_cap(s);
    const size_t W = orc_state_words(s);
    for (int32_t k = 0; k < env_count; ++k) {
        const orc_env* v = &s->env[env_begin + k];
        int32_t* w = words + (size_t)k * W;
        memset(w, 0, W * sizeof(int32_t));
        size_t q = 0;
        w[q++] = v->t; w[q++] = N; w[q++] = R; w[q++] = B; w[q++] = s->p.num_prices; w[q++] = cap;
        w[q++] = v->n_trades; w[q++] = v->n_placed; w[q++] = v->n_invalid; w[q++] = v->n_expired; w[q++] = v->n_bad_gov;
        memcpy(&w[q], &v->u_g_prev, 8); q += 2;
        for (int32_t b = 0; b < B; ++b) w[q++] = f2w(v->rates[b]);
        for (int32_t r = 0; r < R; ++r) w[q++] = v->last_price[r];
        for (int32_t i = 0; i < N; ++i) {
            w[q++] = f2w(v->coin[i]); w[q++] = v->esc_coin[i]; w[q++] = f2w(v->SC[i]);
            w[q++] = f2w(v->labor[i]); w[q++] = f2w(v->income[i]); w[q++] = v->n_live[i];
            for (int32_t r = 0; r < R; ++r) w[q++] = v->inv[i * R + r];
            for (int32_t r = 0; r < R; ++r) w[q++] = v->esc_res[i * R + r];
            for (int32_t r = 0; r < R; ++r) w[q++] = f2w(v->SG[i * R + r]);
        }
        for (int32_t b = 0; b < 2 * R; ++b) {
            const orc_book* bk = &v->book[b];
            const int32_t side = b % 2;
            /* priority order: bids price descending, asks price ascending, then arrival (selection sort on a copy) */
            orc_order* c = (orc_order*)malloc(sizeof(orc_order) * (size_t)(bk->n > 0 ? bk->n : 1));
            memcpy(c, bk->o, sizeof(orc_order) * (size_t)bk->n);
            int32_t n = bk->n;
            w[q++] = n;
            size_t q0 = q;
            for (int32_t out = 0; out < bk->n; ++out) {
                int32_t best = 0;
                for (int32_t i = 1; i < n; ++i) {
                    int better = side == 0 ? (c[i].price > c[best].price) : (c[i].price < c[best].price);
                    if (better || (c[i].price == c[best].price && arrived_after(&c[best], &c[i]))) best = i;
                }
                if (out < cap) { w[q0 + 3 * out] = c[best].price; w[q0 + 3 * out + 1] = c[best].owner; w[q0 + 3 * out + 2] = c[best].placed_at; }
                remove_order(c, &n, best);
            }
            free(c);
            q = q0 + 3 * (size_t)cap;
        }
        w[q++] = v->episode;
    }
}

void orc_set_agent(orc_sim* s, int32_t env, int32_t agent, float coin, const int32_t* inv,
                   const float* SG, float SC) {
    orc_env* v = &s->env[env];
    v->coin[agent] = coin;
    for (int32_t r = 0; r < s->R; ++r) {
        if (inv) v->inv[agent * s->R + r] = inv[r];
        if (SG) v->SG[agent * s->R + r] = SG[r];
    }
    v->SC[agent] = SC;
    v->u_g_prev = env_welfare(s, v);
}

void orc_set_rates(orc_sim* s, int32_t env, const float* rates) {
    for (int32_t b = 0; b < s->p.num_brackets; ++b) s->env[env].rates[b] = rates[b];
}

float orc_get_agent_f(const orc_sim* s, int32_t env, int32_t agent, int32_t what) {
    const orc_env* v = &s->env[env];
    return what == 0 ? v->coin[agent] : what == 1 ? v->labor[agent] : v->income[agent];
}

/* f1: action mask ("unavailable actions ... zero probability"; the availability
 * rules are P:199 "cannot sell a resource it does not have" plus the action preconditions of
 * P:145-168 and the order cap P:277).  Plain definition, one action at a time:
 *   gather r            always available
 *   craft               #{r : inv[r] >= R_kappa} >= R_d  (PER_RESOURCE r: inv[r] >= R_kappa)
 *   buy (r, price)      coin >= price  and  live orders < M
 *   sell (r, price)     inv[r] >= 1    and  live orders < M
 *   no-op               always available
 * The per-book cap K (G15) depends on the arrival order of the step and is not part of the mask.
 * Writes A bytes (0 / 1) per agent: mask[env_count][N][A]. */
void orc_action_mask(const orc_sim* s, int32_t env_begin, int32_t env_count, uint8_t* mask) {
    const orc_params* p = &s->p;
    const int32_t N = s->N, R = s->R, P = p->num_prices;
    const int32_t n_craft = (p->craft_mode == ORC_CRAFT_PER_RESOURCE) ? R : 1;
    const int32_t base_buy = R + n_craft, base_sell = base_buy + R * P;
    const int32_t A = orc_num_actions(R, P, p->craft_mode, p->allow_noop);
    for (int32_t k = 0; k < env_count; ++k) {
        const orc_env* v = &s->env[env_begin + k];
        for (int32_t i = 0; i < N; ++i) {
            uint8_t* m = mask + ((size_t)k * N + i) * A;
            const int32_t room = v->n_live[i] < p->max_active_orders;
            for (int32_t a = 0; a < A; ++a) {
                int32_t ok;
                if (a < R) {
                    ok = 1;
                } else if (a < base_buy) {
                    if (p->craft_mode == ORC_CRAFT_PER_RESOURCE) {
                        ok = v->inv[i * R + (a - R)] >= p->craft_units;
                    } else {
                        int32_t enough = 0;
                        for (int32_t r = 0; r < R; ++r) enough += v->inv[i * R + r] >= p->craft_units;
                        ok = enough >= p->craft_distinct;
                    }
                } else if (a < base_sell) {
                    ok = room && v->coin[i] >= (float)p->prices[(a - base_buy) % P];
                } else if (a < base_sell + R * P) {
                    ok = room && v->inv[i * R + (a - base_sell) / P] >= 1;
                } else {
                    ok = 1;
                }
                m[a] = (uint8_t)ok;
            }
        }
    }
}

/* f1, masked sampling (the policy's categorical gives zero probability to
 * unavailable actions): the rollout-mode generator restricted to the available actions of the
 * current state and renormalised.  With the caller's table, action a has integer weight
 * w_a = cdf[a] - cdf[a-1] (cdf[-1] = 0, the last entry read as 2^32, as in orc_draw_actions);
 * S = sum of w_a over available a;  target = floor(x0 * S / 2^32) with x0 = Philox stream 0
 * word 0;  action = first available a whose running sum of available weights exceeds target.
 * All integers, so the draw is exact.  With every action available S = 2^32, target = x0 and
 * the rule is orc_draw_actions'.  If S = 0 (the table gives the available actions no mass) the
 * first available action is returned.  Government levels are not masked. */
void orc_draw_actions_masked(const orc_sim* s, int32_t env_begin, int32_t env_count, const uint32_t* cdf,
                             int32_t* actions, int32_t* gov_actions) {
    const int32_t N = s->N;
    const int32_t A = orc_num_actions(s->R, s->p.num_prices, s->p.craft_mode, s->p.allow_noop);
    uint8_t* mask = (uint8_t*)malloc((size_t)N * A);
    orc_draw_actions(s, env_begin, env_count, cdf, actions, gov_actions);  /* government part; population overwritten */
    for (int32_t k = 0; k < env_count; ++k) {
        const int32_t e = env_begin + k;
        const uint32_t gid = s->p.env_id_base + (uint32_t)e;
        const uint32_t t = (uint32_t)s->env[e].t;
        orc_action_mask(s, e, 1, mask);
        for (int32_t i = 0; i < N; ++i) {
            uint32_t x[4];
            draw(s, (uint32_t)s->env[e].episode, gid, (uint32_t)i, t, 0u, x);
            uint64_t S = 0;
            for (int32_t a = 0; a < A; ++a) {
                const uint64_t hi = (a == A - 1) ? ((uint64_t)1 << 32) : (uint64_t)cdf[a];
                const uint64_t lo = (a == 0) ? 0 : (uint64_t)cdf[a - 1];
                if (mask[(size_t)i * A + a]) S += hi - lo;
            }
            const uint64_t target = ((uint64_t)x[0] * S) >> 32;  /* S <= 2^32: the product fits 64 bits */
            int32_t pick = -1, first = -1;
            uint64_t run = 0;
            for (int32_t a = 0; a < A && pick < 0; ++a) {
                if (!mask[(size_t)i * A + a]) continue;
                if (first < 0) first = a;
                const uint64_t hi = (a == A - 1) ? ((uint64_t)1 << 32) : (uint64_t)cdf[a];
                const uint64_t lo = (a == 0) ? 0 : (uint64_t)cdf[a - 1];
                run += hi - lo;
                if (run > target) pick = a;
            }
            actions[(size_t)k * N + i] = pick >= 0 ? pick : first;
        }
    }
    free(mask);
}
