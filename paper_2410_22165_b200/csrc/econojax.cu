// econojax.cu -- sm_100a kernels and C ABI of the batched EconoJax environment step.
//
// One CTA per economy; thread i is population agent i.  The whole state of an economy (agent
// arrays, per-level FIFO order books, order pool) is one contiguous "blob" that is copied into
// shared memory at kernel start and written back at kernel end; ej_rollout keeps it there for
// T steps.  Citations: "P:n" = PAPER.md line n, "G#" = DESIGN.md section 3 readings.
//
// Arithmetic contract (G31): agent state is binary32 and every state-changing float operation
// is ONE correctly rounded operation (__fadd_rn / __fmul_rn / __fsub_rn / __fdiv_rn: never
// contracted to FMA); cross-agent accumulations are integers (order-free, atomics allowed);
// rewards and statistics are evaluated in binary64.
//
// Order book: every (resource, side, price) level is a FIFO in arrival order
// because the price grid is discrete and an older step always precedes a newer one (G11), so
// both kinds of removal -- matching (best price first, then earliest arrival) and
// expiry (oldest first) -- pop queue heads.  Levels are singly linked lists threaded
// through a pool in which agent i owns slots [i*Mp, i*Mp+M): an agent places at most one order
// per step and holds at most M, so slot allocation is a private bitmask operation.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <type_traits>
#include <vector>

#include "../../include/econojax.h"

namespace {

constexpr uint32_t NIL = 0xFFFFu;

struct EnvHdr {
    int32_t t;
    int32_t n_trades, n_placed, n_invalid, n_expired, n_bad_gov;
    int32_t pad0[2];
    double u_g_prev;
    double pad1;
    float rates[EJ_MAX_BRACKETS];
    int32_t last_price[EJ_MAX_RESOURCES];
};
static_assert(sizeof(EnvHdr) % 16 == 0, "EnvHdr must keep 16-byte alignment");

struct DevCfg {
    int E, N, R, P, B, L, M, Mp_log2, K, T, period, expiry;
    int craft_units, craft_distinct, craft_mode, allow_noop, taxes_enabled, skill_init;
    int A, base_craft, base_buy, base_sell, n_levels, n_groups, D_pop, D_gov, D_gov_pad;
    int N4, Npad, n_metrics, n_warps, shrow_len, stage_obs;
    int prices[EJ_MAX_PRICES];
    float thresholds[EJ_MAX_BRACKETS];
    float rate_table[EJ_MAX_RATE_LEVELS];
    float starting_coin, labor_craft, labor_gather, labor_trade, eta, omega, craft_scale;
    float clip_lo, clip_hi, s_coin, s_count, s_price, s_labor;
    uint32_t env_id_base, seed_lo, seed_hi;
    // blob section offsets (bytes from the blob base)
    int o_coin, o_labor, o_income, o_SC, o_esc_coin, o_mask, o_cf, o_SG, o_inv, o_esc_res;
    int o_head, o_tail, o_cnt, o_pool, blob_bytes;
    // scratch section offsets (bytes from the shared-memory base; all after the blob)
    int o_key, o_cinfo, o_cslot, o_credit, o_sale, o_mb, o_ma, o_bucket, o_sorted;
    int o_gcnt, o_goff, o_take, o_roff, o_resq, o_resoff, o_red, o_redq, o_hist, o_hovf, o_stage, o_sortbuf, o_shrow, o_med, o_misc, o_cdf;
    int smem_bytes;
    unsigned long long gov_obs_offset, obs_floats;
};

struct StepIO {
    const int32_t* actions;      // [n_steps][E][N] or null (generate)
    const int32_t* gov_actions;  // [n_steps][E][B] or null (generate)
    float* obs;                  // ring of obs buffers or null
    float* rew;                  // ring [E][N+1] or null
    uint8_t* done;               // ring [E] or null
    int32_t* actions_out;        // ring [E][N] or null
    int32_t* gov_out;            // ring [E][B] or null
    const uint32_t* cdf;         // [A] device
    int n_steps, ring_depth;
};

struct Sm {
    EnvHdr* hdr;
    float *coin, *labor, *income, *SC;
    int* esc_coin;
    uint32_t* mask;
    double* cf;
    float* SG;
    int *inv, *esc_res;
    uint16_t *head, *tail;
    int* cnt;
    uint32_t* pool;
    uint32_t* key;
    int* cinfo;
    uint32_t* cslot;
    int *credit, *sale;
    uint32_t *mb, *ma;
    unsigned long long* bucket;
    uint32_t* sorted;
    int *gcnt, *goff, *take, *roff, *resq, *resoff;
    double* red;
    float* redq;
    int *hist, *hovf;
    float *stage, *sortbuf, *shrow, *med;
    unsigned long long* misc;  // [0] tax pool (2^-20 coin), [1] as int: total trades of the step
    uint32_t* cdf;
};

__device__ __forceinline__ Sm carve(const DevCfg& c, uint8_t* s) {
    Sm m;
    m.hdr = (EnvHdr*)s;
    m.coin = (float*)(s + c.o_coin);
    m.labor = (float*)(s + c.o_labor);
    m.income = (float*)(s + c.o_income);
    m.SC = (float*)(s + c.o_SC);
    m.esc_coin = (int*)(s + c.o_esc_coin);
    m.mask = (uint32_t*)(s + c.o_mask);
    m.cf = (double*)(s + c.o_cf);
    m.SG = (float*)(s + c.o_SG);
    m.inv = (int*)(s + c.o_inv);
    m.esc_res = (int*)(s + c.o_esc_res);
    m.head = (uint16_t*)(s + c.o_head);
    m.tail = (uint16_t*)(s + c.o_tail);
    m.cnt = (int*)(s + c.o_cnt);
    m.pool = (uint32_t*)(s + c.o_pool);
    m.key = (uint32_t*)(s + c.o_key);
    m.cinfo = (int*)(s + c.o_cinfo);
    m.cslot = (uint32_t*)(s + c.o_cslot);
    m.credit = (int*)(s + c.o_credit);
    m.sale = (int*)(s + c.o_sale);
    m.mb = (uint32_t*)(s + c.o_mb);
    m.ma = (uint32_t*)(s + c.o_ma);
    m.bucket = (unsigned long long*)(s + c.o_bucket);
    m.sorted = (uint32_t*)(s + c.o_sorted);
    m.gcnt = (int*)(s + c.o_gcnt);
    m.goff = (int*)(s + c.o_goff);
    m.take = (int*)(s + c.o_take);
    m.roff = (int*)(s + c.o_roff);
    m.resq = (int*)(s + c.o_resq);
    m.resoff = (int*)(s + c.o_resoff);
    m.red = (double*)(s + c.o_red);
    m.redq = (float*)(s + c.o_redq);
    m.hist = (int*)(s + c.o_hist);
    m.hovf = (int*)(s + c.o_hovf);
    m.stage = (float*)(s + c.o_stage);
    m.sortbuf = (float*)(s + c.o_sortbuf);
    m.shrow = (float*)(s + c.o_shrow);
    m.med = (float*)(s + c.o_med);
    m.misc = (unsigned long long*)(s + c.o_misc);
    m.cdf = (uint32_t*)(s + c.o_cdf);
    return m;
}

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), G30.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t& o0, uint32_t& o1, uint32_t& o2, uint32_t& o3) {
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

__device__ __forceinline__ float u01(uint32_t x) { return (float)(x >> 8) * (1.0f / 16777216.0f); }

// Coin term of Eq.1: (C^(1-eta) - 1) / (1-eta), binary64.
__device__ __forceinline__ double coin_utility(float C, double a) { return (pow((double)C, a) - 1.0) / a; }

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = __fadd_rn(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// Block-wide bitonic sort network, NV values per thread sorted independently (ascending by
// thread index), fully unrolled: strides below 32 are warp shuffles, larger ones go through a
// double-buffered shared array (one barrier per such stage).
template <int NPAD, int NV>
__device__ __forceinline__ void block_sort(float (&x)[NV], int tid, float* buf) {
    int pb = 0;
#pragma unroll
    for (int k = 2; k <= NPAD; k <<= 1) {
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
            float y[NV];
            if (j >= 32) {
                float* b = buf + pb * (NV * NPAD);
#pragma unroll
                for (int v = 0; v < NV; ++v) b[v * NPAD + tid] = x[v];
                __syncthreads();
#pragma unroll
                for (int v = 0; v < NV; ++v) y[v] = b[v * NPAD + (tid ^ j)];
                pb ^= 1;
            } else {
#pragma unroll
                for (int v = 0; v < NV; ++v) y[v] = __shfl_xor_sync(0xffffffffu, x[v], j);
            }
            const bool keep_min = ((tid & k) == 0) == ((tid & j) == 0);
#pragma unroll
            for (int v = 0; v < NV; ++v) x[v] = keep_min ? fminf(x[v], y[v]) : fmaxf(x[v], y[v]);
        }
    }
}

constexpr int HB = 128;  // histogram bins of the integer-metric medians (inventories)

// Government statistics (mean, std, median of coin, labor, income, inv[r]; Fig.1 P:31, P:426,
// G26), welfare (Eq.3-5, G22/G23), population rewards (Eq.1-2) and both
// observation blocks (G25, G27) of the state currently in shared memory.
//   tq       clock shown by the timers
//   mode     0 = step (rewards from pre-step values, update u_g_prev), 1 = finished env
//            (rewards 0), 2 = observe only (no rewards, u_g_prev untouched)
// Float metrics: sums in binary64 (warp shuffles), squared deviations in binary32 (a sum of
// non-negative terms: relative error < 1e-6), medians and the gini numerator from one
// three-value sorting network.  Integer metrics: exact integer sums (REDUX), medians from a
// shared-memory histogram (values >= HB fall back to the sorting network).
template <int NPAD>
__device__ void stats_rewards_obs(const DevCfg& c, const Sm& m, int tid, int e, int tq, int mode, float coin_pre,
                                  float labor_pre, double cf_pre, float* obs, float* rew) {
    constexpr int NW = NPAD / 32;
    const int N = c.N, R = c.R, nm = c.n_metrics, N4 = c.N4;
    const bool act = tid < N;
    const int lane = tid & 31, warp = tid >> 5;
    const double inv_n = 1.0 / (double)N;

    float xf[3] = {0.f, 0.f, 0.f};
    if (act) { xf[0] = m.coin[tid]; xf[1] = m.labor[tid]; xf[2] = m.income[tid]; }

    // ---- population reward: u(post) - u(pre), u = coin term - labor (Eq.1-2) ----
    if (mode == 0 && act) {
        double cf_post = cf_pre;
        if (__float_as_uint(xf[0]) != __float_as_uint(coin_pre)) {
            cf_post = coin_utility(xf[0], 1.0 - (double)c.eta);
            m.cf[tid] = cf_post;
        }
        const double u_post = cf_post - (double)xf[1];
        const double u_pre = cf_pre - (double)labor_pre;
        if (rew) rew[(size_t)e * (N + 1) + tid] = (float)(u_post - u_pre);
    } else if (mode == 1 && act && rew) {
        rew[(size_t)e * (N + 1) + tid] = 0.0f;
    }

    // ---- pass 1: sums (per-warp partials), histograms of the integer metrics ----
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double s = warp_sum((double)xf[k]);
        if (lane == 0) m.red[k * NW + warp] = s;
    }
    for (int r = 0; r < R; ++r) {
        const int v = act ? m.inv[r * N4 + tid] : 0;
        const int s = __reduce_add_sync(0xffffffffu, v);
        if (lane == 0) m.red[(3 + r) * NW + warp] = (double)s;
        if (act) {
            if (v < HB) atomicAdd(&m.hist[r * HB + v], 1);
            else m.hovf[r] = 1;
        }
    }
    // shared tail of the population rows: market statistics, rates, timers
    if (tid < R) {
        const int r = tid;
        int best_bid = 0, best_ask = 0, nb = 0, na = 0;
        for (int p = 0; p < c.P; ++p) {
            const int cb = m.cnt[(r * 2 + 0) * c.P + p], ca = m.cnt[(r * 2 + 1) * c.P + p];
            nb += cb;
            na += ca;
            if (cb > 0) best_bid = c.prices[p];
            if (ca > 0 && best_ask == 0) best_ask = c.prices[p];
        }
        float* o = m.shrow + r * 5;
        o[0] = __fmul_rn((float)best_bid, c.s_price);
        o[1] = __fmul_rn((float)best_ask, c.s_price);
        o[2] = __fmul_rn((float)nb, c.s_count);
        o[3] = __fmul_rn((float)na, c.s_count);
        o[4] = __fmul_rn((float)m.hdr->last_price[r], c.s_price);
    }
    if (tid >= 32 && tid < 32 + c.B) m.shrow[5 * R + tid - 32] = m.hdr->rates[tid - 32];
    if (NPAD == 32 && tid < c.B) m.shrow[5 * R + tid] = m.hdr->rates[tid];
    if (tid == NPAD - 1) {
        m.shrow[5 * R + c.B] = __fdiv_rn((float)(tq % c.period), (float)c.period);
        m.shrow[5 * R + c.B + 1] = __fdiv_rn((float)tq, (float)c.T);
    }
    // private part of the population rows, staged in shared memory
    const bool staged = c.stage_obs && obs;
    if (staged) {
        if (act) {
            float* o = m.stage + tid * c.D_pop;
            int k = 0;
            o[k++] = __fmul_rn(xf[0], c.s_coin);
            for (int r = 0; r < R; ++r) o[k++] = __fmul_rn((float)m.inv[r * N4 + tid], c.s_count);
            o[k++] = __fmul_rn((float)m.esc_coin[tid], c.s_coin);
            for (int r = 0; r < R; ++r) o[k++] = __fmul_rn((float)m.esc_res[r * N4 + tid], c.s_count);
            for (int r = 0; r < R; ++r) o[k++] = m.SG[r * N4 + tid];
            o[k++] = m.SC[tid];
            o[k++] = __fmul_rn(xf[1], c.s_labor);
        }
    }
    __syncthreads();

    // ---- pass 2: means, squared deviations, sort, medians, gini numerator ----
    // every warp redundantly reduces the per-warp partials: lane k owns metric k
    double mean_l = 0.0;
    if (lane < nm) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < NW; ++w) s += m.red[lane * NW + w];
        mean_l = s * inv_n;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double mean = __shfl_sync(0xffffffffu, mean_l, k);
        const float d = act ? (float)((double)xf[k] - mean) : 0.0f;
        const float q = warp_sum(__fmul_rn(d, d));
        if (lane == 0) m.redq[k * NW + warp] = q;
    }
    for (int r = 0; r < R; ++r) {
        const double mean = __shfl_sync(0xffffffffu, mean_l, 3 + r);
        const float d = act ? (float)((double)m.inv[r * N4 + tid] - mean) : 0.0f;
        const float q = warp_sum(__fmul_rn(d, d));
        if (lane == 0) m.redq[(3 + r) * NW + warp] = q;
    }
    if (staged && act) {  // shared tail of this agent's row
        float* o = m.stage + tid * c.D_pop + (3 * R + 4);
        for (int k = 0; k < c.shrow_len; ++k) o[k] = m.shrow[k];
    }
    {
        float xs[3] = {act ? xf[0] : INFINITY, act ? xf[1] : INFINITY, act ? xf[2] : INFINITY};
        block_sort<NPAD, 3>(xs, tid, m.sortbuf);
        if (tid == (N >> 1) - 1) { m.med[0] = xs[0]; m.med[2] = xs[1]; m.med[4] = xs[2]; }
        if (tid == (N >> 1)) { m.med[1] = xs[0]; m.med[3] = xs[1]; m.med[5] = xs[2]; }
        // sum_i sum_j |c_i - c_j| = 2 sum_k (2k - N + 1) c_(k)   (G23)
        const double g = act ? (double)(2 * tid - N + 1) * (double)xs[0] : 0.0;
        const double gs = warp_sum(g);
        if (lane == 0) m.red[nm * NW + warp] = gs;
    }
    for (int r = 0; r < R; ++r) {  // rare: an inventory >= HB, median from the sorting network
        if (m.hovf[r]) {
            float xs[1] = {act ? (float)m.inv[r * N4 + tid] : INFINITY};
            block_sort<NPAD, 1>(xs, tid, m.sortbuf);
            if (tid == (N >> 1) - 1) m.med[2 * (3 + r)] = xs[0];
            if (tid == (N >> 1)) m.med[2 * (3 + r) + 1] = xs[0];
        }
    }
    if (staged) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    // ---- finals ----
    float* gov = obs ? obs + c.gov_obs_offset + (size_t)e * c.D_gov_pad : nullptr;
    if (staged && tid == 0) {  // one bulk store of the env's contiguous [N][D_pop] block
        float* dst = obs + (size_t)e * N * c.D_pop;
        const uint32_t src = (uint32_t)__cvta_generic_to_shared(m.stage);
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(N * c.D_pop * 4) : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    // integer medians from the histograms: warp w handles metrics w, w + NW, ...
    for (int r = warp; r < R; r += NW) {
        float lo_v, hi_v;
        if (!m.hovf[r]) {
            int4 h4 = ((int4*)(m.hist + r * HB))[lane];
            ((int4*)(m.hist + r * HB))[lane] = make_int4(0, 0, 0, 0);
            const int c0 = h4.x, c1 = c0 + h4.y, c2 = c1 + h4.z, c3 = c2 + h4.w;
            int incl = c3;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += y;
            }
            const int excl = incl - c3;
            int vals[2];
#pragma unroll
            for (int j = 0; j < 2; ++j) {  // value of 0-based rank q = smallest v with cum(v) > q
                const int q = (N >> 1) - 1 + j;
                const unsigned ball = __ballot_sync(0xffffffffu, incl > q);
                const int src = __ffs(ball) - 1;
                const int ex = __shfl_sync(0xffffffffu, excl, src < 0 ? 0 : src);
                const int a0 = __shfl_sync(0xffffffffu, c0, src < 0 ? 0 : src), a1 = __shfl_sync(0xffffffffu, c1, src < 0 ? 0 : src),
                          a2 = __shfl_sync(0xffffffffu, c2, src < 0 ? 0 : src);
                const int rel = q - ex;
                vals[j] = (src < 0 ? 0 : src) * 4 + (rel < a0 ? 0 : rel < a1 ? 1 : rel < a2 ? 2 : 3);
            }
            lo_v = (float)vals[0];
            hi_v = (float)vals[1];
        } else {
            for (int b = lane; b < HB; b += 32) m.hist[r * HB + b] = 0;
            lo_v = m.med[2 * (3 + r)];
            hi_v = m.med[2 * (3 + r) + 1];
            __syncwarp();
            if (lane == 0) m.hovf[r] = 0;
        }
        if (lane == 0) {
            const int k = 3 + r;
            double s1 = 0.0;
            float s2 = 0.0f;
            for (int w = 0; w < NW; ++w) s1 += m.red[k * NW + w];
            for (int w = 0; w < NW; ++w) s2 = __fadd_rn(s2, m.redq[k * NW + w]);
            const double mean = s1 * inv_n;
            const double sd = sqrt((double)s2 * inv_n);
            const float med = (N & 1) ? hi_v : __fmul_rn(0.5f, __fadd_rn(lo_v, hi_v));
            if (gov) {
                gov[3 * k + 0] = (float)(mean * (double)c.s_count);
                gov[3 * k + 1] = (float)(sd * (double)c.s_count);
                gov[3 * k + 2] = __fmul_rn(med, c.s_count);
            }
        }
    }
    if (tid >= NPAD - 3) {  // float metrics: coin, labor, income
        const int k = tid - (NPAD - 3);
        double s1 = 0.0;
        float s2 = 0.0f;
        for (int w = 0; w < NW; ++w) s1 += m.red[k * NW + w];
        for (int w = 0; w < NW; ++w) s2 = __fadd_rn(s2, m.redq[k * NW + w]);
        const double mean = s1 * inv_n;
        const double sd = sqrt((double)s2 * inv_n);
        const float med = (N & 1) ? m.med[2 * k + 1] : __fmul_rn(0.5f, __fadd_rn(m.med[2 * k], m.med[2 * k + 1]));
        const float scale = k == 1 ? c.s_labor : c.s_coin;
        if (gov) {
            gov[3 * k + 0] = (float)(mean * (double)scale);
            gov[3 * k + 1] = (float)(sd * (double)scale);
            gov[3 * k + 2] = __fmul_rn(med, scale);
        }
    }
    if (gov)
        for (int k = tid; k < c.B + 2; k += NPAD) gov[3 * nm + k] = m.shrow[5 * R + k];
    if (tid == 0 && mode != 2) {
        double prod = 0.0, gn = 0.0;
        for (int w = 0; w < NW; ++w) prod += m.red[w];
        for (int w = 0; w < NW; ++w) gn += m.red[nm * NW + w];
        double gini = 0.0;
        if (N > 1 && prod != 0.0) gini = gn / ((double)N * prod);
        const double eq = (double)c.omega * (1.0 - gini) + (1.0 - (double)c.omega);
        const double ug = eq * prod;
        if (mode == 0) {
            if (rew) rew[(size_t)e * (N + 1) + N] = (float)(ug - m.hdr->u_g_prev);
            m.hdr->u_g_prev = ug;
        } else if (rew) {
            rew[(size_t)e * (N + 1) + N] = 0.0f;
        }
    }

    // ---- population rows when they cannot go out as one bulk store: coalesced loop ----
    if (obs && !staged) {
        const int D = c.D_pop, priv = 3 * R + 4, total = N * D;
        float* dst = obs + (size_t)e * total;
        for (int idx = tid; idx < total; idx += NPAD) {
            const int i = idx / D, k = idx - i * D;
            float v;
            if (k >= priv) v = m.shrow[k - priv];
            else if (k == 0) v = __fmul_rn(m.coin[i], c.s_coin);
            else if (k <= R) v = __fmul_rn((float)m.inv[(k - 1) * N4 + i], c.s_count);
            else if (k == R + 1) v = __fmul_rn((float)m.esc_coin[i], c.s_coin);
            else if (k <= 2 * R + 1) v = __fmul_rn((float)m.esc_res[(k - R - 2) * N4 + i], c.s_count);
            else if (k <= 3 * R + 1) v = m.SG[(k - 2 * R - 2) * N4 + i];
            else if (k == 3 * R + 2) v = m.SC[i];
            else v = __fmul_rn(m.labor[i], c.s_labor);
            dst[idx] = v;
        }
    }
}

// One environment step on the state in shared memory (G1: actions -> match -> expire -> tax ->
// rewards -> observations -> t++).
template <int NPAD>
__device__ void env_step(const DevCfg& c, const Sm& m, int tid, int e, const int32_t* actions, const int32_t* gov_actions,
                         float* obs, float* rew, uint8_t* done, int32_t* actions_out, int32_t* gov_out) {
    const int N = c.N, R = c.R, P = c.P, N4 = c.N4;
    const bool act = tid < N;
    const int t = m.hdr->t;
    const uint32_t gid = c.env_id_base + (uint32_t)e;
    // the previous step's bulk store must have read the staging tile before it is rewritten
    if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");

    if (t >= c.T) {  // G28: finished env
        __syncthreads();
        stats_rewards_obs<NPAD>(c, m, tid, e, t, 1, 0.f, 0.f, 0.0, obs, rew);
        if (tid == 0 && done) done[e] = 1;
        __syncthreads();
        return;
    }

    // ---------------- P1 actions (one action per agent per step) ----------------
    uint32_t x0 = 0, x1 = 0, x2 = 0, x3 = 0;
    int a = -1;
    if (act) {
        philox4x32_10(gid, (uint32_t)tid, (uint32_t)t, 0u, c.seed_lo, c.seed_hi, x0, x1, x2, x3);
        if (actions) {
            a = actions[(size_t)e * N + tid];
        } else {  // smallest a with x0 < cdf[a]; last entry read as 2^32 (G30)
            int lo = 0, hi = c.A - 1;
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (x0 < m.cdf[mid]) hi = mid;
                else lo = mid + 1;
            }
            a = lo;
        }
        if (actions_out) actions_out[(size_t)e * N + tid] = a;
        m.key[tid] = x2;
    }
    // government levels for the period boundary
    int gov_lvl = -1;
    if (tid < c.B) {
        if (gov_actions) {
            gov_lvl = gov_actions[(size_t)e * c.B + tid];
        } else {
            uint32_t g0, g1, g2, g3;
            philox4x32_10(gid, (uint32_t)N, (uint32_t)t, (uint32_t)(1 + tid / 4), c.seed_lo, c.seed_hi, g0, g1, g2, g3);
            const uint32_t gx = (tid & 3) == 0 ? g0 : (tid & 3) == 1 ? g1 : (tid & 3) == 2 ? g2 : g3;
            gov_lvl = (int)(((unsigned long long)gx * (unsigned long long)c.L) >> 32);
        }
        if (gov_out) gov_out[(size_t)e * c.B + tid] = gov_lvl;
    }

    float coin_pre = 0.f, labor_pre = 0.f;
    double cf_pre = 0.0;
    int lvl = -1, grp = 0, pos = 0, price_c = 0, r_c = 0, side_c = 0;
    uint32_t slot = 0, mymask = 0;
    if (act) {
        coin_pre = m.coin[tid];
        labor_pre = m.labor[tid];
        cf_pre = m.cf[tid];
        mymask = m.mask[tid];
        bool invalid = false;
        if (a < 0 || a >= c.A) {
            invalid = true;  // G2
        } else if (a < R) {  // gather: floor(SG + rho), rho = u * 1.1 (G8)
            const float rho = __fmul_rn(u01(x1), 1.1f);
            const float s = __fadd_rn(m.SG[a * N4 + tid], rho);
            m.inv[a * N4 + tid] += (int)floorf(s);
            m.labor[tid] = __fadd_rn(labor_pre, c.labor_gather);
        } else if (a < c.base_buy) {  // craft
            bool ok;
            if (c.craft_mode == EJ_CRAFT_PER_RESOURCE) {
                const int r = a - R;
                ok = m.inv[r * N4 + tid] >= c.craft_units;
                if (ok) m.inv[r * N4 + tid] -= c.craft_units;
            } else {
                int enough = 0;
                for (int r = 0; r < R; ++r) enough += m.inv[r * N4 + tid] >= c.craft_units;
                ok = enough >= c.craft_distinct;
                if (ok) {  // the R_d most-held resources, ties to the lowest index (G7)
                    uint32_t used = 0;
                    for (int k = 0; k < c.craft_distinct; ++k) {
                        int best = -1, bestv = 0;
                        for (int r = 0; r < R; ++r) {
                            if ((used >> r) & 1u) continue;
                            const int v = m.inv[r * N4 + tid];
                            if (best < 0 || v > bestv) { best = r; bestv = v; }
                        }
                        used |= 1u << best;
                        m.inv[best * N4 + tid] = bestv - c.craft_units;
                    }
                }
            }
            if (ok) {
                const float pay = __fmul_rn(m.SC[tid], c.craft_scale);
                m.coin[tid] = __fadd_rn(coin_pre, pay);
                m.income[tid] = __fadd_rn(m.income[tid], pay);
                m.labor[tid] = __fadd_rn(labor_pre, c.labor_craft);
            } else {
                invalid = true;
            }
        } else if (a < c.base_sell + R * P) {  // market order
            side_c = a >= c.base_sell;
            const int k = a - (side_c ? c.base_sell : c.base_buy);
            r_c = k / P;
            const int pidx = k - r_c * P;
            price_c = c.prices[pidx];
            bool ok = __popc(mymask) < c.M;
            if (side_c == 0) ok = ok && (coin_pre >= (float)price_c);
            else ok = ok && (m.inv[r_c * N4 + tid] >= 1);
            if (ok) {
                lvl = (r_c * 2 + side_c) * P + pidx;
                grp = c.K ? (r_c * 2 + side_c) : lvl;
                slot = ((uint32_t)tid << c.Mp_log2) + (uint32_t)(__ffs(~mymask) - 1);
                m.cslot[tid] = slot;
                pos = atomicAdd(&m.gcnt[grp], 1);
            } else {
                invalid = true;
            }
        }  // else NO-OP
        m.cinfo[tid] = lvl;
        if (invalid) atomicAdd(&m.hdr->n_invalid, 1);
    }
    __syncthreads();  // #1 group counts complete

    // exclusive scan of the group counts (warp 0)
    if (tid < 32) {
        int carry = 0;
        for (int base = 0; base < c.n_groups; base += 32) {
            const int g = base + tid;
            const int v = g < c.n_groups ? m.gcnt[g] : 0;
            int incl = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, incl, o);
                if (tid >= o) incl += y;
            }
            if (g < c.n_groups) m.goff[g] = carry + incl - v;
            carry += __shfl_sync(0xffffffffu, incl, 31);
        }
    }
    __syncthreads();  // #2
    const unsigned long long mine = ((unsigned long long)x2 << 32) | (unsigned long long)tid;
    if (lvl >= 0) m.bucket[m.goff[grp] + pos] = mine;
    __syncthreads();  // #3 buckets complete

    // arrival order of this step's candidates: (key, agent) (G11); acceptance against the book
    // cap counted from the book size at step start (G15)
    int before = 0, lrank = 0, gbase = 0, gn = 0;
    bool accepted = false;
    uint32_t old_tail = NIL;
    if (lvl >= 0) {
        gbase = m.goff[grp];
        gn = m.gcnt[grp];
        if (c.K) {
            int brank = 0;
            for (int k = 0; k < gn; ++k) {
                const unsigned long long o = m.bucket[gbase + k];
                const int lj = m.cinfo[(int)(o & 0xFFFFFFFFu)];
                const bool earlier = o < mine, same = lj == lvl;
                brank += earlier;
                lrank += same && earlier;
                before += (lj < lvl) || (same && earlier);
            }
            int n_rest = 0;
            for (int p = 0; p < P; ++p) n_rest += m.cnt[grp * P + p];
            accepted = n_rest + brank < c.K;
        } else {
            for (int k = 0; k < gn; ++k) lrank += m.bucket[gbase + k] < mine;
            before = lrank;
            accepted = true;
        }
        old_tail = m.tail[lvl];
        m.sorted[gbase + before] = (uint32_t)tid | (accepted ? 0x10000u : 0u);
    }
    __syncthreads();  // #4 sorted complete

    if (lvl >= 0) {
        if (accepted) {
            uint32_t nxt = NIL;
            if (before + 1 < gn) {
                const uint32_t s = m.sorted[gbase + before + 1];
                const int j = (int)(s & 0xFFFFu);
                if ((s & 0x10000u) && m.cinfo[j] == lvl) nxt = m.cslot[j];
            }
            m.pool[slot] = nxt | (((uint32_t)t & 0xFFFFu) << 16);
            if (lrank == 0) {
                if (old_tail != NIL) m.pool[old_tail] = (m.pool[old_tail] & 0xFFFF0000u) | slot;
                else m.head[lvl] = (uint16_t)slot;
            }
            if (nxt == NIL) m.tail[lvl] = (uint16_t)slot;
            atomicAdd(&m.cnt[lvl], 1);
            m.mask[tid] = mymask | (1u << (slot & ((1u << c.Mp_log2) - 1u)));
            if (side_c == 0) {  // escrow
                m.coin[tid] = __fsub_rn(coin_pre, (float)price_c);
                m.esc_coin[tid] += price_c;
            } else {
                m.inv[r_c * N4 + tid] -= 1;
                m.esc_res[r_c * N4 + tid] += 1;
            }
            m.labor[tid] = __fadd_rn(labor_pre, c.labor_trade);
            atomicAdd(&m.hdr->n_placed, 1);
        } else {
            atomicAdd(&m.hdr->n_invalid, 1);
        }
    }
    __syncthreads();  // #5 books hold this step's arrivals

    // ---------------- P2 match: q = max_p min(#bids >= p, #asks <= p) ----------------
    if (tid < 32) {
        int q = 0;
        if (tid < R) {
            const int lb = (tid * 2 + 0) * P, la = (tid * 2 + 1) * P;
            int totB = 0;
            for (int p = 0; p < P; ++p) totB += m.cnt[lb + p];
            int ale = 0, prefB = 0;
            for (int p = 0; p < P; ++p) {
                ale += m.cnt[la + p];
                const int bge = totB - prefB;
                q = max(q, min(bge, ale));
                prefB += m.cnt[lb + p];
            }
            int rem = q;
            for (int p = P - 1; p >= 0; --p) {  // bids: highest price first
                const int tk = min(m.cnt[lb + p], rem);
                m.take[lb + p] = tk;
                m.roff[lb + p] = q - rem;
                rem -= tk;
            }
            rem = q;
            for (int p = 0; p < P; ++p) {  // asks: lowest price first
                const int tk = min(m.cnt[la + p], rem);
                m.take[la + p] = tk;
                m.roff[la + p] = q - rem;
                rem -= tk;
            }
            m.resq[tid] = q;
        }
        int incl = q;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, o);
            if (tid >= o) incl += y;
        }
        if (tid <= R) m.resoff[tid] = incl - q;  // resoff[R] = total (lanes >= R hold q = 0)
    }
    for (int g = tid; g < c.n_groups; g += NPAD) m.gcnt[g] = 0;  // ready for the next step
    __syncthreads();  // #6

    // pop matched heads, then expired heads (G14), one thread per level
    for (int l = tid; l < c.n_levels; l += NPAD) {
        const int book = l / P, pidx = l - book * P, r = book >> 1, side = book & 1;
        const int price = c.prices[pidx];
        const int tk = m.take[l];
        uint32_t h = m.head[l];
        int n = m.cnt[l];
        if (tk > 0) {
            uint32_t* dst = (side ? m.ma : m.mb) + m.resoff[r] + m.roff[l];
            for (int k = 0; k < tk; ++k) {
                dst[k] = h | ((uint32_t)pidx << 16);
                h = m.pool[h] & 0xFFFFu;
            }
            n -= tk;
        }
        int nexp = 0;
        while (h != NIL) {
            const uint32_t pe = m.pool[h];
            const uint32_t age = ((uint32_t)t - (pe >> 16)) & 0xFFFFu;
            if ((int)age < c.expiry) break;
            const int owner = (int)(h >> c.Mp_log2);
            if (side == 0) {
                atomicSub(&m.esc_coin[owner], price);
                atomicAdd(&m.credit[owner], price);
            } else {
                atomicSub(&m.esc_res[r * N4 + owner], 1);
                atomicAdd(&m.inv[r * N4 + owner], 1);
            }
            atomicAnd(&m.mask[owner], ~(1u << (h & ((1u << c.Mp_log2) - 1u))));
            ++nexp;
            --n;
            h = pe & 0xFFFFu;
        }
        if (tk > 0 || nexp > 0) {
            m.head[l] = (uint16_t)h;
            if (h == NIL) m.tail[l] = (uint16_t)NIL;
            m.cnt[l] = n;
            if (nexp) atomicAdd(&m.hdr->n_expired, nexp);
        }
    }
    __syncthreads();  // #7 matched lists complete

    // settle trade i: bid rank i with ask rank i, at the price of the later arrival
    {
        const int total = m.resoff[R];
        if (tid < total) {
            int r = 0;
            while (tid >= m.resoff[r + 1]) ++r;
            const uint32_t eb = m.mb[tid], ea = m.ma[tid];
            const uint32_t sb = eb & 0xFFFFu, sa = ea & 0xFFFFu;
            const int pb = c.prices[eb >> 16], pa = c.prices[ea >> 16];
            const int ob = (int)(sb >> c.Mp_log2), oa = (int)(sa >> c.Mp_log2);
            const uint32_t age_b = ((uint32_t)t - (m.pool[sb] >> 16)) & 0xFFFFu;
            const uint32_t age_a = ((uint32_t)t - (m.pool[sa] >> 16)) & 0xFFFFu;
            bool bid_later;
            if (age_b != age_a) bid_later = age_b < age_a;
            else if (m.key[ob] != m.key[oa]) bid_later = m.key[ob] > m.key[oa];
            else bid_later = ob > oa;
            const int pi = bid_later ? pb : pa;
            const uint32_t bitmask = (1u << c.Mp_log2) - 1u;
            atomicSub(&m.esc_coin[ob], pb);
            if (pb - pi) atomicAdd(&m.credit[ob], pb - pi);  // refund of the escrowed excess
            atomicAdd(&m.inv[r * N4 + ob], 1);
            atomicAnd(&m.mask[ob], ~(1u << (sb & bitmask)));
            atomicSub(&m.esc_res[r * N4 + oa], 1);
            atomicAdd(&m.credit[oa], pi);
            atomicAdd(&m.sale[oa], pi);
            atomicAnd(&m.mask[oa], ~(1u << (sa & bitmask)));
            if (tid == m.resoff[r + 1] - 1) m.hdr->last_price[r] = pi;
        }
        if (tid == 0) m.hdr->n_trades += total;
    }
    __syncthreads();  // #8 credits complete

    // income from sales (G16), coin credit once per agent
    const bool boundary = c.taxes_enabled && ((t + 1) % c.period == 0);
    if (act) {
        const int sl = m.sale[tid], cr = m.credit[tid];
        if (sl > 0) { m.income[tid] = __fadd_rn(m.income[tid], (float)sl); m.sale[tid] = 0; }
        if (cr > 0) { m.coin[tid] = __fadd_rn(m.coin[tid], (float)cr); m.credit[tid] = 0; }
    }

    // ---------------- P4 tax at period end (G17-G20) ----------------
    if (boundary) {
        long long fx = 0;
        if (act) {
            const float income = m.income[tid];
            float tax = 0.0f, lo = 0.0f;
            for (int b = 0; b < c.B; ++b) {
                const float hi = (b < c.B - 1) ? c.thresholds[b] : INFINITY;
                const float top = (income < hi) ? income : hi;
                float por = __fsub_rn(top, lo);
                if (por < 0.0f) por = 0.0f;
                tax = __fadd_rn(tax, __fmul_rn(m.hdr->rates[b], por));
                lo = hi;
            }
            const float coin = m.coin[tid];
            if (tax > coin) tax = coin;  // G17
            m.coin[tid] = __fsub_rn(coin, tax);
            fx = __double2ll_rn((double)tax * 1048576.0);  // G19
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) fx += __shfl_xor_sync(0xffffffffu, fx, o);
        if ((tid & 31) == 0 && fx != 0) atomicAdd(&m.misc[0], (unsigned long long)fx);
        __syncthreads();
        if (act) {
            const float pool = __double2float_rn((double)(long long)m.misc[0] * (1.0 / 1048576.0));
            const float share = __fdiv_rn(pool, (float)N);  // P:195 "(1/n)"
            m.coin[tid] = __fadd_rn(m.coin[tid], share);
            m.income[tid] = 0.0f;
        }
        if (tid < c.B) {  // rates of the upcoming period
            if (gov_lvl < 0 || gov_lvl >= c.L) atomicAdd(&m.hdr->n_bad_gov, 1);
            else m.hdr->rates[tid] = c.rate_table[gov_lvl];
        }
        __syncthreads();
        if (tid == 0) m.misc[0] = 0ull;
    } else {
        __syncthreads();
    }

    // ---------------- P5 rewards, P6 observations, clock ----------------
    stats_rewards_obs<NPAD>(c, m, tid, e, t + 1, 0, coin_pre, labor_pre, cf_pre, obs, rew);
    if (tid == 0) {
        m.hdr->t = t + 1;
        if (done) done[e] = (uint8_t)(t + 1 == c.T);
    }
    __syncthreads();
}

template <int NPAD>
__global__ void __launch_bounds__(NPAD) ej_step_kernel(const __grid_constant__ DevCfg c, uint8_t* __restrict__ state,
                                                       const StepIO io) {
    extern __shared__ __align__(16) uint8_t smem[];
    const int e = blockIdx.x, tid = threadIdx.x;
    const Sm m = carve(c, smem);
    uint4* blob = (uint4*)(state + (size_t)e * c.blob_bytes);
    for (int i = tid; i < c.blob_bytes / 16; i += NPAD) ((uint4*)smem)[i] = blob[i];
    for (int i = tid; i < (c.smem_bytes - c.blob_bytes) / 4; i += NPAD) ((uint32_t*)(smem + c.blob_bytes))[i] = 0u;
    __syncthreads();
    if (!io.actions)
        for (int i = tid; i < c.A; i += NPAD) m.cdf[i] = io.cdf[i];
    __syncthreads();
    const size_t EN = (size_t)c.E * c.N, EB = (size_t)c.E * c.B;
    for (int s = 0; s < io.n_steps; ++s) {
        const int slot = s % io.ring_depth;
        env_step<NPAD>(c, m, tid, e, io.actions ? io.actions + s * EN : nullptr, io.gov_actions ? io.gov_actions + s * EB : nullptr,
                 io.obs ? io.obs + (size_t)slot * c.obs_floats : nullptr, io.rew ? io.rew + (size_t)slot * (EN + c.E) : nullptr,
                 io.done ? io.done + (size_t)slot * c.E : nullptr, io.actions_out ? io.actions_out + slot * EN : nullptr,
                 io.gov_out ? io.gov_out + slot * EB : nullptr);
    }
    __syncthreads();
    for (int i = tid; i < c.blob_bytes / 16; i += NPAD) blob[i] = ((uint4*)smem)[i];
    if (tid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

template <int NPAD>
__global__ void __launch_bounds__(NPAD) ej_observe_kernel(const __grid_constant__ DevCfg c, const uint8_t* __restrict__ state,
                                                          float* obs) {
    extern __shared__ __align__(16) uint8_t smem[];
    const int e = blockIdx.x, tid = threadIdx.x;
    const Sm m = carve(c, smem);
    const uint4* blob = (const uint4*)(state + (size_t)e * c.blob_bytes);
    for (int i = tid; i < c.blob_bytes / 16; i += NPAD) ((uint4*)smem)[i] = blob[i];
    __syncthreads();
    for (int i = tid; i < (c.smem_bytes - c.blob_bytes) / 4; i += NPAD) ((uint32_t*)(smem + c.blob_bytes))[i] = 0u;
    __syncthreads();
    stats_rewards_obs<NPAD>(c, m, tid, e, m.hdr->t, 2, 0.f, 0.f, 0.0, obs, nullptr);
    if (tid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// Reset (G29, G30): one CTA per env builds the blob in shared memory and stores it.
template <int NPAD>
__global__ void __launch_bounds__(NPAD) ej_reset_kernel(const __grid_constant__ DevCfg c, uint8_t* __restrict__ state) {
    extern __shared__ __align__(16) uint8_t smem[];
    const int e = blockIdx.x, tid = threadIdx.x;
    const Sm m = carve(c, smem);
    for (int i = tid; i < c.blob_bytes / 4; i += NPAD) ((uint32_t*)smem)[i] = 0u;
    __syncthreads();
    const uint32_t gid = c.env_id_base + (uint32_t)e;
    if (tid < c.N) {
        m.coin[tid] = c.starting_coin;
        m.cf[tid] = coin_utility(c.starting_coin, 1.0 - (double)c.eta);
        uint32_t x[4] = {0, 0, 0, 0};
        for (int d = 0; d <= c.R; ++d) {  // skill draw d: Philox stream 16, "t" field d/4, word d%4
            if ((d & 3) == 0) philox4x32_10(gid, (uint32_t)tid, (uint32_t)(d >> 2), 16u, c.seed_lo, c.seed_hi, x[0], x[1], x[2], x[3]);
            const uint32_t w = (d & 3) == 0 ? x[0] : (d & 3) == 1 ? x[1] : (d & 3) == 2 ? x[2] : x[3];
            float v = u01(w);
            if (c.skill_init == EJ_SKILL_PARETO_CLIP) {  // Pareto(4) by inversion: 1/sqrt(sqrt(1-u))
                float rr = __fsqrt_rn(__fsub_rn(1.0f, v));
                rr = __fsqrt_rn(rr);
                v = __fdiv_rn(1.0f, rr);
                if (v < c.clip_lo) v = c.clip_lo;
                if (v > c.clip_hi) v = c.clip_hi;
            }
            if (d < c.R) m.SG[d * c.N4 + tid] = v;
            else m.SC[tid] = v;
        }
    }
    for (int l = tid; l < c.n_levels; l += NPAD) { m.head[l] = (uint16_t)NIL; m.tail[l] = (uint16_t)NIL; }
    if (tid == 0) {  // all coins equal: gini = 0, prod = N * coin (exact)
        const double prod = (double)c.N * (double)c.starting_coin;
        const double eq = (double)c.omega * (1.0 - 0.0) + (1.0 - (double)c.omega);
        m.hdr->u_g_prev = eq * prod;
    }
    __syncthreads();
    uint4* blob = (uint4*)(state + (size_t)e * c.blob_bytes);
    for (int i = tid; i < c.blob_bytes / 16; i += NPAD) blob[i] = ((uint4*)smem)[i];
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
char g_create_err[256] = "";

int align16(int x) { return (x + 15) & ~15; }

}  // namespace

struct ej_env {
    DevCfg c;
    ej_params p;
    uint8_t* d_state = nullptr;
    uint32_t* d_cdf = nullptr;
    cudaStream_t stream = 0;
    bool was_reset = false;
    int64_t launches = 0;
    char err[256] = "";
    // staging for ej_step_host
    int32_t *d_act = nullptr, *d_gov = nullptr;
    float *d_obs = nullptr, *d_rew = nullptr;
    uint8_t* d_done = nullptr;
};

namespace {

int fail(ej_env* h, int code, const char* fmt, const char* what) {
    char* dst = h ? h->err : g_create_err;
    snprintf(dst, 256, fmt, what);
    return code;
}

int cuda_fail(ej_env* h, cudaError_t e, const char* where) {
    char* dst = h ? h->err : g_create_err;
    snprintf(dst, 256, "CUDA error in %s: %s", where, cudaGetErrorString(e));
    return EJ_ERR_CUDA;
}

#define EJ_CUDA(h, call, where)                                  \
    do {                                                         \
        cudaError_t _e = (call);                                 \
        if (_e != cudaSuccess) return cuda_fail(h, _e, where);   \
    } while (0)

void build_layout(DevCfg& c) {
    const int N4 = c.N4, R = c.R, nl = c.n_levels;
    int o = (int)sizeof(EnvHdr);
    auto take = [&](int bytes) { const int at = o; o = align16(o + bytes); return at; };
    c.o_coin = take(N4 * 4);
    c.o_labor = take(N4 * 4);
    c.o_income = take(N4 * 4);
    c.o_SC = take(N4 * 4);
    c.o_esc_coin = take(N4 * 4);
    c.o_mask = take(N4 * 4);
    c.o_cf = take(N4 * 8);
    c.o_SG = take(R * N4 * 4);
    c.o_inv = take(R * N4 * 4);
    c.o_esc_res = take(R * N4 * 4);
    c.o_head = take(nl * 2);
    c.o_tail = take(nl * 2);
    c.o_cnt = take(nl * 4);
    c.o_pool = take((c.N << c.Mp_log2) * 4);
    c.blob_bytes = o;
    c.o_key = take(N4 * 4);
    c.o_cinfo = take(N4 * 4);
    c.o_cslot = take(N4 * 4);
    c.o_credit = take(N4 * 4);
    c.o_sale = take(N4 * 4);
    c.o_mb = take(N4 * 4);
    c.o_ma = take(N4 * 4);
    c.o_bucket = take(N4 * 8);
    c.o_sorted = take(N4 * 4);
    c.o_gcnt = take(nl * 4);
    c.o_goff = take(nl * 4);
    c.o_take = take(nl * 4);
    c.o_roff = take(nl * 4);
    c.o_resq = take(32 * 4);
    c.o_resoff = take(32 * 4);
    c.o_red = take((c.n_metrics + 1) * c.n_warps * 8);
    c.o_redq = take(c.n_metrics * c.n_warps * 4);
    c.o_hist = take(R * HB * 4);
    c.o_hovf = take(EJ_MAX_RESOURCES * 4);
    c.o_sortbuf = take(2 * 3 * c.Npad * 4);
    c.o_shrow = take(c.shrow_len * 4);
    c.o_med = take(2 * c.n_metrics * 4);
    c.o_misc = take(16);
    c.o_cdf = take(c.A * 4);
    c.o_stage = o;
    c.stage_obs = 0;
    if ((c.N * c.D_pop) % 4 == 0 && o + c.N * c.D_pop * 4 <= 100 * 1024) {  // bulk-store staging tile
        c.stage_obs = 1;
        take(c.N * c.D_pop * 4);
    }
    c.smem_bytes = o;
}

template <typename F>
int for_block_size(int Npad, F&& f) {
    switch (Npad) {
        case 32: return f(std::integral_constant<int, 32>());
        case 64: return f(std::integral_constant<int, 64>());
        case 128: return f(std::integral_constant<int, 128>());
        case 256: return f(std::integral_constant<int, 256>());
        case 512: return f(std::integral_constant<int, 512>());
        default: return f(std::integral_constant<int, 1024>());
    }
}

int launch_step(ej_env* h, const StepIO& io) {
    const DevCfg& c = h->c;
    return for_block_size(c.Npad, [&](auto mt) {
        constexpr int MT = decltype(mt)::value;
        ej_step_kernel<MT><<<c.E, c.Npad, c.smem_bytes, h->stream>>>(c, h->d_state, io);
        h->launches++;
        EJ_CUDA(h, cudaGetLastError(), "ej_step_kernel launch");
        return EJ_OK;
    });
}

int set_smem_attr(ej_env* h) {
    const DevCfg& c = h->c;
    return for_block_size(c.Npad, [&](auto mt) {
        constexpr int MT = decltype(mt)::value;
        EJ_CUDA(h, cudaFuncSetAttribute(ej_step_kernel<MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, c.smem_bytes), "smem attr (step)");
        EJ_CUDA(h, cudaFuncSetAttribute(ej_observe_kernel<MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, c.smem_bytes), "smem attr (observe)");
        EJ_CUDA(h, cudaFuncSetAttribute(ej_reset_kernel<MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, c.smem_bytes), "smem attr (reset)");
        return EJ_OK;
    });
}

size_t state_words(const DevCfg& c) {
    const size_t N = c.N, R = c.R, B = c.B, cap = (size_t)c.N * c.M;
    return 13 + B + R + N * (6 + 3 * R) + 2 * R * (1 + 3 * cap);
}

int32_t f2w(float f) { int32_t w; memcpy(&w, &f, 4); return w; }
float w2f(int32_t w) { float f; memcpy(&f, &w, 4); return f; }

}  // namespace

extern "C" {

const char* ej_last_error(const ej_env* h) { return h ? h->err : g_create_err; }

int ej_create(int32_t E, int32_t N, int32_t R, const ej_params* p, ej_env** out) {
    g_create_err[0] = 0;
    if (!out) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "out");
    *out = nullptr;
    if (!p) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "params");
    if (p->struct_size != sizeof(ej_params)) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "struct_size");
    if (E < 1) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "E");
    if (N < 1 || N > EJ_MAX_AGENTS) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "N");
    if (R < 1 || R > EJ_MAX_RESOURCES) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "R");
    if (p->num_prices < 1 || p->num_prices > EJ_MAX_PRICES) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "num_prices");
    for (int i = 0; i < p->num_prices; ++i)
        if (p->prices[i] < 1 || (i > 0 && p->prices[i] <= p->prices[i - 1])) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "prices");
    if (p->num_brackets < 1 || p->num_brackets > EJ_MAX_BRACKETS) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "num_brackets");
    for (int i = 0; i + 1 < p->num_brackets; ++i)
        if (!(p->thresholds[i] > (i ? p->thresholds[i - 1] : 0.0f))) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "thresholds");
    if (p->num_rate_levels < 1 || p->num_rate_levels > EJ_MAX_RATE_LEVELS) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "num_rate_levels");
    if (p->craft_mode != EJ_CRAFT_SINGLE && p->craft_mode != EJ_CRAFT_PER_RESOURCE) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "craft_mode");
    if (p->craft_mode == EJ_CRAFT_SINGLE && (p->craft_distinct < 1 || p->craft_distinct > R)) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "craft_distinct");
    if (p->craft_units < 0) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "craft_units");
    if (p->eta == 1.0f) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "eta");
    if (p->episode_length < 1 || p->episode_length > 65535) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "episode_length");
    if (p->tax_period < 1) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "tax_period");
    if (p->order_expiry < 1) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "order_expiry");
    if (p->max_active_orders < 1 || p->max_active_orders > EJ_MAX_ACTIVE_ORDERS) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "max_active_orders");
    if (p->book_cap < 0) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "book_cap");
    if (p->skill_init != EJ_SKILL_UNIFORM01 && p->skill_init != EJ_SKILL_PARETO_CLIP) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "skill_init");
    int mp_log2 = 0;
    while ((1 << mp_log2) < p->max_active_orders) ++mp_log2;
    if (((int64_t)N << mp_log2) >= 65535) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "max_active_orders (N * M too large)");

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, EJ_ERR_CUDA, "%s", "no CUDA device: this library has no CPU fallback");
    }
    ej_env* h = new (std::nothrow) ej_env();
    if (!h) return fail(nullptr, EJ_ERR_NOMEM, "%s", "host allocation failed");
    h->p = *p;
    DevCfg& c = h->c;
    memset(&c, 0, sizeof(c));
    c.E = E; c.N = N; c.R = R; c.P = p->num_prices; c.B = p->num_brackets; c.L = p->num_rate_levels;
    c.M = p->max_active_orders; c.Mp_log2 = mp_log2; c.K = p->book_cap; c.T = p->episode_length;
    c.period = p->tax_period; c.expiry = p->order_expiry > 65535 ? 65535 : p->order_expiry;
    c.craft_units = p->craft_units; c.craft_distinct = p->craft_distinct; c.craft_mode = p->craft_mode;
    c.allow_noop = p->allow_noop ? 1 : 0; c.taxes_enabled = p->taxes_enabled ? 1 : 0; c.skill_init = p->skill_init;
    const int n_craft = c.craft_mode == EJ_CRAFT_PER_RESOURCE ? R : 1;
    c.base_craft = R; c.base_buy = R + n_craft; c.base_sell = c.base_buy + R * c.P;
    c.A = c.base_sell + R * c.P + c.allow_noop;
    c.n_levels = 2 * R * c.P;
    c.n_groups = c.K ? 2 * R : c.n_levels;
    c.D_pop = 6 + 8 * R + c.B;
    c.D_gov = 3 * (3 + R) + c.B + 2;
    c.D_gov_pad = (c.D_gov + 3) & ~3;
    c.N4 = (N + 3) & ~3;
    c.Npad = 32;
    while (c.Npad < N) c.Npad <<= 1;
    c.n_metrics = 3 + R;
    c.n_warps = c.Npad / 32;
    c.shrow_len = 5 * R + c.B + 2;
    for (int i = 0; i < c.P; ++i) c.prices[i] = p->prices[i];
    for (int i = 0; i + 1 < c.B; ++i) c.thresholds[i] = p->thresholds[i];
    for (int i = 0; i < c.L; ++i) c.rate_table[i] = p->rate_table[i];
    c.starting_coin = p->starting_coin; c.labor_craft = p->labor_craft; c.labor_gather = p->labor_gather;
    c.labor_trade = p->labor_trade; c.eta = p->eta; c.omega = p->omega; c.craft_scale = p->craft_scale;
    c.clip_lo = p->skill_clip_lo; c.clip_hi = p->skill_clip_hi;
    c.s_coin = p->obs_scale_coin; c.s_count = p->obs_scale_count; c.s_price = p->obs_scale_price; c.s_labor = p->obs_scale_labor;
    c.env_id_base = p->env_id_base;
    c.gov_obs_offset = ((unsigned long long)E * N * c.D_pop + 3ull) & ~3ull;
    c.obs_floats = c.gov_obs_offset + (unsigned long long)E * c.D_gov_pad;
    build_layout(c);
    if (c.smem_bytes > 227 * 1024) {
        delete h;
        return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "N/R/max_active_orders (state exceeds 227 KB of shared memory)");
    }
    int rc = set_smem_attr(h);
    if (rc != EJ_OK) { memcpy(g_create_err, h->err, 256); delete h; return rc; }
    cudaError_t ce = cudaMalloc(&h->d_state, (size_t)E * c.blob_bytes);
    if (ce == cudaSuccess) ce = cudaMalloc(&h->d_cdf, (size_t)c.A * 4);
    if (ce != cudaSuccess) {
        cudaGetLastError();
        if (h->d_state) cudaFree(h->d_state);
        delete h;
        return fail(nullptr, EJ_ERR_NOMEM, "%s", "device allocation failed");
    }
    std::vector<uint32_t> cdf(c.A);  // default: uniform over the A actions
    for (int a = 0; a < c.A; ++a) {
        const uint64_t v = (((uint64_t)(a + 1)) << 32) / (uint64_t)c.A;
        cdf[a] = (uint32_t)(v > 0xFFFFFFFFull ? 0xFFFFFFFFull : v);
    }
    cdf[c.A - 1] = 0xFFFFFFFFu;
    ce = cudaMemcpy(h->d_cdf, cdf.data(), (size_t)c.A * 4, cudaMemcpyHostToDevice);
    if (ce != cudaSuccess) { cuda_fail(nullptr, ce, "cdf upload"); ej_destroy(h); return EJ_ERR_CUDA; }
    *out = h;
    return EJ_OK;
}

int ej_destroy(ej_env* h) {
    if (!h) return EJ_OK;
    cudaStreamSynchronize(h->stream);
    cudaFree(h->d_state); cudaFree(h->d_cdf);
    cudaFree(h->d_act); cudaFree(h->d_gov); cudaFree(h->d_obs); cudaFree(h->d_rew); cudaFree(h->d_done);
    delete h;
    return EJ_OK;
}

int ej_set_stream(ej_env* h, void* s) {
    if (!h) return EJ_ERR_PARAM;
    h->stream = (cudaStream_t)s;
    return EJ_OK;
}

int ej_layout(const ej_env* h, ej_layout_info* o) {
    if (!h || !o) return EJ_ERR_PARAM;
    const DevCfg& c = h->c;
    memset(o, 0, sizeof(*o));
    o->E = c.E; o->N = c.N; o->R = c.R; o->P = c.P; o->B = c.B; o->L = c.L; o->A = c.A;
    o->base_craft = c.base_craft; o->base_buy = c.base_buy; o->base_sell = c.base_sell;
    o->noop_action = c.allow_noop ? c.A - 1 : -1;
    o->D_pop = c.D_pop; o->D_gov = c.D_gov; o->D_gov_pad = c.D_gov_pad;
    o->gov_obs_offset = (size_t)c.gov_obs_offset; o->obs_floats = (size_t)c.obs_floats;
    o->rew_floats = (size_t)c.E * (c.N + 1);
    o->state_words = state_words(c);
    o->device_state_bytes = (size_t)c.blob_bytes;
    o->smem_bytes = (size_t)c.smem_bytes;
    o->threads_per_env = c.Npad;
    return EJ_OK;
}

int ej_reset(ej_env* h, uint64_t seed) {
    if (!h) return EJ_ERR_PARAM;
    DevCfg& c = h->c;
    c.seed_lo = (uint32_t)(seed & 0xFFFFFFFFull);
    c.seed_hi = (uint32_t)(seed >> 32);
    int rc = for_block_size(c.Npad, [&](auto mt) {
        constexpr int MT = decltype(mt)::value;
        ej_reset_kernel<MT><<<c.E, c.Npad, c.smem_bytes, h->stream>>>(c, h->d_state);
        h->launches++;
        EJ_CUDA(h, cudaGetLastError(), "ej_reset_kernel launch");
        return EJ_OK;
    });
    if (rc == EJ_OK) h->was_reset = true;
    return rc;
}

int ej_observe(ej_env* h, float* obs_out) {
    if (!h || !obs_out) return h ? fail(h, EJ_ERR_PARAM, "bad field: %s", "obs_out") : EJ_ERR_PARAM;
    if (!h->was_reset) return fail(h, EJ_ERR_STATE, "%s", "ej_observe before ej_reset / ej_set_state");
    const DevCfg& c = h->c;
    return for_block_size(c.Npad, [&](auto mt) {
        constexpr int MT = decltype(mt)::value;
        ej_observe_kernel<MT><<<c.E, c.Npad, c.smem_bytes, h->stream>>>(c, h->d_state, obs_out);
        h->launches++;
        EJ_CUDA(h, cudaGetLastError(), "ej_observe_kernel launch");
        return EJ_OK;
    });
}

int ej_step(ej_env* h, const int32_t* actions, const int32_t* gov_actions, float* obs_out, float* rew_out, uint8_t* done_out) {
    if (!h) return EJ_ERR_PARAM;
    if (!actions) return fail(h, EJ_ERR_PARAM, "bad field: %s", "actions");
    if (!gov_actions) return fail(h, EJ_ERR_PARAM, "bad field: %s", "gov_actions");
    if (!h->was_reset) return fail(h, EJ_ERR_STATE, "%s", "ej_step before ej_reset / ej_set_state");
    StepIO io;
    memset(&io, 0, sizeof(io));
    io.actions = actions; io.gov_actions = gov_actions; io.obs = obs_out; io.rew = rew_out; io.done = done_out;
    io.cdf = h->d_cdf; io.n_steps = 1; io.ring_depth = 1;
    return launch_step(h, io);
}

int ej_step_host(ej_env* h, const int32_t* actions, const int32_t* gov_actions, float* obs_out, float* rew_out, uint8_t* done_out) {
    if (!h) return EJ_ERR_PARAM;
    if (!actions) return fail(h, EJ_ERR_PARAM, "bad field: %s", "actions");
    if (!gov_actions) return fail(h, EJ_ERR_PARAM, "bad field: %s", "gov_actions");
    const DevCfg& c = h->c;
    const size_t EN = (size_t)c.E * c.N, EB = (size_t)c.E * c.B;
    if (!h->d_act) {
        cudaError_t ce = cudaMalloc(&h->d_act, EN * 4);
        if (ce == cudaSuccess) ce = cudaMalloc(&h->d_gov, EB * 4);
        if (ce == cudaSuccess) ce = cudaMalloc(&h->d_obs, (size_t)c.obs_floats * 4);
        if (ce == cudaSuccess) ce = cudaMalloc(&h->d_rew, (EN + c.E) * 4);
        if (ce == cudaSuccess) ce = cudaMalloc(&h->d_done, (size_t)c.E);
        if (ce != cudaSuccess) { cudaGetLastError(); return fail(h, EJ_ERR_NOMEM, "%s", "staging allocation failed"); }
    }
    EJ_CUDA(h, cudaMemcpyAsync(h->d_act, actions, EN * 4, cudaMemcpyHostToDevice, h->stream), "H2D actions");
    EJ_CUDA(h, cudaMemcpyAsync(h->d_gov, gov_actions, EB * 4, cudaMemcpyHostToDevice, h->stream), "H2D gov_actions");
    int rc = ej_step(h, h->d_act, h->d_gov, obs_out ? h->d_obs : nullptr, rew_out ? h->d_rew : nullptr, done_out ? h->d_done : nullptr);
    if (rc != EJ_OK) return rc;
    if (obs_out) EJ_CUDA(h, cudaMemcpyAsync(obs_out, h->d_obs, (size_t)c.obs_floats * 4, cudaMemcpyDeviceToHost, h->stream), "D2H obs");
    if (rew_out) EJ_CUDA(h, cudaMemcpyAsync(rew_out, h->d_rew, (EN + c.E) * 4, cudaMemcpyDeviceToHost, h->stream), "D2H rewards");
    if (done_out) EJ_CUDA(h, cudaMemcpyAsync(done_out, h->d_done, (size_t)c.E, cudaMemcpyDeviceToHost, h->stream), "D2H done");
    EJ_CUDA(h, cudaStreamSynchronize(h->stream), "ej_step_host sync");
    return EJ_OK;
}

int ej_rollout(ej_env* h, int32_t T, const ej_rollout_io* rio) {
    if (!h) return EJ_ERR_PARAM;
    if (T < 0) return fail(h, EJ_ERR_PARAM, "bad field: %s", "T");
    if (!h->was_reset) return fail(h, EJ_ERR_STATE, "%s", "ej_rollout before ej_reset / ej_set_state");
    if (T == 0) return EJ_OK;
    StepIO io;
    memset(&io, 0, sizeof(io));
    io.cdf = h->d_cdf; io.n_steps = T; io.ring_depth = 1;
    if (rio) {
        if (rio->struct_size != sizeof(ej_rollout_io)) return fail(h, EJ_ERR_PARAM, "bad field: %s", "io.struct_size");
        if (rio->ring_depth < 1) return fail(h, EJ_ERR_PARAM, "bad field: %s", "io.ring_depth");
        io.ring_depth = rio->ring_depth;
        io.actions = rio->actions_in; io.gov_actions = rio->gov_actions_in;
        io.obs = rio->obs_ring; io.rew = rio->rew_ring; io.done = rio->done_ring;
        io.actions_out = rio->actions_ring; io.gov_out = rio->gov_actions_ring;
    }
    return launch_step(h, io);
}

int ej_set_action_cdf(ej_env* h, const uint32_t* cdf, int32_t A) {
    if (!h) return EJ_ERR_PARAM;
    if (!cdf) return fail(h, EJ_ERR_PARAM, "bad field: %s", "cdf");
    if (A != h->c.A) return fail(h, EJ_ERR_PARAM, "bad field: %s", "A");
    for (int a = 1; a < A; ++a)
        if (cdf[a] < cdf[a - 1]) return fail(h, EJ_ERR_PARAM, "bad field: %s", "cdf (not monotone)");
    EJ_CUDA(h, cudaMemcpyAsync(h->d_cdf, cdf, (size_t)A * 4, cudaMemcpyHostToDevice, h->stream), "cdf upload");
    EJ_CUDA(h, cudaStreamSynchronize(h->stream), "cdf upload sync");
    return EJ_OK;
}

int64_t ej_launch_count(const ej_env* h) { return h ? h->launches : 0; }

int ej_get_state(ej_env* h, int32_t env_begin, int32_t env_count, int32_t* words, size_t n_words) {
    if (!h) return EJ_ERR_PARAM;
    const DevCfg& c = h->c;
    if (env_begin < 0 || env_count < 0 || env_begin + env_count > c.E) return fail(h, EJ_ERR_PARAM, "bad field: %s", "env range");
    const size_t W = state_words(c);
    if (!words || n_words < W * (size_t)env_count) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words / n_words");
    if (!h->was_reset) return fail(h, EJ_ERR_STATE, "%s", "ej_get_state before ej_reset / ej_set_state");
    std::vector<uint8_t> blobs((size_t)env_count * c.blob_bytes);
    EJ_CUDA(h, cudaStreamSynchronize(h->stream), "get_state sync");
    EJ_CUDA(h, cudaMemcpy(blobs.data(), h->d_state + (size_t)env_begin * c.blob_bytes, blobs.size(), cudaMemcpyDeviceToHost), "get_state copy");
    const int N = c.N, R = c.R, B = c.B, P = c.P, cap = c.N * c.M, N4 = c.N4;
    for (int k = 0; k < env_count; ++k) {
        const uint8_t* s = blobs.data() + (size_t)k * c.blob_bytes;
        const EnvHdr* hd = (const EnvHdr*)s;
        const float* coin = (const float*)(s + c.o_coin); const float* labor = (const float*)(s + c.o_labor);
        const float* income = (const float*)(s + c.o_income); const float* SC = (const float*)(s + c.o_SC);
        const int* esc_coin = (const int*)(s + c.o_esc_coin); const uint32_t* mask = (const uint32_t*)(s + c.o_mask);
        const float* SG = (const float*)(s + c.o_SG); const int* inv = (const int*)(s + c.o_inv);
        const int* esc_res = (const int*)(s + c.o_esc_res);
        const uint16_t* head = (const uint16_t*)(s + c.o_head); const int* cnt = (const int*)(s + c.o_cnt);
        const uint32_t* pool = (const uint32_t*)(s + c.o_pool);
        int32_t* w = words + (size_t)k * W;
        memset(w, 0, W * 4);
        size_t q = 0;
        w[q++] = hd->t; w[q++] = N; w[q++] = R; w[q++] = B; w[q++] = P; w[q++] = cap;
        w[q++] = hd->n_trades; w[q++] = hd->n_placed; w[q++] = hd->n_invalid; w[q++] = hd->n_expired; w[q++] = hd->n_bad_gov;
        memcpy(&w[q], &hd->u_g_prev, 8); q += 2;
        for (int b = 0; b < B; ++b) w[q++] = f2w(hd->rates[b]);
        for (int r = 0; r < R; ++r) w[q++] = hd->last_price[r];
        for (int i = 0; i < N; ++i) {
            int nlive = 0;
            for (uint32_t mm = mask[i]; mm; mm &= mm - 1) ++nlive;
            w[q++] = f2w(coin[i]); w[q++] = esc_coin[i]; w[q++] = f2w(SC[i]);
            w[q++] = f2w(labor[i]); w[q++] = f2w(income[i]); w[q++] = nlive;
            for (int r = 0; r < R; ++r) w[q++] = inv[r * N4 + i];
            for (int r = 0; r < R; ++r) w[q++] = esc_res[r * N4 + i];
            for (int r = 0; r < R; ++r) w[q++] = f2w(SG[r * N4 + i]);
        }
        for (int b = 0; b < 2 * R; ++b) {
            const int side = b & 1;
            int n = 0;
            for (int p = 0; p < P; ++p) n += cnt[b * P + p];
            w[q++] = n;
            const size_t q0 = q;
            int out = 0;
            for (int pp = 0; pp < P; ++pp) {  // priority: bids price descending, asks ascending, then FIFO
                const int p = side == 0 ? P - 1 - pp : pp;
                uint32_t hh = head[b * P + p];
                int guard = 0;
                while (hh != NIL && guard++ < cap + 1) {
                    const uint32_t pe = pool[hh];
                    const int age = (int)(((uint32_t)hd->t - (pe >> 16)) & 0xFFFFu);
                    if (out < cap) {
                        w[q0 + 3 * out] = c.prices[p];
                        w[q0 + 3 * out + 1] = (int32_t)(hh >> c.Mp_log2);
                        w[q0 + 3 * out + 2] = hd->t - age;
                    }
                    ++out;
                    hh = pe & 0xFFFFu;
                }
            }
            q = q0 + 3 * (size_t)cap;
        }
    }
    return EJ_OK;
}

int ej_set_state(ej_env* h, int32_t env_begin, int32_t env_count, const int32_t* words, size_t n_words) {
    if (!h) return EJ_ERR_PARAM;
    const DevCfg& c = h->c;
    if (env_begin < 0 || env_count < 0 || env_begin + env_count > c.E) return fail(h, EJ_ERR_PARAM, "bad field: %s", "env range");
    const size_t W = state_words(c);
    if (!words || n_words < W * (size_t)env_count) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words / n_words");
    const int N = c.N, R = c.R, B = c.B, P = c.P, cap = c.N * c.M, N4 = c.N4;
    std::vector<uint8_t> blobs((size_t)env_count * c.blob_bytes, 0);
    for (int k = 0; k < env_count; ++k) {
        uint8_t* s = blobs.data() + (size_t)k * c.blob_bytes;
        EnvHdr* hd = (EnvHdr*)s;
        float* coin = (float*)(s + c.o_coin); float* labor = (float*)(s + c.o_labor);
        float* income = (float*)(s + c.o_income); float* SC = (float*)(s + c.o_SC);
        int* esc_coin = (int*)(s + c.o_esc_coin); uint32_t* mask = (uint32_t*)(s + c.o_mask);
        double* cf = (double*)(s + c.o_cf);
        float* SG = (float*)(s + c.o_SG); int* inv = (int*)(s + c.o_inv); int* esc_res = (int*)(s + c.o_esc_res);
        uint16_t* head = (uint16_t*)(s + c.o_head); uint16_t* tail = (uint16_t*)(s + c.o_tail);
        int* cnt = (int*)(s + c.o_cnt); uint32_t* pool = (uint32_t*)(s + c.o_pool);
        const int32_t* w = words + (size_t)k * W;
        size_t q = 0;
        hd->t = w[q++];
        if (w[q] != N || w[q + 1] != R || w[q + 2] != B || w[q + 3] != P || w[q + 4] != cap) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words (shape header mismatch)");
        q += 5;
        if (hd->t < 0 || hd->t > c.T) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words (t)");
        hd->n_trades = w[q++]; hd->n_placed = w[q++]; hd->n_invalid = w[q++]; hd->n_expired = w[q++]; hd->n_bad_gov = w[q++];
        memcpy(&hd->u_g_prev, &w[q], 8); q += 2;
        for (int b = 0; b < B; ++b) hd->rates[b] = w2f(w[q++]);
        for (int r = 0; r < R; ++r) hd->last_price[r] = w[q++];
        for (int i = 0; i < N; ++i) {
            coin[i] = w2f(w[q++]); esc_coin[i] = w[q++]; SC[i] = w2f(w[q++]);
            labor[i] = w2f(w[q++]); income[i] = w2f(w[q++]); q++;  // n_live is implied by the books
            for (int r = 0; r < R; ++r) inv[r * N4 + i] = w[q++];
            for (int r = 0; r < R; ++r) esc_res[r * N4 + i] = w[q++];
            for (int r = 0; r < R; ++r) SG[r * N4 + i] = w2f(w[q++]);
            const double a = 1.0 - (double)c.eta;
            cf[i] = (pow((double)coin[i], a) - 1.0) / a;
        }
        for (int l = 0; l < c.n_levels; ++l) { head[l] = (uint16_t)NIL; tail[l] = (uint16_t)NIL; }
        for (int b = 0; b < 2 * R; ++b) {
            const int n = w[q++];
            if (n < 0 || n > cap) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words (book size)");
            for (int o = 0; o < n; ++o) {  // priority order keeps each level's FIFO order
                const int price = w[q + 3 * o], owner = w[q + 3 * o + 1], placed = w[q + 3 * o + 2];
                int p = -1;
                for (int pp = 0; pp < P; ++pp) if (c.prices[pp] == price) p = pp;
                if (p < 0 || owner < 0 || owner >= N || placed < 0 || placed > hd->t) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words (order)");
                uint32_t free_bits = ~mask[owner] & (c.M >= 32 ? 0xFFFFFFFFu : ((1u << c.M) - 1u));
                if (!free_bits) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words (more than M orders for one agent)");
                int bit = 0;
                while (!((free_bits >> bit) & 1u)) ++bit;
                mask[owner] |= 1u << bit;
                const uint32_t slot = ((uint32_t)owner << c.Mp_log2) + (uint32_t)bit;
                pool[slot] = NIL | (((uint32_t)placed & 0xFFFFu) << 16);
                const int l = b * P + p;
                if (tail[l] != NIL) pool[tail[l]] = (pool[tail[l]] & 0xFFFF0000u) | slot;
                else head[l] = (uint16_t)slot;
                tail[l] = (uint16_t)slot;
                cnt[l]++;
            }
            q += 3 * (size_t)cap;
        }
    }
    EJ_CUDA(h, cudaStreamSynchronize(h->stream), "set_state sync");
    EJ_CUDA(h, cudaMemcpy(h->d_state + (size_t)env_begin * c.blob_bytes, blobs.data(), blobs.size(), cudaMemcpyHostToDevice), "set_state copy");
    h->was_reset = true;
    return EJ_OK;
}

}  // extern "C"
