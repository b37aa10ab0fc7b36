// ej_device.cuh -- device side of the batched EconoJax environment step (sm_100a).
//
// One CTA per economy; thread i is population agent i.  The whole state of an economy (agent
// arrays, per-level FIFO order books, order pool) is one contiguous "blob" that is copied into
// shared memory at kernel start and written back at kernel end; ej_rollout keeps it there for
// T steps.  Citations: "P:n" = PAPER.md line n, "G#" = DESIGN.md section 3 readings.
//
// Arithmetic contract (G31): agent state is binary32 and every state-changing float operation
// is ONE correctly rounded operation (__fadd_rn / __fmul_rn / __fsub_rn / __fdiv_rn: never
// contracted to FMA); cross-agent accumulations are integers (order-free, atomics allowed);
// rewards and statistics are evaluated in binary64 where cancellation matters.
//
// Order book: every (resource, side, price) level is a FIFO in arrival order
// because the price grid is discrete and an older step always precedes a newer one (G11), so
// both kinds of removal -- matching (best price first, then earliest arrival) and
// expiry (oldest first) -- pop queue heads.  Levels are singly linked lists threaded
// through a pool in which agent i owns slots [i*Mp, i*Mp+M): an agent places at most one order
// per step and holds at most M, so slot allocation is a private bitmask operation.
//
// Barriers per step (book_cap == 0): arrivals pushed | linked | level pops | trades settled |
// state final | outputs staged.  Government statistics are warp-specialised: one warp owns one
// metric, holds all N values in registers (N/32 per lane) and needs no block barrier.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#ifdef EJ_PHASE_CLOCK
#include <stdio.h>
#endif

#include "../../include/econojax.h"

#ifndef EJ_CTAS_128_FX
#define EJ_CTAS_128_FX 10  // the shape-specialised factored variants: their small tile lets 10 CTAs fit an SM (47 registers, no spills)
#endif
#ifndef EJ_CTAS_128
#define EJ_CTAS_128 8  // resident 128-thread CTAs per SM the step kernel is compiled for (register budget 64; 9 fit the shared memory at the headline shape but measured no faster)
#endif

namespace {

// Debug builds (-DEJ_PHASE_CLOCK): block 0 accumulates the cycles between the barriers of a step and prints them at
// the end of the launch.  Not compiled into the product library.
#ifdef EJ_PHASE_CLOCK
__device__ unsigned long long ej_phase_cycles[16];
__device__ unsigned long long ej_phase_last;
#define EJ_MARK(k)                                                                     \
    do {                                                                               \
        if (blockIdx.x == 0 && threadIdx.x == 0) {                                     \
            const unsigned long long now_ = clock64();                                 \
            ej_phase_cycles[k] += now_ - ej_phase_last;                                \
            ej_phase_last = now_;                                                      \
        }                                                                              \
    } while (0)
#else
#define EJ_MARK(k) do { } while (0)
#endif

constexpr uint32_t NIL = 0xFFFFu;      // null slot of the order pool
// Order-pool word of a slot: next slot of its price level's FIFO | step at which the order was placed.  Two formats:
//   W = 0  32 bits: next (16) | placed_at (16): any shape;
//   W = 1  16 bits: next (11, 0x7FF = none) | placed_at mod 32 (5): the paper's mechanics at N <= 127 (16 slots per agent:
//          N * 16 <= 2032 slots) with order_expiry <= 31 (30) -- an order's age t - placed_at never exceeds the
//          expiry, so five bits of the clock identify it.  Halves the pool (3.2 KB per economy at N = 100), which
//          is what lets one more CTA stay resident per SM.
template <int W> struct PoolW;
template <> struct PoolW<0> {
    using T = uint32_t;
    __device__ __forceinline__ static T make(uint32_t nxt, int t) { return nxt | (((uint32_t)t & 0xFFFFu) << 16); }
    __device__ __forceinline__ static uint32_t next(T w) { return w & 0xFFFFu; }
    __device__ __forceinline__ static uint32_t age(T w, int t) { return ((uint32_t)t - (w >> 16)) & 0xFFFFu; }
    __device__ __forceinline__ static T with_next(T w, uint32_t nxt) { return (w & 0xFFFF0000u) | nxt; }
};
template <> struct PoolW<1> {
    using T = uint16_t;
    __device__ __forceinline__ static T make(uint32_t nxt, int t) { return (T)((nxt & 0x7FFu) | (((uint32_t)t & 31u) << 11)); }  // NIL & 0x7FF = 0x7FF
    __device__ __forceinline__ static uint32_t next(T w) { const uint32_t n = w & 0x7FFu; return n == 0x7FFu ? NIL : n; }
    __device__ __forceinline__ static uint32_t age(T w, int t) { return ((uint32_t)t - ((uint32_t)w >> 11)) & 31u; }
    __device__ __forceinline__ static T with_next(T w, uint32_t nxt) { return (T)((w & 0xF800u) | (nxt & 0x7FFu)); }
};

// Book-cap path: a step's candidates are binned by the top bits of their arrival key (a uniform Philox word, G11):
// 256 bins per book give the rank of a candidate on its book, 32 bins per level its neighbours on its level.
constexpr int BOOK_BINS = 256, BOOK_BIN_SHIFT = 24, LEVEL_BINS = 32, LEVEL_BIN_SHIFT = 27;
constexpr uint32_t FULL = 0xffffffffu;

struct EnvHdr {
    int32_t t;
    int32_t n_trades, n_placed, n_invalid, n_expired, n_bad_gov;
    uint32_t med_prev[2 + EJ_MAX_RESOURCES];  // previous lower medians of labor, income (float bits) and inv[r]: hints, not state
    double u_g_prev;
    int32_t t_in_period;  // t % tax_period, kept incrementally (no integer division on the step path)
    int32_t episode;      // f4: episode index (0 after ej_reset), part of every Philox counter: stream | episode << 8 (G44)
    float rates[EJ_MAX_BRACKETS];
    int32_t last_price[EJ_MAX_RESOURCES];
};
static_assert(sizeof(EnvHdr) % 16 == 0, "EnvHdr must keep 16-byte alignment");

struct DevCfg {
    int E, N, R, P, B, L, M, Mp_log2, K, T, period, expiry;
    int craft_units, craft_distinct, craft_mode, allow_noop, taxes_enabled, skill_init;
    int recipP;  // ceil(2^16 / P): k / P == (k * recipP) >> 16 for k < 2RP <= 512
    int A, base_craft, base_buy, base_sell, n_levels, n_groups, D_pop, D_gov, D_gov_pad;
    int N4, Npad, n_metrics, n_warps, shrow_len, stage_obs;
    int pool16;             // order-pool words are 16 bits (PoolW<1>): the shape-specialised paper-mechanics kernels
    int stage_alias_bytes;  // head of the staging tile that the matched-order lists overwrite every step
    int prices[EJ_MAX_PRICES];
    float thresholds[EJ_MAX_BRACKETS];
    float rate_table[EJ_MAX_RATE_LEVELS];
    float starting_coin, labor_craft, labor_gather, labor_trade, eta, omega, craft_scale;
    float clip_lo, clip_hi, s_coin, s_count, s_price, s_labor;
    float skill_rate, skill_max;  // f3: skill_rate == 0 keeps the skills fixed
    float skill_mean, skill_std;  // f3: EJ_SKILL_NORMAL_CLIP
    double inv_n;  // 1 / N
    double ua, inv_ua;  // 1 - eta and its reciprocal (Eq.1)
    uint32_t env_id_base, seed_lo, seed_hi;
    // blob section offsets (bytes from the blob base)
    int o_coin, o_labor, o_income, o_SC, o_esc_coin, o_mask, o_cf, o_SG, o_inv, o_esc_res;
    int o_head, o_tail, o_cnt, o_pool, o_spl, blob_bytes;
    int o_blob, o_scratch1;  // absolute: blob start (= Lay<Npad>::blob), first byte after the blob
    // scratch section offsets (bytes from the shared-memory base; all after the blob)
    int o_key, o_cinfo, o_cslot, o_anext, o_ahead, o_credit, o_sale, o_mb, o_ma;
    int o_bbh, o_bbc, o_lbh, o_lmask;  // book-cap path (K > 0): arrival bins per book and per level
    int o_bk2;                         // bucket keys of labor and income (CTAs of 512 / 1024 threads)
    int o_resq, o_shrow, o_govrow, o_misc, o_cdf, o_rowbuf, o_stage;
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
    int masked;                  // f1: the generator draws among the available actions only
    int auto_reset;              // f4: an env whose episode ends starts the next one in the same step (G44)
    float* obs_priv;             // f2 rings (factored observations): [E][N][3R+4], [E][ceil4(5R+B+2)], [E][D_gov_pad]
    float* obs_shared;
    float* obs_gov;
};

// Shared-memory layout of one economy.  Everything whose size depends only on the CTA size NP
// sits at a COMPILE-TIME offset, with per-agent arrays strided by NP: an access is then one
// LDS/STS [tid*4 + immediate] instead of a rematerialised base pointer (the first version kept
// ~30 generic pointers in a struct; rebuilding them cost ~10 % of all executed instructions).
//   [fixed scratch][blob: header | per-agent scalars | inv | esc_res | SG | levels | pool][scratch]
// Offsets of the R-, P- and M-dependent sections are runtime values in DevCfg (relative to the
// blob for blob sections, absolute otherwise).  The host reads the same constants (econojax.cu).
template <int NP>
struct Lay {
    // fixed scratch (absolute byte offsets)
    static constexpr int key = 0;                 // arrival tie keys (Philox x2), u32 [NP]
    static constexpr int cslot = key + NP * 4;    // pool slot of this step's candidate order
    static constexpr int anext = cslot + NP * 4;  // arrival stacks: next candidate (K == 0); cinfo (K > 0)
    static constexpr int credit = anext + NP * 4; // coin credited this step, i32
    static constexpr int sale = credit + NP * 4;  // sale proceeds this step, i32
    static constexpr int resq = sale + NP * 4;    // trades per resource, i32 [16]
    static constexpr int shrow = resq + EJ_MAX_RESOURCES * 4;  // shared tail of the population rows
    static constexpr int shrow_cap = 5 * EJ_MAX_RESOURCES + EJ_MAX_BRACKETS + 4;
    static constexpr int govrow = shrow + shrow_cap * 4;
    static constexpr int govrow_cap = 80;  // >= ceil4(3 (3 + 16) + 16 + 2)
    static constexpr int misc = govrow + govrow_cap * 4;       // u64 [2]: tax pool
    // block-wide sort of the float metrics (bucket_fill / bucket_sort below): one bucket per warp and metric.  NP is the
    // array stride (13/16 of the CTA size, or the CTA size): CTAs of 512 / 1024 threads sort coin, labor and income this way.
    static constexpr int bk_warps = NP >= 832 ? 32 : NP >= 416 ? 16 : NP >= 208 ? 8 : 4;
    // (measured at N = 100: bucketing the coin across the four warps of a 128-thread CTA cost 9 us per batched step,
    // 32.4 -> 42 us; the register network on one warp is cheaper there, so small CTAs do not bucket)
    static constexpr int bk_metrics = NP >= 416 ? 3 : 0;
    static constexpr bool bucketed = bk_metrics > 0;
    // the coin's bucket keys live in key | cslot | anext (3 NP words): those are dead between the settlement of a
    // step's trades and the next step's arrivals, which is when the buckets are filled and sorted
    static constexpr int bk_keys = key;
    static constexpr int bk_cap = (3 * NP / bk_warps) < 128 ? (3 * NP / bk_warps) : 128;  // keys per bucket (sorted 4 per lane at most)
    static constexpr int bk_cnt_words = 2 * bk_warps + 4;       // per metric: bucket sizes | values equal to a bound | overflow flag, two medians
    static constexpr int bk_cnt = misc + 16;
    static constexpr int bk_part = bk_cnt + ((bk_metrics * bk_cnt_words * 4 + 15) & ~15);  // f64 [metrics][warps][3]: gini, sum, sum of squares per bucket
    static constexpr int blob = bk_part + ((bk_metrics * bk_warps * 3 * 8 + 15) & ~15);
    // bucket bounds (hints, kept in the blob): u32 [metrics][2][warps] double-buffered, then the index of the buffer in force
    static constexpr int spl_bytes = bucketed ? ((bk_metrics * 2 * bk_warps * 4 + 4 + 15) & ~15) : 0;
    // blob sections (byte offsets relative to the blob)
    static constexpr int coin = (int)sizeof(EnvHdr);
    static constexpr int labor = coin + NP * 4;
    static constexpr int income = labor + NP * 4;
    static constexpr int SC = income + NP * 4;
    static constexpr int esc_coin = SC + NP * 4;
    static constexpr int mask = esc_coin + NP * 4;
    static constexpr int cf = mask + NP * 4;      // cached coin utility, f64 [NP]
    static constexpr int inv = cf + NP * 8;       // i32 [R][NP]; esc_res and SG follow (runtime offsets)
    static_assert(blob % 16 == 0 && inv % 16 == 0, "16-byte alignment");
};

// Offsets of the R-, P-, N-dependent sections when those are compile-time constants and the
// paper's mechanics hold (16 pool slots per agent, no book cap: PF = 1 in the step kernel): the
// same arithmetic as build_layout() in econojax.cu, which checks the two against each other
// before it selects a kernel that relies on this.
constexpr int lay_align16(int x) { return (x + 15) & ~15; }
template <int NP, int R, int P, int N>
struct StaticLay {
    static constexpr int nl = 2 * R * P, A = 2 * R * P + R + 2;
    static constexpr int esc_res = lay_align16(Lay<NP>::inv + R * NP * 4);
    static constexpr int SG = lay_align16(esc_res + R * NP * 4);
    static constexpr int head = lay_align16(SG + R * NP * 4);
    static constexpr int tail = lay_align16(head + nl * 2);
    static constexpr int cnt = lay_align16(tail + nl * 2);
    static constexpr int pool = lay_align16(cnt + 2 * nl * 4);
    static constexpr int spl = lay_align16(pool + (N << 4) * 2);  // 16-bit pool words (PoolW<1>)
    static constexpr int blob_bytes = spl + Lay<NP>::spl_bytes;
    static constexpr int ahead = Lay<NP>::blob + blob_bytes;  // absolute from here on
    static constexpr int cdf = lay_align16(ahead + nl * 4);
    static constexpr int stage = lay_align16(cdf + A * 4);
    static constexpr int mb = stage, ma = stage + R * NP * 4;
};

// View of one economy's shared memory.  SR > 0: static layout (StaticLay<NP, SR, SP, SN>).
template <int NP, int SR = 0, int SP = 0, int SN = 0>
struct Sm {
    using L = Lay<NP>;
    using S = StaticLay<NP, (SR > 0 ? SR : 1), (SP > 0 ? SP : 1), (SN > 0 ? SN : 1)>;
    static constexpr bool ST = SR > 0;
    const DevCfg& c;
    template <class T>
    __device__ __forceinline__ static T* at(int off) {
        extern __shared__ __align__(16) uint8_t ej_smem[];
        return reinterpret_cast<T*>(ej_smem + off);
    }
    __device__ __forceinline__ EnvHdr* hdr() const { return at<EnvHdr>(L::blob); }
    __device__ __forceinline__ float* coin() const { return at<float>(L::blob + L::coin); }
    __device__ __forceinline__ float* labor() const { return at<float>(L::blob + L::labor); }
    __device__ __forceinline__ float* income() const { return at<float>(L::blob + L::income); }
    __device__ __forceinline__ float* SC() const { return at<float>(L::blob + L::SC); }
    __device__ __forceinline__ int* esc_coin() const { return at<int>(L::blob + L::esc_coin); }
    __device__ __forceinline__ uint32_t* mask() const { return at<uint32_t>(L::blob + L::mask); }
    __device__ __forceinline__ double* cf() const { return at<double>(L::blob + L::cf); }
    __device__ __forceinline__ int* inv() const { return at<int>(L::blob + L::inv); }
    __device__ __forceinline__ int* esc_res() const { return at<int>(L::blob + (ST ? S::esc_res : c.o_esc_res)); }
    __device__ __forceinline__ float* SG() const { return at<float>(L::blob + (ST ? S::SG : c.o_SG)); }
    __device__ __forceinline__ uint16_t* head() const { return at<uint16_t>(L::blob + (ST ? S::head : c.o_head)); }
    __device__ __forceinline__ uint16_t* tail() const { return at<uint16_t>(L::blob + (ST ? S::tail : c.o_tail)); }
    __device__ __forceinline__ int* cnt() const { return at<int>(L::blob + (ST ? S::cnt : c.o_cnt)); }  // [2][n_levels]: buffer (t & 1) is current
    template <int W>
    __device__ __forceinline__ typename PoolW<W>::T* pool() const { return at<typename PoolW<W>::T>(L::blob + (ST ? S::pool : c.o_pool)); }
    __device__ __forceinline__ uint32_t* key() const { return at<uint32_t>(L::key); }
    __device__ __forceinline__ uint32_t* cslot() const { return at<uint32_t>(L::cslot); }
    __device__ __forceinline__ uint32_t* anext() const { return at<uint32_t>(L::anext); }
    __device__ __forceinline__ int* cinfo() const { return at<int>(L::anext); }
    __device__ __forceinline__ int* credit() const { return at<int>(L::credit); }
    __device__ __forceinline__ int* sale() const { return at<int>(L::sale); }
    __device__ __forceinline__ int* resq() const { return at<int>(L::resq); }
    __device__ __forceinline__ float* shrow() const { return at<float>(L::shrow); }
    __device__ __forceinline__ float* govrow() const { return at<float>(L::govrow); }
    __device__ __forceinline__ unsigned long long* misc() const { return at<unsigned long long>(L::misc); }  // [0] tax pool in 2^-20 coin
    __device__ __forceinline__ uint32_t* bk_cnt(int k) const { return at<uint32_t>(L::bk_cnt) + k * L::bk_cnt_words; }
    __device__ __forceinline__ double* bk_part(int k) const { return at<double>(L::bk_part) + k * (L::bk_warps * 3); }
    __device__ __forceinline__ uint32_t* spl(int k, uint32_t buf) const { return at<uint32_t>(L::blob + (ST ? S::spl : c.o_spl)) + (k * 2 + (int)buf) * L::bk_warps; }
    __device__ __forceinline__ uint32_t* spl_cur() const { return at<uint32_t>(L::blob + (ST ? S::spl : c.o_spl)) + L::bk_metrics * 2 * L::bk_warps; }
    // bucket keys: coin in key | cslot | anext, labor and income in a region of their own (or over the matched lists)
    __device__ __forceinline__ uint32_t* bk_keys(int k) const {
        return k == 0 ? at<uint32_t>(L::bk_keys) : at<uint32_t>(c.o_bk2) + (k - 1) * (L::bk_warps * L::bk_cap);
    }
    __device__ __forceinline__ uint32_t* ahead() const { return at<uint32_t>(ST ? S::ahead : c.o_ahead); }
    __device__ __forceinline__ uint32_t* mb() const { return at<uint32_t>(ST ? S::mb : c.o_mb); }
    __device__ __forceinline__ uint32_t* ma() const { return at<uint32_t>(ST ? S::ma : c.o_ma); }
    // book-cap path: this step's candidates binned by arrival key (G11, G15)
    __device__ __forceinline__ uint32_t* bbh() const { return at<uint32_t>(c.o_bbh); }    // [2R][BOOK_BINS] chain heads
    __device__ __forceinline__ uint32_t* bbc() const { return at<uint32_t>(c.o_bbc); }    // [2R][BOOK_BINS] counts -> exclusive prefix
    __device__ __forceinline__ uint32_t* lbh() const { return at<uint32_t>(c.o_lbh); }    // [levels][LEVEL_BINS] chain heads
    __device__ __forceinline__ uint32_t* lmask() const { return at<uint32_t>(c.o_lmask); }  // [levels] occupied level bins
    __device__ __forceinline__ uint32_t* cdf() const { return at<uint32_t>(ST ? S::cdf : c.o_cdf); }
    __device__ __forceinline__ float* stage() const { return at<float>(ST ? S::stage : c.o_stage); }
    __device__ __forceinline__ float* rowbuf() const { return at<float>(c.o_rowbuf); }  // [warps][8][D_pop]: unstaged observation rows
};

// f3, skill growth ("the respective skill is increased by 0.5%.  This 0.5% bonus shrinks as the agent
// approaches the maximum skill level of 5"; linear damping, G41): min(max, s + s * (rate * (1 - s / max))),
// every operation one correctly rounded binary32 operation.
__device__ __forceinline__ float progress_skill(float s, float rate, float mx) {
    const float room = __fsub_rn(1.0f, __fdiv_rn(s, mx));
    return fminf(__fadd_rn(s, __fmul_rn(s, __fmul_rn(rate, room))), mx);
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

// Coin term of Eq.1: (C^(1-eta) - 1) / (1-eta) in binary64, C >= 0 a binary32 value.
// C^a = exp(a ln C) with ln m = 2 atanh((m-1)/(m+1)) on m in [sqrt(1/2), sqrt 2) (7 terms:
// truncation < 5e-13 absolute) and a degree-11 Taylor polynomial of exp on |r| <= ln2 / 2
// (truncation < 7e-15 relative): relative error of C^a below 1e-12, four orders of magnitude
// inside what the reward tolerance needs; about 55 instructions, where
// the library pow() costs ~230.
__device__ __forceinline__ double coin_utility(float C, double a, double inv_a) {
    if (C == 0.0f) return -inv_a;  // G36
    const double x = (double)C;    // exact; normal in binary64 even for a subnormal C
    int hi = __double2hiint(x);
    int e = (hi >> 20) - 1023;
    hi = (hi & 0x000FFFFF) | 0x3FF00000;
    if (hi >= 0x3FF6A09F) { hi -= 0x00100000; e += 1; }  // m >= ~sqrt 2: halve
    const double m = __hiloint2double(hi, __double2loint(x));
    const double d = m + 1.0;
    double rc = (double)__frcp_rn((float)d);
    rc = fma(rc, fma(-d, rc, 1.0), rc);  // one Newton step: 1/d to ~4e-15
    const double s = (m - 1.0) * rc, z = s * s;
    double q = 1.0 / 13.0;
    q = fma(q, z, 1.0 / 11.0);
    q = fma(q, z, 1.0 / 9.0);
    q = fma(q, z, 1.0 / 7.0);
    q = fma(q, z, 1.0 / 5.0);
    q = fma(q, z, 1.0 / 3.0);
    q = fma(q, z, 1.0);
    const double lnC = fma((double)e, 0.6931471805599453094, 2.0 * s * q);
    const double tt = a * lnC;
    const double nn = rint(tt * 1.4426950408889634074);
    double r = fma(-nn, 0.693147180369123816490, tt);  // ln2 hi / lo (Cody-Waite)
    r = fma(-nn, 1.90821492927058770002e-10, r);
    double y = 1.0 / 39916800.0;
    y = fma(y, r, 1.0 / 3628800.0);
    y = fma(y, r, 1.0 / 362880.0);
    y = fma(y, r, 1.0 / 40320.0);
    y = fma(y, r, 1.0 / 5040.0);
    y = fma(y, r, 1.0 / 720.0);
    y = fma(y, r, 1.0 / 120.0);
    y = fma(y, r, 1.0 / 24.0);
    y = fma(y, r, 1.0 / 6.0);
    y = fma(y, r, 0.5);
    y = fma(y, r, 1.0);
    y = fma(y, r, 1.0);
    const int n = (int)nn;  // |n| <= ~190: the scaled result stays normal
    y = __hiloint2double(__double2hiint(y) + (n << 20), __double2loint(y));
    return (y - 1.0) * inv_a;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
    return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = __fadd_rn(v, __shfl_xor_sync(FULL, v, o));
    return v;
}

// Bitonic sorting network over 32*EPL values held by one warp in BLOCKED layout, element
// idx = lane*EPL + q, ascending in idx.  Strides below EPL exchange registers of one lane,
// strides of EPL and more are warp shuffles: 15 shuffle stages at EPL = 4 where the striped
// layout (idx = q*32 + lane) needs 25.  Fully unrolled: a looped version (~80 instead of ~400
// instructions of footprint) was measured 5 % slower end to end.  No barriers.
template <int EPL>
__device__ __forceinline__ void warp_sort(float (&x)[EPL], int lane) {
    // levels inside one lane's block with compile-time directions (k < EPL)
#pragma unroll
    for (int k = 2; k < EPL; k <<= 1) {
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
#pragma unroll
            for (int q = 0; q < EPL; ++q) {
                if ((q & j) == 0) {
                    const float lo = fminf(x[q], x[q | j]), hi = fmaxf(x[q], x[q | j]);
                    const bool up = (q & k) == 0;
                    x[q] = up ? lo : hi;
                    x[q | j] = up ? hi : lo;
                }
            }
        }
    }
#pragma unroll
    for (int k = (EPL > 2 ? EPL : 2); k <= 32 * EPL; k <<= 1) {
        const bool up = ((lane * EPL) & k) == 0;  // k = 32*EPL: always ascending
#pragma unroll
        for (int jl = k / (2 * EPL); jl > 0; jl >>= 1) {  // partner in lane ^ jl, same q
            const bool keep_min = ((lane & jl) == 0) == up;
#pragma unroll
            for (int q = 0; q < EPL; ++q) {
                const float y = __shfl_xor_sync(FULL, x[q], jl);
                x[q] = keep_min ? fminf(x[q], y) : fmaxf(x[q], y);
            }
        }
#pragma unroll
        for (int j = EPL >> 1; j > 0; j >>= 1) {  // partner in the same lane
#pragma unroll
            for (int q = 0; q < EPL; ++q) {
                if ((q & j) == 0) {
                    const float lo = fminf(x[q], x[q | j]), hi = fmaxf(x[q], x[q | j]);
                    x[q] = up ? lo : hi;
                    x[q | j] = up ? hi : lo;
                }
            }
        }
    }
}

// Element of rank `rank` (0-based) of a sorted warp-held array (blocked layout).
template <int EPL>
__device__ __forceinline__ float warp_pick(const float (&x)[EPL], int rank) {
    const int q = rank & (EPL - 1);
    float v = x[0];
#pragma unroll
    for (int qq = 1; qq < EPL; ++qq) v = (q == qq) ? x[qq] : v;
    return __shfl_sync(FULL, v, rank / EPL);
}

// Order statistics r0 <= r1 <= r0 + 1 of the N non-negative values a warp holds (pads = +inf),
// by walking from a pivot: the previous step's lower median.  With c_lt = #{x < p} and
// c_le = #{x <= p}, p is the statistic of rank r exactly when c_lt <= r < c_le; otherwise the
// pivot moves to the next distinct value below (above).  Medians drift by 1-2 distinct values
// per step on the paper-shaped workloads, so this costs ~100 instructions
// where the sorting network costs ~450.  Exact for any pivot; gives up (returns false, caller
// sorts) after WALK_MAX moves or if a value has its sign bit set (keys would not be monotone).
constexpr int WALK_MAX = 8;
template <int EPL>
__device__ __forceinline__ bool walk_select(const uint32_t (&key)[EPL], int lane, int r0, int r1, uint32_t* pivot, uint32_t& lo,
                                            uint32_t& hi) {
    uint32_t any = 0;
#pragma unroll
    for (int q = 0; q < EPL; ++q) any |= key[q];
    if (__reduce_or_sync(FULL, any) & 0x80000000u) return false;
    uint32_t p = *pivot;
    int a = 0, b = 0;
#pragma unroll
    for (int q = 0; q < EPL; ++q) { a += key[q] < p; b += key[q] <= p; }
    int c_lt = __reduce_add_sync(FULL, a), c_le = __reduce_add_sync(FULL, b);
    int moves = 0;
    while (r0 < c_lt) {  // the statistic is below the pivot
        if (++moves > WALK_MAX) return false;
        uint32_t mx = 0;
#pragma unroll
        for (int q = 0; q < EPL; ++q) mx = max(mx, key[q] < p ? key[q] : 0u);
        p = __reduce_max_sync(FULL, mx);
        a = 0;
#pragma unroll
        for (int q = 0; q < EPL; ++q) a += key[q] < p;
        c_le = c_lt;
        c_lt = __reduce_add_sync(FULL, a);
    }
    while (r0 >= c_le) {  // above the pivot
        if (++moves > WALK_MAX) return false;
        uint32_t mn = 0xFFFFFFFFu;
#pragma unroll
        for (int q = 0; q < EPL; ++q) mn = min(mn, key[q] > p ? key[q] : 0xFFFFFFFFu);
        p = __reduce_min_sync(FULL, mn);
        b = 0;
#pragma unroll
        for (int q = 0; q < EPL; ++q) b += key[q] <= p;
        c_lt = c_le;
        c_le = __reduce_add_sync(FULL, b);
    }
    uint32_t p1 = p;
    if (r1 >= c_le) {
        uint32_t mn = 0xFFFFFFFFu;
#pragma unroll
        for (int q = 0; q < EPL; ++q) mn = min(mn, key[q] > p ? key[q] : 0xFFFFFFFFu);
        p1 = __reduce_min_sync(FULL, mn);
    }
    if (lane == 0) *pivot = p;
    lo = p;
    hi = p1;
    return true;
}

// The same two order statistics without a hint, by bitwise search on the keys (31 counting
// rounds in a loop of a dozen instructions): the rarely taken fall-back of the integer metrics.
template <int EPL>
__device__ __forceinline__ void bit_select(const uint32_t (&key)[EPL], int r0, int r1, uint32_t& lo, uint32_t& hi) {
    uint32_t res = 0;
#pragma unroll 1
    for (int bit = 30; bit >= 0; --bit) {  // largest res with #{x < res} <= r0 = the statistic of rank r0
        const uint32_t cand = res | (1u << bit);
        int a = 0;
#pragma unroll
        for (int q = 0; q < EPL; ++q) a += key[q] < cand;
        if (__reduce_add_sync(FULL, a) <= r0) res = cand;
    }
    int b = 0;
    uint32_t mn = 0xFFFFFFFFu;
#pragma unroll
    for (int q = 0; q < EPL; ++q) { b += key[q] <= res; mn = min(mn, key[q] > res ? key[q] : 0xFFFFFFFFu); }
    lo = res;
    hi = r1 >= __reduce_add_sync(FULL, b) ? __reduce_min_sync(FULL, mn) : res;
}

template <int NP, int NT, class SM>
__device__ __forceinline__ void gov_triple(const DevCfg& c, const SM& m, int k, double mean, double var, float lo, float hi,
                                           float scale) {
    const int N = NT > 0 ? NT : c.N;
    const float sd = __fsqrt_rn((float)var);
    const float med = (N & 1) ? hi : __fmul_rn(0.5f, __fadd_rn(lo, hi));
    m.govrow()[3 * k + 0] = (float)(mean * (double)scale);
    m.govrow()[3 * k + 1] = __fmul_rn(sd, scale);
    m.govrow()[3 * k + 2] = __fmul_rn(med, scale);
}

// One warp computes mean, std, median (Fig.1, G26) of FLOAT metric k (0 coin,
// 1 labor, 2 income); for coin also the welfare u_g = eq * prod (Eq.3-5; G22, G23)
// and the government reward.  Sum in binary64; squared deviations in binary32 (non-negative
// terms: relative error < 1e-6).  Median: labor and income walk from last step's median (the
// sorting network when the walk gives up), coin is sorted (the order also gives gini).  ONE
// instance of this code per kernel (the caller loops over k without unrolling): the unrolled
// network is most of the kernel's instruction footprint.
//   mode 0 = step, 1 = finished env (reward 0), 2 = observe only
template <int EPL, int NS, int NT, class SM>
__device__ __forceinline__ void metric_stats(const DevCfg& c, const SM& m, int k, int lane, int mode, int e, float* rew) {
    const int N = NT > 0 ? NT : c.N;  // NT > 0: population size known at compile time
    const double inv_n = NT > 0 ? 1.0 / (double)(NT > 0 ? NT : 1) : c.inv_n;
    const float* farr = k == 0 ? m.coin() : k == 1 ? m.labor() : m.income();
    float x[EPL];
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < EPL; ++q) {
        const int idx = lane * EPL + q;  // blocked layout (warp_sort)
        const float v = farr[idx < N ? idx : 0];
        x[q] = idx < N ? v : INFINITY;
        s += idx < N ? (double)v : 0.0;
    }
    s = warp_sum(s);
    const double mean = s * inv_n;
    float qs = 0.0f;
#pragma unroll
    for (int q = 0; q < EPL; ++q) {
        const float d = (lane * EPL + q) < N ? (float)((double)x[q] - mean) : 0.0f;
        qs = __fadd_rn(qs, __fmul_rn(d, d));
    }
    qs = warp_sum(qs);
    float lo, hi;
    const int r0 = N >= 2 ? (N >> 1) - 1 : 0, r1 = N >> 1;
    bool found = false;
    if (k != 0 && k >= SM::L::bk_metrics) {  // labor, income (when not bucketed): med_prev holds last step's lower median
        uint32_t key[EPL], klo, khi;
#pragma unroll
        for (int q = 0; q < EPL; ++q) key[q] = __float_as_uint(x[q]);
        found = walk_select<EPL>(key, lane, r0, r1, &m.hdr()->med_prev[k - 1], klo, khi);
        lo = __uint_as_float(klo);
        hi = __uint_as_float(khi);
    }
    if (!found) {
        warp_sort<EPL>(x, lane);
        lo = warp_pick<EPL>(x, r0);
        hi = warp_pick<EPL>(x, r1);
        if (k != 0 && lane == 0) m.hdr()->med_prev[k - 1] = __float_as_uint(lo);
        if (k < SM::L::bk_metrics) {  // EPL = warps of the CTA: renew this metric's bucket bounds of the block-wide sort
            const uint32_t nxt = (*m.spl_cur() & 1u) ^ 1u;
#pragma unroll 1
            for (int b = 0; b + 1 < EPL; ++b) {
                const float v = warp_pick<EPL>(x, ((b + 1) * N) / EPL);
                if (lane == 0) m.spl(k, nxt)[b] = __float_as_uint(v);
            }
        }
        if (k == 0 && mode != 2) {
            // sum_i sum_j |c_i - c_j| = 2 sum_k (2k - N + 1) c_(k)  =>  gini * prod = gn / N   (G23)
            double g = 0.0;
#pragma unroll
            for (int q = 0; q < EPL; ++q) {
                const int idx = lane * EPL + q;
                g += idx < N ? (double)(2 * idx - N + 1) * (double)x[q] : 0.0;
            }
            g = warp_sum(g);
            if (lane == 0) {
                // u_g = (omega (1 - gini) + (1 - omega)) prod = prod - omega * gini * prod; gini = 0 when
                // prod = 0 or N = 1 (then gn = 0 as well)
                const double ug = s - (double)c.omega * (g * inv_n);
                if (mode == 0) {
                    if (rew) rew[(uint32_t)(e * (N + 1) + N)] = (float)(ug - m.hdr()->u_g_prev);
                    m.hdr()->u_g_prev = ug;
                } else if (rew) {
                    rew[(uint32_t)(e * (N + 1) + N)] = 0.0f;
                }
            }
        }
    }
    if (lane == 0) gov_triple<NS, NT>(c, m, k, mean, (double)qs * inv_n, lo, hi, k == 1 ? c.s_labor : c.s_coin);
}

// The same triple for the INTEGER metric "inventory of resource r" (metric 3 + r).  Sum and
// sum of squares are exact integers (REDUX), so mean and variance (N sum x^2 - (sum x)^2) / N^2
// need no second pass; the median walks from last step's value on the integer keys, with the
// bitwise search as fall-back.
template <int EPL, int NS, int NT, class SM>
__device__ __forceinline__ void int_metric_stats(const DevCfg& c, const SM& m, int r, int lane) {
    const int N = NT > 0 ? NT : c.N;
    const double inv_n = NT > 0 ? 1.0 / (double)(NT > 0 ? NT : 1) : c.inv_n;
    const int* iarr = m.inv() + r * NS;
    uint32_t key[EPL];
    int si = 0, mx = 0;
    uint32_t sq = 0;
#pragma unroll
    for (int q = 0; q < EPL; ++q) {
        const int idx = lane * EPL + q;
        const int v = iarr[idx < N ? idx : 0];
        key[q] = idx < N ? (uint32_t)v : 0x7FFFFFFFu;  // pads sort last; a negative value makes the walk give up
        si += idx < N ? v : 0;
        mx = max(mx, idx < N ? (v < 0 ? 0x7FFFFFFF : v) : 0);
        sq += idx < N ? (uint32_t)(v * v) : 0u;
    }
    const long long sum = (long long)__reduce_add_sync(FULL, si);
    unsigned long long sum2;
    if (EPL <= 8 && __reduce_max_sync(FULL, mx) < 4096) {  // 32 x EPL x 4096^2 <= 2^32 - 1 for EPL <= 8
        sum2 = (unsigned long long)__reduce_add_sync(FULL, sq);
    } else {
        unsigned long long w = 0;
#pragma unroll
        for (int q = 0; q < EPL; ++q) {
            const long long v = (lane * EPL + q) < N ? (long long)(int)key[q] : 0ll;
            w += (unsigned long long)(v * v);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(FULL, w, o);
        sum2 = w;
    }
    const double mean = (double)sum * inv_n;
    const double var = (double)((long long)N * (long long)sum2 - sum * sum) * inv_n * inv_n;
    const int r0 = N >= 2 ? (N >> 1) - 1 : 0, r1 = N >> 1;
    uint32_t klo, khi;
    if (!walk_select<EPL>(key, lane, r0, r1, &m.hdr()->med_prev[2 + r], klo, khi)) {
        bit_select<EPL>(key, r0, r1, klo, khi);
        if (lane == 0) m.hdr()->med_prev[2 + r] = klo;
    }
    if (lane == 0) gov_triple<NS, NT>(c, m, 3 + r, mean, var, (float)(int)klo, (float)(int)khi, c.s_count);
}

// ---- block-wide statistics of the float metrics of large populations (CTAs of 512 / 1024 threads) ----
// Coin, labor and income need order statistics (the median; coin also gini in its sorted-rank form, G23).  One warp
// holding all N values of a metric in registers was the longest branch of the N = 1000 step: 20,000 of its 56,000
// cycles went by waiting for those three warps (profiles/r2c).  Here every warp sorts one BUCKET per metric: bucket b
// holds the values strictly between the bounds spl[b-1] and spl[b], the bounds being last step's order statistics
// of rank (b+1) N / NW (the metrics drift slowly, so a bucket stays near N / NW values).  Values EQUAL to a bound are
// only counted (they need no sorting), which keeps large groups of equal values -- every income 0 after a tax
// collection, many agents on the same coin -- out of the buckets.  Rank of a value = sizes of the lower buckets and
// bound groups + its place in its bucket.  Exact for any bounds; if a bucket overflows (start of an episode, a
// redistribution) that metric falls back to the single-warp sort, which also renews its bounds.

// Thread `tid` files the final value x of metric k of its agent; called before the barrier that ends the state update.
template <int NPAD, class SM>
__device__ __forceinline__ void bucket_fill(const SM& m, int k, float x) {
    constexpr int NW = NPAD / 32, CAP = SM::L::bk_cap;
    const uint32_t key = __float_as_uint(x);
    const uint32_t* spl = m.spl(k, *m.spl_cur() & 1u);
    int lo = 0, hi = NW - 1;  // bucket = number of bounds <= key
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (key < spl[mid]) hi = mid;
        else lo = mid + 1;
    }
    uint32_t* cnt = m.bk_cnt(k);
    if (lo > 0 && spl[lo - 1] == key) {
        atomicAdd(&cnt[NW + lo - 1], 1u);  // equal to bound lo-1 (the last of equal bounds): counted, not stored
    } else {
        const uint32_t pos = atomicAdd(&cnt[lo], 1u);
        if (pos < (uint32_t)CAP && !(key >> 31)) m.bk_keys(k)[lo * CAP + (int)pos] = key;
        else cnt[2 * NW] = 1u;  // overflow (or a negative value): fall back
    }
}
template <int NPAD, class SM>
__device__ __forceinline__ void bucket_fill_all(const SM& m, int tid, bool act) {
    if (!act) return;
    bucket_fill<NPAD>(m, 0, m.coin()[tid]);
    if (SM::L::bk_metrics > 1) {
        bucket_fill<NPAD>(m, 1, m.labor()[tid]);
        bucket_fill<NPAD>(m, 2, m.income()[tid]);
    }
}

// Warp `warp` sorts its bucket of metric k (n <= 32 EPL values, blocked layout), followed in rank order by the ne
// values equal to its upper bound v; leaves its share of (gini,) sum and sum of squares; the warp that holds a wanted
// rank writes that order statistic (the two medians, next step's bounds).
template <int EPL, int NPAD, class SM>
__device__ __forceinline__ void bucket_sort(const SM& m, int k, int warp, int lane, int n, int ne, int off, int N) {
    constexpr int NW = NPAD / 32, CAP = SM::L::bk_cap;
    const uint32_t cur = *m.spl_cur() & 1u;
    const float v_eq = __uint_as_float(m.spl(k, cur)[warp < NW - 1 ? warp : 0]);  // ne = 0 for the last warp
    float x[EPL];
#pragma unroll
    for (int q = 0; q < EPL; ++q) {
        const int idx = lane * EPL + q;
        x[q] = idx < n ? __uint_as_float(m.bk_keys(k)[warp * CAP + idx]) : INFINITY;
    }
    warp_sort<EPL>(x, lane);
    double g = 0.0, s1 = 0.0, s2 = 0.0;
#pragma unroll
    for (int q = 0; q < EPL; ++q) {
        const int idx = lane * EPL + q;
        const double v = idx < n ? (double)x[q] : 0.0;
        if (k == 0) g += (double)(2 * (off + idx) - N + 1) * v;  // sum_j (2j - N + 1) c_(j)  (G23)
        s1 += v;
        s2 += v * v;
    }
    if (k == 0) g = warp_sum(g);
    s1 = warp_sum(s1);
    s2 = warp_sum(s2);
    if (lane == 0) {
        if (ne > 0) {  // ranks off+n .. off+n+ne-1 all hold v_eq
            const double v = (double)v_eq, o = (double)(off + n), c = (double)ne;
            g += v * (c * (2.0 * o - (double)N + 1.0) + c * (c - 1.0));
            s1 += c * v;
            s2 += c * v * v;
        }
        double* part = m.bk_part(k) + warp * 3;
        part[0] = g; part[1] = s1; part[2] = s2;
    }
    // order statistics held by this warp: lane b < NW - 1 looks for next step's bound of rank (b+1) N / NW
    {
        const int want = lane < NW - 1 ? ((lane + 1) * N) / NW - off : -1;
        const bool mine = want >= 0 && want < n + ne;
        const int src = (mine && want < n) ? want : 0;
        float v = __shfl_sync(FULL, x[0], src / EPL);
#pragma unroll
        for (int q = 1; q < EPL; ++q) {
            const float y = __shfl_sync(FULL, x[q], src / EPL);
            v = (src % EPL) == q ? y : v;
        }
        if (mine) m.spl(k, cur ^ 1u)[lane] = __float_as_uint(want < n ? v : v_eq);
    }
    const int r0 = (N >= 2 ? (N >> 1) - 1 : 0) - off, r1 = (N >> 1) - off;
    if (r0 >= 0 && r0 < n + ne) { const float v = r0 < n ? warp_pick<EPL>(x, r0) : v_eq; if (lane == 0) m.bk_cnt(k)[2 * NW + 1] = __float_as_uint(v); }
    if (r1 >= 0 && r1 < n + ne) { const float v = r1 < n ? warp_pick<EPL>(x, r1) : v_eq; if (lane == 0) m.bk_cnt(k)[2 * NW + 2] = __float_as_uint(v); }
}

// All warps: sort the own bucket of metric k.  Nothing to do if the buckets overflowed (the caller falls back).
template <int NPAD, class SM>
__device__ __forceinline__ void bucket_stats(const SM& m, int k, int warp, int lane, int N) {
    constexpr int NW = NPAD / 32;
    const uint32_t* cnt = m.bk_cnt(k);
    if (cnt[2 * NW]) return;
    const int nb = lane < NW ? (int)cnt[lane] : 0, neq = lane < NW - 1 ? (int)cnt[NW + lane] : 0;
    int incl = nb + neq;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(FULL, incl, o);
        if (lane >= o) incl += y;
    }
    const int n = __shfl_sync(FULL, nb, warp), ne = __shfl_sync(FULL, neq, warp), off = __shfl_sync(FULL, incl - nb - neq, warp);
    if (n <= 32) bucket_sort<1, NPAD>(m, k, warp, lane, n, ne, off, N);
    else if (n <= 64) bucket_sort<2, NPAD>(m, k, warp, lane, n, ne, off, N);
    else bucket_sort<4, NPAD>(m, k, warp, lane, n, ne, off, N);
}

// Shared tail of the population rows: market statistics of the post-step books.
template <int PT, class SM>
__device__ __forceinline__ void write_market_row(const DevCfg& c, const SM& m, int r, const int* cnt) {
    const int P = PT > 0 ? PT : c.P;
    int best_bid = 0, best_ask = 0, nb = 0, na = 0;
    for (int p = 0; p < P; ++p) {
        const int cb = cnt[(r * 2 + 0) * P + p], ca = cnt[(r * 2 + 1) * P + p];
        nb += cb;
        na += ca;
        if (cb > 0) best_bid = c.prices[p];
        if (ca > 0 && best_ask == 0) best_ask = c.prices[p];
    }
    float* o = m.shrow() + r * 5;
    o[0] = __fmul_rn((float)best_bid, c.s_price);
    o[1] = __fmul_rn((float)best_ask, c.s_price);
    o[2] = __fmul_rn((float)nb, c.s_count);
    o[3] = __fmul_rn((float)na, c.s_count);
    o[4] = __fmul_rn((float)m.hdr()->last_price[r], c.s_price);
}
template <class SM>
__device__ __forceinline__ void write_timers(const DevCfg& c, const SM& m, int tq, int tq_in_period) {
    m.shrow()[5 * c.R + c.B] = __fdiv_rn((float)tq_in_period, (float)c.period);
    m.shrow()[5 * c.R + c.B + 1] = __fdiv_rn((float)tq, (float)c.T);
}

// Rewards, government statistics and both observation blocks of the state in shared memory.
// Called after a block barrier that made the state (and m.shrow()) final.
//   mode     0 = step, 1 = finished env (rewards 0), 2 = observe only
//   rows     0 = rewrite only the columns that change every step, 1 = also the tax rates,
//            2 = every column (first step of a launch, every step under skill growth: skills)
//   FX       f2, factored observations: the staging tile holds only the 3R + 4 agent-private columns
//            (-> priv), the env-wide tail leaves once per env from m.shrow() (-> shared), the
//            government row goes to govp
template <int NPAD, int NS, int RT, int NT, int BT, int PF, int FX, class SM>
__device__ void outputs(const DevCfg& c, const SM& m, int tid, int e, int mode, int rows, float coin_pre, float labor_pre,
                        double cf_pre, float* obs, float* rew, float* priv = nullptr, float* shared = nullptr, float* govp = nullptr) {
    constexpr int NW = NPAD / 32, EPL = NPAD / 32;
    // RT, NT, BT > 0: resource count, population size, bracket count known at compile time
    const int N = NT > 0 ? NT : c.N, R = RT > 0 ? RT : c.R, B = BT > 0 ? BT : c.B;
    const int D_pop = (RT > 0 && BT > 0) ? 6 + 8 * RT + BT : c.D_pop;
    constexpr int N4 = NS;  // stride of the per-agent arrays
    const bool act = tid < N;
    const int lane = tid & 31, warp = tid >> 5;
    const bool staged = FX ? priv != nullptr : ((PF || c.stage_obs) && obs);
    const bool any_obs = FX ? (priv != nullptr || govp != nullptr) : obs != nullptr;
    const int DP = FX ? 3 * R + 4 : D_pop;  // row stride of the staging tile
    const int stage_alias_bytes = PF ? 2 * R * NS * 4 : c.stage_alias_bytes, n_metrics = RT > 0 ? 3 + RT : c.n_metrics;

    if (act) {
        const float coin = m.coin()[tid], labor = m.labor()[tid];
        // ---- population reward: u(post) - u(pre), u = coin term - labor (Eq.1-2) ----
        if (mode == 0) {
            double cf_post = cf_pre;
            if (__float_as_uint(coin) != __float_as_uint(coin_pre)) {
                cf_post = coin_utility(coin, c.ua, c.inv_ua);
                m.cf()[tid] = cf_post;
            }
            if (rew) rew[(uint32_t)(e * (N + 1) + tid)] = (float)((cf_post - (double)labor) - (cf_pre - (double)labor_pre));
        } else if (mode == 1 && rew) {
            rew[(uint32_t)(e * (N + 1) + tid)] = 0.0f;
        }
        // ---- this agent's observation row (G25) in the staging tile ----
        if (staged) {
            float* o = m.stage() + tid * DP;
            o[0] = __fmul_rn(coin, c.s_coin);
            for (int r = 0; r < R; ++r) o[1 + r] = __fmul_rn((float)m.inv()[r * N4 + tid], c.s_count);
            o[R + 1] = __fmul_rn((float)m.esc_coin()[tid], c.s_coin);
            for (int r = 0; r < R; ++r) o[R + 2 + r] = __fmul_rn((float)m.esc_res()[r * N4 + tid], c.s_count);
            o[3 * R + 3] = __fmul_rn(labor, c.s_labor);
            // rows whose bytes the matched-order lists reuse are rewritten in full every step
            const int rows_eff = (tid * DP * 4 < stage_alias_bytes) ? 2 : rows;
            if (!FX) {
                float* tl = o + 3 * R + 4;
                for (int k = 0; k < 5 * R; ++k) tl[k] = m.shrow()[k];
                tl[5 * R + B] = m.shrow()[5 * R + B];
                tl[5 * R + B + 1] = m.shrow()[5 * R + B + 1];
                if (rows_eff >= 1)
                    for (int b = 0; b < B; ++b) tl[5 * R + b] = m.shrow()[5 * R + b];
            }
            if (rows_eff >= 2) {
                for (int r = 0; r < R; ++r) o[2 * R + 2 + r] = m.SG()[r * N4 + tid];
                o[3 * R + 2] = m.SC()[tid];
            }
        }
    }

    // ---- government statistics: metric k is owned by one warp (floats from warp 0 up, integer
    // metrics from the last warp down) ----
    constexpr bool BKT = SM::L::bucketed;  // coin (large CTAs: labor and income too): every warp sorts one bucket per metric, filled before the caller's barrier
    constexpr int BKM = SM::L::bk_metrics, BKF = 2 * SM::L::bk_warps;  // bucketed metrics; index of a metric's overflow flag
    bool fell_back = false;  // some metric's buckets overflowed (the same answer in every thread)
    if (BKT) {
#pragma unroll 1
        for (int k = 0; k < BKM; ++k) {
            fell_back = fell_back || m.bk_cnt(k)[BKF] != 0u;
            bucket_stats<NPAD>(m, k, warp, lane, N);
        }
    }
#pragma unroll 1
    for (int k = BKM + warp; k < 3; k += NW) metric_stats<EPL, NS, NT>(c, m, k, lane, mode, e, rew);
#pragma unroll 1
    // integer metrics: from the last warp down; in bucketed kernels from warp 0 up (their last warp closes the float
    // metrics after the barrier and has the fewest observation rows to write)
    for (int r = BKT ? warp : NW - 1 - warp; r < R; r += NW) int_metric_stats<EPL, NS, NT>(c, m, r, lane);
    if (tid < B + 2) m.govrow()[3 * n_metrics + tid] = m.shrow()[5 * R + tid];  // B + 2 <= 18 < NPAD

    if (any_obs) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    EJ_MARK(6);
    __syncthreads();
    EJ_MARK(7);

    constexpr int CLOSER = BKT ? NW - 1 : 0;  // warp that closes the statistics and issues the bulk stores
    if (BKT && warp == CLOSER) {  // the three triples and the welfare from the buckets' shares (or the single-warp sort)
#pragma unroll 1
        for (int k = 0; k < BKM; ++k) {
            uint32_t* cnt = m.bk_cnt(k);
            if (!cnt[BKF]) {
                double g = 0.0, s1 = 0.0, s2 = 0.0;
                if (lane < NW) { const double* part = m.bk_part(k) + lane * 3; g = part[0]; s1 = part[1]; s2 = part[2]; }
                g = warp_sum(g); s1 = warp_sum(s1); s2 = warp_sum(s2);
                if (lane == 0) {
                    const double inv_n = NT > 0 ? 1.0 / (double)(NT > 0 ? NT : 1) : c.inv_n;
                    const double mean = s1 * inv_n;
                    double var = (s2 - s1 * mean) * inv_n;  // population variance from sum and sum of squares (binary64)
                    if (var < 0.0) var = 0.0;
                    gov_triple<NS, NT>(c, m, k, mean, var, __uint_as_float(cnt[BKF + 1]), __uint_as_float(cnt[BKF + 2]), k == 1 ? c.s_labor : c.s_coin);
                    if (k == 0 && mode != 2) {
                        const double ug = s1 - (double)c.omega * (g * inv_n);  // Eq.3-5 as in metric_stats
                        if (mode == 0) {
                            if (rew) rew[(uint32_t)(e * (N + 1) + N)] = (float)(ug - m.hdr()->u_g_prev);
                            m.hdr()->u_g_prev = ug;
                        } else if (rew) {
                            rew[(uint32_t)(e * (N + 1) + N)] = 0.0f;
                        }
                    }
                }
            } else {
                metric_stats<EPL, NS, NT>(c, m, k, lane, mode, e, rew);
            }
            __syncwarp();
            for (int i = lane; i < SM::L::bk_cnt_words; i += 32) cnt[i] = 0u;  // empty buckets for the next step
        }
        if (lane == 0) *m.spl_cur() ^= 1u;  // the bounds written during this step are in force from now on
        __syncwarp();
        if (any_obs) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
    }
    if (BKT && fell_back) __syncthreads();  // the single-warp sort read the agents' state: nobody may start the next step before it is done

    if (any_obs && tid == CLOSER * 32) {  // bulk stores: the env's contiguous tile, (f2) its env-wide tail, its government row
        if (staged) {
            float* dst = FX ? priv + (uint32_t)(e * N * DP) : obs + (uint32_t)(e * N * D_pop);
            const uint32_t src = (uint32_t)__cvta_generic_to_shared(m.stage());
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(N * DP * 4) : "memory");
        }
        if (FX && shared) {
            const int dsp = (5 * R + B + 2 + 3) & ~3;
            float* sdst = shared + (uint32_t)(e * dsp);
            const uint32_t ssrc = (uint32_t)__cvta_generic_to_shared(m.shrow());
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(sdst), "r"(ssrc), "r"(dsp * 4) : "memory");
        }
        float* gdst = FX ? (govp ? govp + (uint32_t)(e * c.D_gov_pad) : nullptr)
                         : obs + (uint32_t)((uint32_t)c.gov_obs_offset + (uint32_t)(e * c.D_gov_pad));
        if (gdst) {
            const uint32_t gsrc = (uint32_t)__cvta_generic_to_shared(m.govrow());
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(gsrc), "r"(c.D_gov_pad * 4) : "memory");
        }
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    // ---- population rows when the env's tile does not fit in shared memory: every warp sends its 32 rows in chunks
    // of 8 through a private row-major buffer (odd row length: the 8 writers hit distinct banks), then copies the
    // chunk out with 128-bit coalesced stores.  The env-wide tail of the 8 buffer rows is written once per step.
    if (!FX && obs && !staged) {
        const int D = D_pop, npriv = 3 * R + 4;
        float* buf = m.rowbuf() + warp * (8 * D);
        float* dst = obs + (size_t)e * (size_t)(N * D);
        for (int r = 0; r < 8; ++r)
            for (int k = lane; k < D - npriv; k += 32) buf[r * D + npriv + k] = m.shrow()[k];
        const bool vec = (((size_t)N * (size_t)D) & 3u) == 0 && ((8 * D) & 3) == 0;  // 16-byte aligned chunks
#pragma unroll 1
        for (int ch = 0; ch < 4; ++ch) {
            const int row0 = warp * 32 + ch * 8;
            if (row0 >= N) break;
            if ((lane >> 3) == ch && act) {
                float* o = buf + (lane & 7) * D;
                o[0] = __fmul_rn(m.coin()[tid], c.s_coin);
                for (int r = 0; r < R; ++r) o[1 + r] = __fmul_rn((float)m.inv()[r * N4 + tid], c.s_count);
                o[R + 1] = __fmul_rn((float)m.esc_coin()[tid], c.s_coin);
                for (int r = 0; r < R; ++r) o[R + 2 + r] = __fmul_rn((float)m.esc_res()[r * N4 + tid], c.s_count);
                for (int r = 0; r < R; ++r) o[2 * R + 2 + r] = m.SG()[r * N4 + tid];
                o[3 * R + 2] = m.SC()[tid];
                o[3 * R + 3] = __fmul_rn(m.labor()[tid], c.s_labor);
            }
            __syncwarp();
            const int rows = N - row0 < 8 ? N - row0 : 8, n = rows * D;
            float* out = dst + row0 * D;
            if (vec && rows == 8) {
                for (int j = lane; j < n / 4; j += 32) reinterpret_cast<float4*>(out)[j] = reinterpret_cast<const float4*>(buf)[j];
            } else {
                for (int j = lane; j < n; j += 32) out[j] = buf[j];
            }
            __syncwarp();
        }
    }
}

// f1 masked sampling, the table generator.  Out of line: the unmasked hot path
// keeps its registers and instruction footprint.
template <int NS, class SM>
__device__ __noinline__ int masked_draw(const DevCfg& c, const SM& m, int tid, uint32_t x0, int R, int P, int M, int craft_mode,
                            int craft_units, int craft_distinct, int base_buy, int base_sell, int A) {
    constexpr int N4 = NS;
    // f1: the table restricted to this agent's available actions, renormalised with
    // integer weights w_a = cdf[a] - cdf[a-1]: target = floor(x0 S / 2^32), S = sum of available
    // w_a; action = first available a whose running sum exceeds target (first available if S = 0)
    const float coin = m.coin()[tid];
    const bool room = __popc(m.mask()[tid]) < M;
    bool craft_ok = false;
    if (craft_mode != EJ_CRAFT_PER_RESOURCE) {
        int enough = 0;
        for (int r = 0; r < R; ++r) enough += m.inv()[r * N4 + tid] >= craft_units;
        craft_ok = enough >= craft_distinct;
    }
    const int end_sell = base_sell + R * P;
    unsigned long long S = 0, run = 0, target = 0;
    int pick = -1, first_ok = -1;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        uint32_t prev = 0;
#pragma unroll 1
        for (int k = 0; k < A && pick < 0; ++k) {
            const unsigned long long hi = k == A - 1 ? (1ull << 32) : (unsigned long long)m.cdf()[k];
            const unsigned long long w = hi - (unsigned long long)prev;
            prev = (uint32_t)hi;
            bool ok = true;
            if (k >= R && k < base_buy) {
                ok = craft_mode == EJ_CRAFT_PER_RESOURCE ? m.inv()[(k - R) * N4 + tid] >= craft_units : craft_ok;
            } else if (k >= base_buy && k < base_sell) {
                const int j = k - base_buy, rr = (j * c.recipP) >> 16;
                ok = room && coin >= (float)c.prices[j - rr * P];
            } else if (k >= base_sell && k < end_sell) {
                ok = room && m.inv()[(((k - base_sell) * c.recipP) >> 16) * N4 + tid] >= 1;
            }
            if (!ok) continue;
            if (pass == 0) {
                S += w;
                if (first_ok < 0) first_ok = k;
            } else {
                run += w;
                if (run > target) pick = k;
            }
        }
        target = ((unsigned long long)x0 * S) >> 32;  // S <= 2^32: no overflow
    }
    return pick >= 0 ? pick : first_ok;
}

// Inputs and outputs of step `s` of a launch (ring slot `slot`), resolved where they are used:
// keeping seven running pointers alive in every thread cost ~6 % of the executed instructions.
struct StepPtrs {
    // element offsets are 32-bit (the host rejects rings / action streams of 2^32 elements or more)
    const StepIO& io;
    const DevCfg& c;
    int s, slot;
    __device__ __forceinline__ const int32_t* actions() const { return io.actions ? io.actions + (uint32_t)s * (uint32_t)(c.E * c.N) : nullptr; }
    __device__ __forceinline__ const int32_t* gov_actions() const { return io.gov_actions ? io.gov_actions + (uint32_t)s * (uint32_t)(c.E * c.B) : nullptr; }
    __device__ __forceinline__ float* obs() const { return io.obs ? io.obs + (uint32_t)slot * (uint32_t)c.obs_floats : nullptr; }
    __device__ __forceinline__ float* priv() const { return io.obs_priv ? io.obs_priv + (uint32_t)slot * (uint32_t)(c.E * c.N * (3 * c.R + 4)) : nullptr; }
    __device__ __forceinline__ float* shared() const { return io.obs_shared ? io.obs_shared + (uint32_t)slot * (uint32_t)(c.E * ((5 * c.R + c.B + 2 + 3) & ~3)) : nullptr; }
    __device__ __forceinline__ float* govp() const { return io.obs_gov ? io.obs_gov + (uint32_t)slot * (uint32_t)(c.E * c.D_gov_pad) : nullptr; }
    __device__ __forceinline__ float* rew() const { return io.rew ? io.rew + (uint32_t)slot * (uint32_t)(c.E * (c.N + 1)) : nullptr; }
    __device__ __forceinline__ uint8_t* done() const { return io.done ? io.done + (uint32_t)slot * (uint32_t)c.E : nullptr; }
    __device__ __forceinline__ int32_t* actions_out() const { return io.actions_out ? io.actions_out + (uint32_t)slot * (uint32_t)(c.E * c.N) : nullptr; }
    __device__ __forceinline__ int32_t* gov_out() const { return io.gov_out ? io.gov_out + (uint32_t)slot * (uint32_t)(c.E * c.B) : nullptr; }
};

// Phases P1-P4 of one environment step on the state in shared memory (G1: actions -> match ->
// expire -> tax); returns the pre-step values the rewards need.  `first` = first step of this
// launch (full observation rows).
template <int NPAD, int NS, int RT, int PT, int NT, int BT, int PF, class SM>
__device__ __forceinline__ void step_body(const DevCfg& c, const SM& m, int tid, int e, const StepPtrs& io, bool first, int t,
                                          float& coin_pre, float& labor_pre, double& cf_pre, int& rows) {
    // RT, PT > 0: resource and price counts known at compile time (shape-specialised variants)
    const int N = NT > 0 ? NT : c.N, B = BT > 0 ? BT : c.B, R = RT > 0 ? RT : c.R, P = PT > 0 ? PT : c.P, nl = (RT > 0 && PT > 0) ? 2 * RT * PT : c.n_levels;
    // PF = 1: the paper's mechanics (Table 2: 15 live orders per agent, one craft action
    // over R_d = R_kappa = 2, no-op on) with no book cap, as compile-time constants
    const int K = PF ? 0 : c.K, M = PF ? 15 : c.M, MPL = PF ? 4 : c.Mp_log2;
    const int craft_mode = PF ? EJ_CRAFT_SINGLE : c.craft_mode, craft_units = PF ? 2 : c.craft_units, craft_distinct = PF ? 2 : c.craft_distinct;
    const int base_buy = PF ? R + 1 : c.base_buy, base_sell = PF ? R + 1 + R * P : c.base_sell, A = PF ? 2 * R * P + R + 2 : c.A;
    constexpr int N4 = NS;  // stride of the per-agent arrays
    const bool act = tid < N;
    const uint32_t gid = c.env_id_base + (uint32_t)e;
    const uint32_t ep_bits = (uint32_t)m.hdr()->episode << 8;  // G44: the episode index in the upper bits of the stream word
    int* cnt_cur = m.cnt() + (t & 1) * nl;
    int* cnt_nxt = m.cnt() + ((t & 1) ^ 1) * nl;

    // ---------------- P1 actions (one action per agent per step) ----------------
    uint32_t x0 = 0, x1 = 0, x2 = 0, x3 = 0;
    int a = -1;
    if (act) {
        philox4x32_10(gid, (uint32_t)tid, (uint32_t)t, ep_bits, c.seed_lo, c.seed_hi, x0, x1, x2, x3);
        if (io.io.actions) {
            a = io.actions()[(uint32_t)(e * N + tid)];
        } else if (io.io.masked) {
            a = masked_draw<NS>(c, m, tid, x0, R, P, M, craft_mode, craft_units, craft_distinct, base_buy, base_sell, A);
        } else {  // smallest a with x0 < cdf[a]; last entry read as 2^32 (G30)
            int lo = 0, hi = A - 1;
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (x0 < m.cdf()[mid]) hi = mid;
                else lo = mid + 1;
            }
            a = lo;
        }
        if (io.io.actions_out) io.actions_out()[(uint32_t)(e * N + tid)] = a;
        m.key()[tid] = x2;
    }
    // government levels for the period boundary
    int gov_lvl = -1;
    const int tp = m.hdr()->t_in_period;
    const bool period_end = tp + 1 == c.period;
    const bool boundary = c.taxes_enabled && period_end;
    if (tid < B && (boundary || io.io.gov_out)) {
        if (io.io.gov_actions) {
            gov_lvl = io.gov_actions()[(uint32_t)(e * B + tid)];
        } else {
            uint32_t g0, g1, g2, g3;
            philox4x32_10(gid, (uint32_t)N, (uint32_t)t, (uint32_t)(1 + tid / 4) | ep_bits, c.seed_lo, c.seed_hi, g0, g1, g2, g3);
            const uint32_t gx = (tid & 3) == 0 ? g0 : (tid & 3) == 1 ? g1 : (tid & 3) == 2 ? g2 : g3;
            gov_lvl = (int)(((unsigned long long)gx * (unsigned long long)c.L) >> 32);
        }
        if (io.io.gov_out) io.gov_out()[(uint32_t)(e * B + tid)] = gov_lvl;
    }

    int lvl = -1, grp = 0, price_c = 0, r_c = 0, side_c = 0;
    uint32_t slot = 0, mymask = 0, old_tail = NIL;
    if (act) {
        coin_pre = m.coin()[tid];
        labor_pre = m.labor()[tid];
        cf_pre = m.cf()[tid];
        mymask = m.mask()[tid];
        bool invalid = false;
        if (a < 0 || a >= A) {
            invalid = true;  // G2
        } else if (a < R) {  // gather: floor(SG + rho), rho = u * 1.1 (G8)
            const float rho = __fmul_rn(u01(x1), 1.1f);
            const float s = __fadd_rn(m.SG()[a * N4 + tid], rho);
            m.inv()[a * N4 + tid] += (int)floorf(s);
            m.labor()[tid] = __fadd_rn(labor_pre, c.labor_gather);
            if (c.skill_rate > 0.0f)  // f3: the amount above used the skill before the increase
                m.SG()[a * N4 + tid] = progress_skill(m.SG()[a * N4 + tid], c.skill_rate, c.skill_max);
        } else if (a < base_buy) {  // craft
            bool ok;
            if (craft_mode == EJ_CRAFT_PER_RESOURCE) {
                const int r = a - R;
                ok = m.inv()[r * N4 + tid] >= craft_units;
                if (ok) m.inv()[r * N4 + tid] -= craft_units;
            } else {
                int enough = 0;
                for (int r = 0; r < R; ++r) enough += m.inv()[r * N4 + tid] >= craft_units;
                ok = enough >= craft_distinct;
                if (ok) {  // the R_d most-held resources, ties to the lowest index (G7)
                    uint32_t used = 0;
                    for (int k = 0; k < craft_distinct; ++k) {
                        int best = -1, bestv = 0;
                        for (int r = 0; r < R; ++r) {
                            if ((used >> r) & 1u) continue;
                            const int v = m.inv()[r * N4 + tid];
                            if (best < 0 || v > bestv) { best = r; bestv = v; }
                        }
                        used |= 1u << best;
                        m.inv()[best * N4 + tid] = bestv - craft_units;
                    }
                }
            }
            if (ok) {
                const float pay = __fmul_rn(m.SC()[tid], c.craft_scale);
                m.coin()[tid] = __fadd_rn(coin_pre, pay);
                m.income()[tid] = __fadd_rn(m.income()[tid], pay);
                m.labor()[tid] = __fadd_rn(labor_pre, c.labor_craft);
                if (c.skill_rate > 0.0f)  // f3: the payout above used the skill before the increase
                    m.SC()[tid] = progress_skill(m.SC()[tid], c.skill_rate, c.skill_max);
            } else {
                invalid = true;
            }
        } else if (a < base_sell + R * P) {  // market order
            side_c = a >= base_sell;
            const int k = a - (side_c ? base_sell : base_buy);
            r_c = PT > 0 ? k / (PT > 0 ? PT : 1) : (k * c.recipP) >> 16;
            const int pidx = k - r_c * P;
            price_c = c.prices[pidx];
            bool ok = __popc(mymask) < M;
            if (side_c == 0) ok = ok && (coin_pre >= (float)price_c);
            else ok = ok && (m.inv()[r_c * N4 + tid] >= 1);
            if (ok) {
                lvl = (r_c * 2 + side_c) * P + pidx;
                slot = ((uint32_t)tid << MPL) + (uint32_t)(__ffs(~mymask) - 1);
                m.cslot()[tid] = slot;
                old_tail = m.tail()[lvl];  // read before anyone links (tails change after barrier #1)
                if (K) {  // book cap: push on the key bins of the level and of the book
                    grp = r_c * 2 + side_c;
                    const uint32_t n1 = atomicExch(&m.lbh()[(uint32_t)lvl * LEVEL_BINS + (x2 >> LEVEL_BIN_SHIFT)], (uint32_t)tid);
                    atomicOr(&m.lmask()[lvl], 1u << (x2 >> LEVEL_BIN_SHIFT));
                    const uint32_t bb = (uint32_t)grp * BOOK_BINS + (x2 >> BOOK_BIN_SHIFT);
                    const uint32_t n2 = atomicExch(&m.bbh()[bb], (uint32_t)tid);
                    atomicAdd(&m.bbc()[bb], 1u);
                    m.anext()[tid] = n1 | (n2 << 16);  // next candidate of the level bin | of the book bin
                } else {  // push on the level's arrival stack
                    m.anext()[tid] = atomicExch(&m.ahead()[lvl], (uint32_t)tid);
                }
            } else {
                invalid = true;
            }
        }  // else NO-OP
        if (invalid) atomicAdd(&m.hdr()->n_invalid, 1);
    }
    __syncthreads();  // #1 arrivals registered
    EJ_MARK(1);

    // Arrival order of this step's candidates: (key, agent) (G11).  Each candidate finds its rank
    // among the step's arrivals on its level and its successor; with a book cap also its rank on
    // the book, counted from the book size at step start (G15).
    int lrank = 0;
    bool accepted = false;
    uint32_t nxt = NIL;
    if (K == 0) {
        if (lvl >= 0) {
            int succ = -1;
            uint32_t sk = 0;
            uint32_t j = m.ahead()[lvl];
            while (j != NIL) {
                if ((int)j != tid) {
                    const uint32_t kj = m.key()[j];
                    const bool later = (kj > x2) || (kj == x2 && (int)j > tid);
                    if (!later) ++lrank;
                    else if (succ < 0 || kj < sk || (kj == sk && (int)j < succ)) { succ = (int)j; sk = kj; }
                }
                j = m.anext()[j];
            }
            if (succ >= 0) nxt = m.cslot()[succ];
            accepted = true;
        }
    } else {
        // Book cap (G15): the j-th candidate of a book in arrival order is accepted iff n_rest + j < K.  Rank on the
        // book = candidates in lower key bins (exclusive prefix of the bin counts) + earlier candidates of the own bin.
        for (int w = tid >> 5; w < 2 * R; w += NPAD / 32) {  // a warp scans the bins of one book: 8 bins per lane
            const int lane = tid & 31;
            uint32_t* cnt = m.bbc() + w * BOOK_BINS + lane * (BOOK_BINS / 32);
            uint32_t v[BOOK_BINS / 32], sum = 0;
#pragma unroll
            for (int q = 0; q < BOOK_BINS / 32; ++q) { v[q] = cnt[q]; sum += v[q]; }
            uint32_t incl = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += y;
            }
            uint32_t run = incl - sum;
#pragma unroll
            for (int q = 0; q < BOOK_BINS / 32; ++q) { cnt[q] = run; run += v[q]; }
        }
        __syncthreads();
        int succ = -1;
        if (lvl >= 0) {
            const uint32_t bb = (uint32_t)grp * BOOK_BINS + (x2 >> BOOK_BIN_SHIFT);
            int brank = (int)m.bbc()[bb];
            for (uint32_t j = m.bbh()[bb]; j != NIL; j = m.anext()[j] >> 16) {
                const uint32_t kj = m.key()[j];
                brank += (kj < x2) || (kj == x2 && (int)j < tid);
            }
            int n_rest = 0;
            for (int p = 0; p < P; ++p) n_rest += cnt_cur[grp * P + p];
            accepted = n_rest + brank < K;
            m.cslot()[tid] = slot | (accepted ? 0x10000u : 0u);
            // neighbours on the level: an earlier arrival (then this one is not the level's first) and the next one
            const uint32_t b5 = x2 >> LEVEL_BIN_SHIFT, lmask = m.lmask()[lvl];
            lrank = (lmask & ((1u << b5) - 1u)) != 0u;
            uint32_t sk = 0;
            for (uint32_t j = m.lbh()[(uint32_t)lvl * LEVEL_BINS + b5]; j != NIL; j = m.anext()[j] & 0xFFFFu) {
                if ((int)j == tid) continue;
                const uint32_t kj = m.key()[j];
                const bool later = (kj > x2) || (kj == x2 && (int)j > tid);
                if (!later) lrank = 1;
                else if (succ < 0 || kj < sk || (kj == sk && (int)j < succ)) { succ = (int)j; sk = kj; }
            }
            const uint32_t above = (lmask >> b5) >> 1;
            if (succ < 0 && above) {  // the earliest arrival of the next occupied bin
                const uint32_t b2 = b5 + (uint32_t)__ffs(above);
                for (uint32_t j = m.lbh()[(uint32_t)lvl * LEVEL_BINS + b2]; j != NIL; j = m.anext()[j] & 0xFFFFu) {
                    const uint32_t kj = m.key()[j];
                    if (succ < 0 || kj < sk || (kj == sk && (int)j < succ)) { succ = (int)j; sk = kj; }
                }
            }
        }
        __syncthreads();  // acceptance flags of every candidate
        if (lvl >= 0) {
            if (accepted && succ >= 0) {  // acceptance is a prefix of the book's arrival order: only the successor can fail
                const uint32_t cs = m.cslot()[succ];
                if (cs & 0x10000u) nxt = cs & 0xFFFFu;
            }
            // bins ready for the next step (every member of a bin writes the same values)
            m.lbh()[(uint32_t)lvl * LEVEL_BINS + (x2 >> LEVEL_BIN_SHIFT)] = NIL;
            m.lmask()[lvl] = 0u;
            m.bbh()[(uint32_t)grp * BOOK_BINS + (x2 >> BOOK_BIN_SHIFT)] = NIL;
        }
        for (int g = tid; g < 2 * R * BOOK_BINS; g += NPAD) m.bbc()[g] = 0u;
    }

    if (lvl >= 0) {
        if (accepted) {
            m.template pool<PF>()[slot] = PoolW<PF>::make(nxt, t);
            if (lrank == 0) {
                if (old_tail != NIL) m.template pool<PF>()[old_tail] = PoolW<PF>::with_next(m.template pool<PF>()[old_tail], slot);
                else m.head()[lvl] = (uint16_t)slot;
            }
            if (nxt == NIL) m.tail()[lvl] = (uint16_t)slot;
            atomicAdd(&cnt_cur[lvl], 1);
            m.mask()[tid] = mymask | (1u << (slot & ((1u << MPL) - 1u)));
            if (side_c == 0) {  // escrow
                m.coin()[tid] = __fsub_rn(coin_pre, (float)price_c);
                m.esc_coin()[tid] += price_c;
            } else {
                m.inv()[r_c * N4 + tid] -= 1;
                m.esc_res()[r_c * N4 + tid] += 1;
            }
            m.labor()[tid] = __fadd_rn(labor_pre, c.labor_trade);
            atomicAdd(&m.hdr()->n_placed, 1);
        } else {
            atomicAdd(&m.hdr()->n_invalid, 1);
        }
    }
    __syncthreads();  // #2 books hold this step's arrivals
    EJ_MARK(2);

    // ---------------- P2 match + P3 expire (G14) ----------------
    // One thread per level.  Trades of a resource: q = max_p min(#bids >= p, #asks <= p); the
    // q best bids and q best asks are popped from the queue heads, then the expired heads.
    for (int l = tid; l < nl; l += NPAD) {
        const int book = PT > 0 ? l / (PT > 0 ? PT : 1) : (l * c.recipP) >> 16, pidx = l - book * P, r = book >> 1, side = book & 1;
        const int price = c.prices[pidx];
        const int lb = (r * 2) * P, la = lb + P;
        int totB = 0;
        for (int p = 0; p < P; ++p) totB += cnt_cur[lb + p];
        int q = 0, ale = 0, prefB = 0, alt_me = 0, bgt_me = 0;
        for (int p = 0; p < P; ++p) {
            if (p == pidx) alt_me = ale;
            ale += cnt_cur[la + p];
            const int cb = cnt_cur[lb + p];
            q = max(q, min(totB - prefB, ale));
            prefB += cb;
            if (p == pidx) bgt_me = totB - prefB;
        }
        const int better = side ? alt_me : bgt_me;  // orders ahead of this level on its side
        int n = cnt_cur[l];
        const int tk = max(0, min(n, q - better));
        uint32_t h = m.head()[l];
        if (tk > 0) {
            uint32_t* dst = (side ? m.ma() : m.mb()) + r * N4 + better;
            for (int k = 0; k < tk; ++k) {
                dst[k] = h | ((uint32_t)pidx << 16);
                h = PoolW<PF>::next(m.template pool<PF>()[h]);
            }
            n -= tk;
        }
        int nexp = 0;
        while (h != NIL) {
            const typename PoolW<PF>::T pe = m.template pool<PF>()[h];
            const uint32_t age = PoolW<PF>::age(pe, t);
            if ((int)age < c.expiry) break;
            const int owner = (int)(h >> MPL);
            if (side == 0) {
                atomicSub(&m.esc_coin()[owner], price);
                atomicAdd(&m.credit()[owner], price);
            } else {
                atomicSub(&m.esc_res()[r * N4 + owner], 1);
                atomicAdd(&m.inv()[r * N4 + owner], 1);
            }
            atomicAnd(&m.mask()[owner], ~(1u << (h & ((1u << MPL) - 1u))));
            ++nexp;
            --n;
            h = PoolW<PF>::next(pe);
        }
        if (tk > 0 || nexp > 0) {
            m.head()[l] = (uint16_t)h;
            if (h == NIL) m.tail()[l] = (uint16_t)NIL;
            if (nexp) atomicAdd(&m.hdr()->n_expired, nexp);
        }
        cnt_nxt[l] = n;
        if (K == 0) m.ahead()[l] = NIL;
        if (side == 0 && pidx == 0) m.resq()[r] = q;
    }
    __syncthreads();  // #3 matched lists complete
    EJ_MARK(3);

    // settle trade i of resource r: bid rank i with ask rank i, at the price of the later arrival
    {
        int total = 0;
        for (int r = 0; r < R; ++r) {
            const int q = m.resq()[r];
            total += q;
            if (tid < q) {
                const uint32_t eb = m.mb()[r * N4 + tid], ea = m.ma()[r * N4 + tid];
                const uint32_t sb = eb & 0xFFFFu, sa = ea & 0xFFFFu;
                const int pb = c.prices[eb >> 16], pa = c.prices[ea >> 16];
                const int ob = (int)(sb >> MPL), oa = (int)(sa >> MPL);
                const uint32_t age_b = PoolW<PF>::age(m.template pool<PF>()[sb], t);
                const uint32_t age_a = PoolW<PF>::age(m.template pool<PF>()[sa], t);
                bool bid_later;
                if (age_b != age_a) bid_later = age_b < age_a;
                else if (m.key()[ob] != m.key()[oa]) bid_later = m.key()[ob] > m.key()[oa];
                else bid_later = ob > oa;
                const int pi = bid_later ? pb : pa;
                const uint32_t bitmask = (1u << MPL) - 1u;
                atomicSub(&m.esc_coin()[ob], pb);
                if (pb - pi) atomicAdd(&m.credit()[ob], pb - pi);  // refund of the escrowed excess
                atomicAdd(&m.inv()[r * N4 + ob], 1);
                atomicAnd(&m.mask()[ob], ~(1u << (sb & bitmask)));
                atomicSub(&m.esc_res()[r * N4 + oa], 1);
                atomicAdd(&m.credit()[oa], pi);
                atomicAdd(&m.sale()[oa], pi);
                atomicAnd(&m.mask()[oa], ~(1u << (sa & bitmask)));
                if (tid == q - 1) m.hdr()->last_price[r] = pi;
            }
        }
        if (tid == 0) m.hdr()->n_trades += total;
    }
    __syncthreads();  // #4 credits complete
    EJ_MARK(4);
#ifdef EJ_DEBUG_POISON
    // Debug builds (-DEJ_DEBUG_POISON): everything that is dead from here to the next step's arrivals -- the matched-order
    // lists (they alias the head of the staging tile), arrival keys, candidate slots, arrival stacks -- is overwritten
    // with a pattern, so that a stale read of aliased bytes shows up as a parity failure instead of going unnoticed.
    for (int i = tid; i < 2 * R * N4; i += NPAD) m.mb()[i] = 0xDEADBEEFu;
    if (tid < N4) { m.key()[tid] = 0xDEADBEEFu; m.cslot()[tid] = 0xDEADBEEFu; m.anext()[tid] = 0xDEADBEEFu; }
    __syncthreads();
#endif

    // income from sales (G16), coin credit once per agent
    if (act) {
        const int sl = m.sale()[tid], cr = m.credit()[tid];
        if (sl > 0) { m.income()[tid] = __fadd_rn(m.income()[tid], (float)sl); m.sale()[tid] = 0; }
        if (cr > 0) { m.coin()[tid] = __fadd_rn(m.coin()[tid], (float)cr); m.credit()[tid] = 0; }
    }
    if (tid >= NPAD - R) write_market_row<PT>(c, m, NPAD - 1 - tid, cnt_nxt);
    if (tid == 0) write_timers(c, m, t + 1, period_end ? 0 : tp + 1);

    // ---------------- P4 tax at period end (G17-G20) ----------------
    if (boundary) {
        long long fx = 0;
        if (act) {
            const float income = m.income()[tid];
            float tax = 0.0f, lo = 0.0f;
            for (int b = 0; b < B; ++b) {
                const float hi = (b < B - 1) ? c.thresholds[b] : INFINITY;
                const float top = (income < hi) ? income : hi;
                float por = __fsub_rn(top, lo);
                if (por < 0.0f) por = 0.0f;
                tax = __fadd_rn(tax, __fmul_rn(m.hdr()->rates[b], por));
                lo = hi;
            }
            const float coin = m.coin()[tid];
            if (tax > coin) tax = coin;  // G17
            m.coin()[tid] = __fsub_rn(coin, tax);
            fx = __double2ll_rn((double)tax * 1048576.0);  // G19
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) fx += __shfl_xor_sync(FULL, fx, o);
        if ((tid & 31) == 0 && fx != 0) atomicAdd(&m.misc()[0], (unsigned long long)fx);
        __syncthreads();
        if (act) {
            const float pool = __double2float_rn((double)(long long)m.misc()[0] * (1.0 / 1048576.0));
            const float share = __fdiv_rn(pool, (float)N);  // P:195 "(1/n)"
            m.coin()[tid] = __fadd_rn(m.coin()[tid], share);
            m.income()[tid] = 0.0f;
        }
        if (tid < B) {  // rates of the upcoming period
            if (gov_lvl < 0 || gov_lvl >= c.L) atomicAdd(&m.hdr()->n_bad_gov, 1);
            else m.hdr()->rates[tid] = c.rate_table[gov_lvl];
        }
    }
    if (tid < B && (boundary || first)) m.shrow()[5 * R + tid] = m.hdr()->rates[tid];
    if (SM::L::bucketed) bucket_fill_all<NPAD>(m, tid, act);  // coin, labor, income are final: file them for the block-wide sort
    __syncthreads();  // #5 state final
    EJ_MARK(5);
    if (tid == 0) {
        m.hdr()->t = t + 1;
        m.hdr()->t_in_period = period_end ? 0 : tp + 1;
        if (boundary) m.misc()[0] = 0ull;
        if (io.io.done) io.done()[e] = (uint8_t)(t + 1 == c.T);
    }

    // f3: growing skills change the skill columns of the staged rows at any step
    rows = (first || c.skill_rate > 0.0f) ? 2 : (boundary ? 1 : 0);
}

// Initial state of an episode (G29, G30, G44) in the shared-memory blob: every agent holds starting_coin and
// nothing else, books empty, rates 0, t = 0, skills drawn from the counters of (seed, global env, agent, episode).  The
// env's event counters are cleared only by ej_reset.  Called by all threads; the caller synchronises afterwards.
template <int NPAD, int NS, class SM>
__device__ __noinline__ void init_env_state(const DevCfg& c, const SM& m, int tid, uint32_t gid, int episode, bool clear_counters) {
    const uint32_t ep = (uint32_t)episode << 8;
    if (tid < c.N) {
        m.coin()[tid] = c.starting_coin;
        m.cf()[tid] = coin_utility(c.starting_coin, c.ua, c.inv_ua);
        m.labor()[tid] = 0.0f;
        m.income()[tid] = 0.0f;
        m.esc_coin()[tid] = 0;
        m.mask()[tid] = 0u;
        for (int r = 0; r < c.R; ++r) { m.inv()[r * NS + tid] = 0; m.esc_res()[r * NS + tid] = 0; }
        uint32_t x[4] = {0, 0, 0, 0};
        for (int d = 0; d <= c.R; ++d) {  // skill draw d: Philox stream 16, "t" field d/4, word d%4
            if ((d & 3) == 0) philox4x32_10(gid, (uint32_t)tid, (uint32_t)(d >> 2), 16u | ep, c.seed_lo, c.seed_hi, x[0], x[1], x[2], x[3]);
            const uint32_t w = (d & 3) == 0 ? x[0] : (d & 3) == 1 ? x[1] : (d & 3) == 2 ? x[2] : x[3];
            float v = u01(w);
            if (c.skill_init == EJ_SKILL_NORMAL_CLIP) {
                // f3 (G42): z = sum of twelve 24-bit uniforms - 6 (stream 17, "t" fields 3d .. 3d+2); the
                // sum is an integer, z and std * z are exact in binary64, one rounding to binary32, then the clip
                long long sum = 0;
                for (int j = 0; j < 3; ++j) {
                    uint32_t y0, y1, y2, y3;
                    philox4x32_10(gid, (uint32_t)tid, (uint32_t)(3 * d + j), 17u | ep, c.seed_lo, c.seed_hi, y0, y1, y2, y3);
                    sum += (long long)(y0 >> 8) + (long long)(y1 >> 8) + (long long)(y2 >> 8) + (long long)(y3 >> 8);
                }
                const double z = __dsub_rn(__dmul_rn((double)sum, 1.0 / 16777216.0), 6.0);
                v = __double2float_rn(__dadd_rn((double)c.skill_mean, __dmul_rn((double)c.skill_std, z)));
                if (v < c.clip_lo) v = c.clip_lo;
                if (v > c.clip_hi) v = c.clip_hi;
            } else if (c.skill_init == EJ_SKILL_PARETO_CLIP) {  // Pareto(4) by inversion: 1/sqrt(sqrt(1-u))
                float rr = __fsqrt_rn(__fsub_rn(1.0f, v));
                rr = __fsqrt_rn(rr);
                v = __fdiv_rn(1.0f, rr);
                if (v < c.clip_lo) v = c.clip_lo;
                if (v > c.clip_hi) v = c.clip_hi;
            }
            if (d < c.R) m.SG()[d * NS + tid] = v;
            else m.SC()[tid] = v;
        }
    }
    for (int l = tid; l < c.n_levels; l += NPAD) {
        m.head()[l] = (uint16_t)NIL;
        m.tail()[l] = (uint16_t)NIL;
        m.cnt()[l] = 0;
        m.cnt()[c.n_levels + l] = 0;
    }
    if (tid < EJ_MAX_BRACKETS) m.hdr()->rates[tid] = 0.0f;
    if (tid < EJ_MAX_RESOURCES) m.hdr()->last_price[tid] = 0;
    if (tid == 0) {  // all coins equal: gini = 0, prod = N * coin (exact)
        EnvHdr* hd = m.hdr();
        hd->t = 0;
        hd->t_in_period = 0;
        hd->episode = episode;
        if (clear_counters) hd->n_trades = hd->n_placed = hd->n_invalid = hd->n_expired = hd->n_bad_gov = 0;
        const double prod = (double)c.N * (double)c.starting_coin;
        const double eq = (double)c.omega * (1.0 - 0.0) + (1.0 - (double)c.omega);
        hd->u_g_prev = eq * prod;
    }
}

// f4 (G44), the cold half of an auto-resetting step: the episode has just ended and its rewards are out; start the next
// episode and write the fresh state's observation.  Out of line, with its own copy of outputs(): the hot path of a
// step keeps its single inlined call.
template <int NPAD, int NS, int RT, int NT, int BT, int PF, int FX, class SM>
__device__ __noinline__ void renew_episode(const DevCfg& c, const SM& m, int tid, int e, const StepPtrs& io) {
    const int ep = m.hdr()->episode + 1;
    __syncthreads();  // the rewards and statistics of the terminal state are done
    init_env_state<NPAD, NS>(c, m, tid, c.env_id_base + (uint32_t)e, ep, false);
    __syncthreads();
    if (tid < c.R) write_market_row<0>(c, m, tid, m.cnt());
    if (tid < c.B) m.shrow()[5 * c.R + tid] = 0.0f;
    if (tid == NPAD - 1) write_timers(c, m, 0, 0);
    if (SM::L::bucketed) bucket_fill_all<NPAD>(m, tid, tid < c.N);
    __syncthreads();
    outputs<NPAD, NS, RT, NT, BT, PF, FX>(c, m, tid, e, 2, 2, 0.f, 0.f, 0.0, io.obs(), nullptr, FX ? io.priv() : nullptr, FX ? io.shared() : nullptr,
                                          FX ? io.govp() : nullptr);
}

// One environment step: P1-P4 (or nothing for a finished env, G28), then P5 rewards and P6
// observations.  outputs() has this single call site on the hot path (instruction footprint).
// f4 (G44), auto-reset: a step that ends an episode gives its rewards and done as usual, then the env starts its next
// episode at once and the step's observation is the one of the fresh state (renew_episode).
template <int NPAD, int NS, int RT, int PT, int NT, int BT, int PF, int FX, int AR, class SM>
__device__ void env_step(const DevCfg& c, const SM& m, int tid, int e, const StepPtrs& io, bool first) {
    int t = m.hdr()->t;
    // the previous step's bulk stores must have read the staging tile before it is rewritten
    if (tid == (SM::L::bucketed ? NPAD - 32 : 0)) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");  // the thread that issued them
    // AR = 1: the kernel variant launched for auto-resetting rollouts.  A template parameter because the renewal code,
    // compiled into the one kernel, cost the plain rollout 2-8 % while unused (registers: spills at 1024 threads).
    const bool auto_reset = AR != 0 && io.io.auto_reset != 0;
    const uint32_t gid = c.env_id_base + (uint32_t)e;
    if (auto_reset && t >= c.T) {  // finished before this call began: its next episode starts with this step
        const int ep = m.hdr()->episode + 1;
        __syncthreads();
        init_env_state<NPAD, NS>(c, m, tid, gid, ep, false);
        __syncthreads();
        t = 0;
        first = true;
    }
    float coin_pre = 0.f, labor_pre = 0.f;
    double cf_pre = 0.0;
    int mode = 0, rows = 2;
    if (t >= c.T) {  // G28: finished env
        __syncthreads();  // thread 0 has waited for the previous step's bulk reads of shrow / the staging tile
        if (tid < c.R) write_market_row<0>(c, m, tid, m.cnt() + (t & 1) * c.n_levels);
        if (tid < c.B) m.shrow()[5 * c.R + tid] = m.hdr()->rates[tid];
        if (tid == NPAD - 1) write_timers(c, m, t, m.hdr()->t_in_period);
        if (SM::L::bucketed) bucket_fill_all<NPAD>(m, tid, tid < c.N);
        __syncthreads();
        mode = 1;
    } else {
        step_body<NPAD, NS, RT, PT, NT, BT, PF>(c, m, tid, e, io, first, t, coin_pre, labor_pre, cf_pre, rows);
    }
    // ---------------- P5 rewards, P6 observations ----------------
    const bool renew = auto_reset && mode == 0 && t + 1 == c.T;  // this step ended the episode: its observation comes from renew_episode
    outputs<NPAD, NS, RT, NT, BT, PF, FX>(c, m, tid, e, mode, rows, coin_pre, labor_pre, cf_pre, renew ? nullptr : io.obs(), io.rew(),
                                          (FX && !renew) ? io.priv() : nullptr, (FX && !renew) ? io.shared() : nullptr,
                                          (FX && !renew) ? io.govp() : nullptr);
    if (AR != 0 && renew) renew_episode<NPAD, NS, RT, NT, BT, PF, FX>(c, m, tid, e, io);
    EJ_MARK(8);
    if (mode == 1) {
        if (tid == 0 && io.io.done) io.done()[e] = 1;
        __syncthreads();  // shrow is rewritten at the very start of the next finished step
    }
}

template <int NPAD, int NS, int RT, int PT, int NT, int BT, int PF, int FX = 0, int AR = 0>
__global__ void __launch_bounds__(NPAD, (NPAD == 128 ? ((PF && FX) ? EJ_CTAS_128_FX : EJ_CTAS_128) : 1024 / NPAD < 8 ? 1024 / NPAD : 8)) ej_step_kernel(const __grid_constant__ DevCfg c, uint8_t* __restrict__ state,
                                                       const __grid_constant__ StepIO io) {
    extern __shared__ __align__(16) uint8_t ej_smem[];
    uint8_t* const sblob = ej_smem + Lay<NS>::blob;
    const int e = blockIdx.x, tid = threadIdx.x;
    const Sm<NS, (PF ? RT : 0), (PF ? PT : 0), (PF ? NT : 0)> m{c};
    uint8_t* const blob = state + (size_t)e * c.blob_bytes;
    // The state blob comes in as ONE 1-D TMA bulk copy that completes on an mbarrier (misc()[1]) while the CTA
    // clears its scratch and builds its tables, and leaves as one bulk store: with one launch per step (ej_step)
    // the blob traffic is as large as the outputs, and a copy loop costs issue slots the step itself needs.
    const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&m.misc()[1]);
    for (int i = tid; i < Lay<NS>::blob / 16; i += NPAD) ((uint4*)ej_smem)[i] = make_uint4(0u, 0u, 0u, 0u);
    for (int i = tid; i < (c.o_stage - c.o_scratch1) / 16; i += NPAD) ((uint4*)(ej_smem + c.o_scratch1))[i] = make_uint4(0u, 0u, 0u, 0u);
    __syncthreads();
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(c.blob_bytes) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                         (uint32_t)__cvta_generic_to_shared(sblob)),
                     "l"(blob), "r"(c.blob_bytes), "r"(bar)
                     : "memory");
    }
    if (c.K == 0) {
        for (int l = tid; l < c.n_levels; l += NPAD) m.ahead()[l] = NIL;
    } else {
        for (int l = tid; l < c.n_levels * LEVEL_BINS; l += NPAD) m.lbh()[l] = NIL;
        for (int l = tid; l < 2 * c.R * BOOK_BINS; l += NPAD) m.bbh()[l] = NIL;
    }
    if (!io.actions)
        for (int i = tid; i < c.A; i += NPAD) m.cdf()[i] = io.cdf[i];
    __syncthreads();  // the tables above, and the mbarrier's initialisation, for every thread
    asm volatile(
        "{\n\t.reg .pred p;\n\tEJ_BLOB_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0;\n\t"
        "@p bra EJ_BLOB_DONE_%=;\n\tbra EJ_BLOB_WAIT_%=;\n\tEJ_BLOB_DONE_%=:\n\t}" ::"r"(bar)
        : "memory");
    StepPtrs p{io, c, 0, 0};
#ifdef EJ_PHASE_CLOCK
    if (blockIdx.x == 0 && tid == 0) { for (int k = 0; k < 16; ++k) ej_phase_cycles[k] = 0; ej_phase_last = clock64(); }
#endif
#pragma unroll 1
    for (int s = 0; s < io.n_steps; ++s) {
        p.s = s;
        env_step<NPAD, NS, RT, PT, NT, BT, PF, FX, AR>(c, m, tid, e, p, s == 0);
        p.slot = (p.slot + 1 == io.ring_depth) ? 0 : p.slot + 1;
    }
#ifdef EJ_PHASE_CLOCK
    if (blockIdx.x == 0 && tid == 0 && io.n_steps > 1) {
        printf("phase cycles per step over %d steps (thread 0 of block 0):", io.n_steps);
        for (int k = 1; k <= 8; ++k) printf(" [%d] %.0f", k, (double)ej_phase_cycles[k] / io.n_steps);
        printf("\n");
    }
#endif
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // this thread's state writes, for the bulk store below
    __syncthreads();
    if (tid == 0) {
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(blob), "r"((uint32_t)__cvta_generic_to_shared(sblob)),
                     "r"(c.blob_bytes)
                     : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }
    // bucketed kernels: the observation stores of the last step were issued by the first thread of the last warp
    if (Lay<NS>::bucketed && tid == NPAD - 32) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

template <int NPAD, int NS>
__global__ void __launch_bounds__(NPAD) ej_observe_kernel(const __grid_constant__ DevCfg c, const uint8_t* __restrict__ state,
                                                          float* obs) {
    extern __shared__ __align__(16) uint8_t ej_smem[];
    uint8_t* const sblob = ej_smem + Lay<NS>::blob;
    const int e = blockIdx.x, tid = threadIdx.x;
    const Sm<NS> m{c};
    const uint4* blob = (const uint4*)(state + (size_t)e * c.blob_bytes);
    for (int i = tid; i < c.blob_bytes / 16; i += NPAD) ((uint4*)sblob)[i] = blob[i];
    if (Lay<NS>::bucketed && tid < Lay<NS>::bk_metrics * Lay<NS>::bk_cnt_words) m.bk_cnt(0)[tid] = 0u;
    __syncthreads();
    const int t = m.hdr()->t;
    if (tid < c.R) write_market_row<0>(c, m, tid, m.cnt() + (t & 1) * c.n_levels);
    if (tid < c.B) m.shrow()[5 * c.R + tid] = m.hdr()->rates[tid];
    if (tid == NPAD - 1) write_timers(c, m, t, m.hdr()->t_in_period);
    if (Lay<NS>::bucketed) bucket_fill_all<NPAD>(m, tid, tid < c.N);
    __syncthreads();
    outputs<NPAD, NS, 0, 0, 0, 0, 0>(c, m, tid, e, 2, 2, 0.f, 0.f, 0.0, obs, nullptr);
    if (tid == (Lay<NS>::bucketed ? NPAD - 32 : 0)) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");  // the thread that issued the stores
}

// Reset (ej_reset): one CTA per env builds the blob of episode 0 in shared memory and stores it.
template <int NPAD, int NS>
__global__ void __launch_bounds__(NPAD) ej_reset_kernel(const __grid_constant__ DevCfg c, uint8_t* __restrict__ state) {
    extern __shared__ __align__(16) uint8_t ej_smem[];
    uint8_t* const sblob = ej_smem + Lay<NS>::blob;
    const int e = blockIdx.x, tid = threadIdx.x;
    const Sm<NS> m{c};
    for (int i = tid; i < c.blob_bytes / 4; i += NPAD) ((uint32_t*)sblob)[i] = 0u;
    __syncthreads();
    init_env_state<NPAD, NS>(c, m, tid, c.env_id_base + (uint32_t)e, 0, true);
    __syncthreads();
    uint4* blob = (uint4*)(state + (size_t)e * c.blob_bytes);
    for (int i = tid; i < c.blob_bytes / 16; i += NPAD) blob[i] = ((uint4*)sblob)[i];
}

// f1: action mask of the current state (unavailable actions get zero probability;
// P:199 "cannot sell a resource it does not have"; preconditions of P:145-168; order cap P:277):
//   gather, no-op: 1;  craft: #{r : inv[r] >= R_kappa} >= R_d (PER_RESOURCE r: inv[r] >= R_kappa);
//   buy (r, p): coin >= price_p and live orders < M;  sell (r, p): inv[r] >= 1 and live orders < M.
// The per-book cap K (G15) depends on the step's arrival order and is not part of the mask.
// HBM-bound writer of [E][N][A] bytes: one thread per 4 output bytes (the flat byte index is
// split into env / agent / action once, then carried), state read from the blob in HBM (a few
// words per agent, L1/L2 hits); a 32-bit store per thread, coalesced.
__global__ void __launch_bounds__(256) ej_mask_kernel(const __grid_constant__ DevCfg c, const uint8_t* __restrict__ state,
                                                      uint8_t* __restrict__ mask_out, unsigned long long total) {
    const unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long g = w * 4ull;
    if (g >= total) return;
    const int A = c.A, N = c.N, R = c.R, P = c.P, NS = c.N4;
    unsigned long long row = g / (unsigned long long)A;  // e * N + i
    int a = (int)(g - row * (unsigned long long)A);
    int e = (int)(row / (unsigned long long)N), i = (int)(row - (unsigned long long)e * N);
    const int n_out = (total - g) < 4ull ? (int)(total - g) : 4;
    uint32_t packed = 0;
    const uint8_t* blob = state + (size_t)e * c.blob_bytes;
    int cached_i = -1, cached_e = -1;
    bool room = false, craft_ok = false;
    float coin = 0.f;
    for (int k = 0; k < n_out; ++k) {
        if (i != cached_i || e != cached_e) {
            blob = state + (size_t)e * c.blob_bytes;
            coin = ((const float*)(blob + c.o_coin))[i];
            room = __popc(((const uint32_t*)(blob + c.o_mask))[i]) < c.M;
            int enough = 0;
            const int* inv = (const int*)(blob + c.o_inv);
            for (int r = 0; r < R; ++r) enough += inv[r * NS + i] >= c.craft_units;
            craft_ok = enough >= c.craft_distinct;
            cached_i = i; cached_e = e;
        }
        const int* inv = (const int*)(blob + c.o_inv);
        bool ok;
        if (a < R) ok = true;
        else if (a < c.base_buy) ok = c.craft_mode == EJ_CRAFT_PER_RESOURCE ? inv[(a - R) * NS + i] >= c.craft_units : craft_ok;
        else if (a < c.base_sell) ok = room && coin >= (float)c.prices[(a - c.base_buy) % P];
        else if (a < c.base_sell + R * P) ok = room && inv[((a - c.base_sell) / P) * NS + i] >= 1;
        else ok = true;
        packed |= (ok ? 1u : 0u) << (8 * k);
        if (++a == A) { a = 0; if (++i == N) { i = 0; ++e; } }
    }
    if (n_out == 4) *(uint32_t*)(mask_out + g) = packed;
    else for (int k = 0; k < n_out; ++k) mask_out[g + k] = (uint8_t)(packed >> (8 * k));
}

}  // namespace
