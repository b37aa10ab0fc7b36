// ej_policy.cuh -- a12 of the hot path (BASELINE.json configs[4]): forward pass of the shared
// population policy MLP and of the government MLP (obs -> 128 -> 128 -> logits, tanh; P:240,
// Table 2) on the 5th-generation tensor cores, followed by categorical sampling with
// the counter-based Philox of G30 (G33).
//
// One CTA of 128 threads works on tiles of 128 observation rows (thread i = row i = TMEM lane
// i).  The three weight matrices stay resident in shared memory in the canonical K-major
// no-swizzle UMMA layout (8-row x 16-byte core matrices); the activation tile is rebuilt in the
// same layout between layers.  Each layer is a chain of tcgen05.mma (M=128, N=128|Op, K=16)
// issued by one thread, accumulating in TMEM; completion comes back through tcgen05.commit on
// an mbarrier; the epilogue reads its row with tcgen05.ld, adds the bias, applies tanh, rounds
// to bf16 and writes the next layer's A operand.  One CTA per SM holds the weights once and runs
// TWO such 128-thread groups on alternating tiles (own A tile, own half of TMEM, own named
// barrier), so one group's epilogue overlaps the other's MMAs; the fp32 observation tile of the
// group's next tile is prefetched by a 1-D TMA bulk copy (cp.async.bulk) while it computes.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int PH = 128;        // hidden width (B:configs[4]: 128 -> 128)
constexpr int PTILE = 128;     // rows per tile = UMMA M
constexpr int P_TMEM_ALLOC = 512;  // whole TMEM of the SM (one CTA per SM); group g uses columns [g * tmem_cols, ...)
constexpr int PGROUPS = 3;         // 128-thread groups per CTA (a job may use fewer)

struct PolicyNet {
    const uint8_t* blob;   // device: W1 | W2 | W3 (canonical bf16) | b1 | b2 | b3 (f32)
    int D_in, K1p;         // input width and its multiple-of-16 padding
    int n_out, Op;         // logits and their multiple-of-16 padding (<= 256)
    int n_heads, head;     // categorical heads of `head` logits each (n_out = n_heads * head)
    int w1_bytes, w2_bytes, w3_bytes, blob_bytes;
    uint32_t recipK1p;     // ceil(2^32 / K1p)
    int nch;               // 16-column chunks a head's logits span at most (register-resident sampler if <= 5)
};

// f1: what the masked sampler needs to rebuild a row's action mask from the env state blob
// (same rules as ej_mask_kernel).
struct PolicyMask {
    int on;
    int o_coin, o_mask, o_inv, NS;  // blob-relative byte offsets, stride of the per-agent arrays
    int R, P, M, craft_mode, craft_units, craft_distinct, base_buy, base_sell, A, allow_noop;
    int prices[EJ_MAX_PRICES];
};

struct PolicyArgs {
    PolicyNet net;
    PolicyMask mask;         // population job only
    const float* obs;        // first row
    int row_stride;          // floats between rows
    int rows;                // number of rows
    int rows_per_env;        // N for the population, 1 for the government
    int fixed_agent;         // Philox "agent" field when rows_per_env == 1 (government: N), else -1
    const uint8_t* state;    // env state blobs: the clock t is the first int32 of each
    int blob_stride;         // bytes between env blobs
    uint32_t env_id_base, seed_lo, seed_hi;
    uint32_t stream_base;    // Philox stream of head 0 (population 0, government 1); head h uses word h % 4 of stream + h / 4
    int32_t* actions;        // [rows][n_heads]
    float* logits;           // [rows][n_out] or null
    int smem_W1, smem_W2, smem_W3, smem_bias;  // byte offsets in dynamic shared memory (shared by both groups)
    int smem_group, group_bytes, stage_off;     // group g: A tile at smem_group + g * group_bytes, fp32 staging at + stage_off
    int groups, tmem_cols;   // active groups of this job (<= PGROUPS) and TMEM columns per group (128 or 256)
};

// One launch runs up to two jobs side by side: CTAs [0, split) work on job 0 (population),
// CTAs [split, gridDim.x) on job 1 (government), each with its own weights in shared memory.
struct PolicyLaunch {
    PolicyArgs job[2];
    int split;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// K-major, no-swizzle shared-memory matrix descriptor: 8 x 16 B core matrices, `lbo` bytes
// between the two core matrices of one K = 16 step, `sbo` bytes between 8-row groups.
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFFu) >> 4);
    d |= (uint64_t)((lbo >> 4) & 0x3FFFu) << 16;
    d |= (uint64_t)((sbo >> 4) & 0x3FFFu) << 32;
    d |= (uint64_t)1 << 46;  // descriptor version of sm_100
    return d;                // base offset 0, layout type 0 = no swizzle
}

// Instruction descriptor of kind::f16: bf16 x bf16 -> f32, A and B K-major, M = 128.
__device__ __forceinline__ uint32_t umma_idesc(int n) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(PTILE >> 4) << 24);
}

__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(tmem_d),
        "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

__device__ __forceinline__ void tmem_ld8(uint32_t taddr, float (&v)[8]) {
    uint32_t r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = __uint_as_float(r[j]);
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = __uint_as_float(r[j]);
}

__device__ __forceinline__ float tanh_fast(float x) {
    float y;
    asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Byte offset of element (row, k) in a K-major no-swizzle operand with `kp` columns.
__device__ __forceinline__ uint32_t op_off(int row, int k, int kp) {
    return (uint32_t)((row & 7) * 16 + (row >> 3) * (kp * 16) + (k >> 3) * 128 + (k & 7) * 2);
}

// Issue one layer: D[128 x n] (+)= A[128 x kp] * W[n x kp]^T, then commit to the mbarrier.
__device__ __forceinline__ void issue_layer(uint32_t a_addr, uint32_t w_addr, int kp, int n, uint32_t tmem_d, uint32_t bar) {
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const uint32_t idesc = umma_idesc(n);
    const uint32_t sbo = (uint32_t)kp * 16u;  // (kp / 8) core matrices of 128 B per 8-row group
    for (int k = 0; k < kp / 16; ++k) {
        const uint64_t da = umma_desc(a_addr + k * 256, 128, sbo);
        const uint64_t db = umma_desc(w_addr + k * 256, 128, sbo);
        umma_bf16(tmem_d, da, db, idesc, k > 0 ? 1u : 0u);
    }
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" ::"r"(bar) : "memory");
}

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];\n"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
          "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
          "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
}

// Hidden-layer epilogue: this thread's accumulator row -> +bias -> tanh -> bf16 -> A operand (kp = 128).
__device__ __forceinline__ void hidden_epilogue(uint32_t taddr_row, const float* bias, uint8_t* A, int row) {
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
#pragma unroll 1
    for (int c = 0; c < PH; c += 32) {
        uint32_t r[32];
        tmem_ld32(taddr_row + c, r);
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            uint32_t w[4];
            const float4 bl = *reinterpret_cast<const float4*>(bias + c + g * 8), bh = *reinterpret_cast<const float4*>(bias + c + g * 8 + 4);
            const float bb[8] = {bl.x, bl.y, bl.z, bl.w, bh.x, bh.y, bh.z, bh.w};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int k = g * 8 + 2 * j;
                const float a0 = tanh_fast(__uint_as_float(r[k]) + bb[2 * j]), a1 = tanh_fast(__uint_as_float(r[k + 1]) + bb[2 * j + 1]);
                const __nv_bfloat162 h = __floats2bfloat162_rn(a0, a1);
                w[j] = *reinterpret_cast<const uint32_t*>(&h);
            }
            *reinterpret_cast<uint4*>(A + op_off(row, c + g * 8, PH)) = make_uint4(w[0], w[1], w[2], w[3]);
        }
    }
}

template <int OFF, int LEN>
__device__ __forceinline__ void tmem_ld16_async(uint32_t taddr, float (&r)[LEN]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
        : "=f"(r[OFF + 0]), "=f"(r[OFF + 1]), "=f"(r[OFF + 2]), "=f"(r[OFF + 3]), "=f"(r[OFF + 4]), "=f"(r[OFF + 5]), "=f"(r[OFF + 6]),
          "=f"(r[OFF + 7]), "=f"(r[OFF + 8]), "=f"(r[OFF + 9]), "=f"(r[OFF + 10]), "=f"(r[OFF + 11]), "=f"(r[OFF + 12]),
          "=f"(r[OFF + 13]), "=f"(r[OFF + 14]), "=f"(r[OFF + 15])
        : "r"(taddr)
        : "memory");
}

template <int CH, int NCH>
__device__ __forceinline__ void load_window(uint32_t taddr, int c0, int op, float (&l)[NCH * 16]) {
    if constexpr (CH < NCH) {
        if (c0 + 16 * CH < op) tmem_ld16_async<16 * CH>(taddr + c0 + 16 * CH, l);
        else {
#pragma unroll
            for (int j = 0; j < 16; ++j) l[16 * CH + j] = 0.0f;
        }
        load_window<CH + 1, NCH>(taddr, c0, op, l);
    }
}

// One categorical head whose logits span at most NCH 16-column chunks: the whole window is read
// into registers once; maximum, exponentials, their sum and the cumulative search all run on
// registers (masked columns carry -inf, whose exponential is 0).  Returns the sampled index.
template <int NCH>
__device__ __forceinline__ int sample_head(uint32_t taddr_row, const float* b3, int lo, int hi, int op, float u, float* logits_row) {
    const int c0 = lo & ~15;
    float l[NCH * 16];
    load_window<0, NCH>(taddr_row, c0, op, l);
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
    float mx = -INFINITY;
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int col = c0 + 16 * ch + 4 * q;
            float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
            if (col < op) b = *reinterpret_cast<const float4*>(b3 + col);
            const float bb[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int k = 16 * ch + 4 * q + j;
                const bool in = (col + j >= lo) && (col + j < hi);
                l[k] = in ? l[k] + bb[j] : -INFINITY;
                mx = fmaxf(mx, l[k]);
            }
        }
    }
    if (logits_row) {
#pragma unroll
        for (int k = 0; k < NCH * 16; ++k)
            if (c0 + k >= lo && c0 + k < hi) logits_row[c0 + k] = l[k];
    }
    const float mneg = -mx * 1.4426950408889634f;
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < NCH * 16; ++k) {
        l[k] = exp2f(__fmaf_rn(l[k], 1.4426950408889634f, mneg));  // exp(l - max); 0 for masked columns
        s += l[k];
    }
    const float target = u * s;
    float cum = 0.0f;
    int below = 0;  // number of leading window slots whose cumulative weight is <= target
#pragma unroll
    for (int k = 0; k < NCH * 16; ++k) {
        cum += l[k];
        below += (cum <= target) ? 1 : 0;
    }
    int pick = c0 + below - lo;  // cum is non-decreasing: `below` slots precede the first index with target < cum
    const int last = hi - lo - 1;
    pick = pick < 0 ? 0 : pick;
    return pick > last ? last : pick;
}

// Fallback for heads wider than 80 logits: three sweeps over the TMEM row (maximum; sum of
// exp(l - max); first index whose cumulative weight exceeds u * sum).
__device__ __forceinline__ int sample_head_sweeps(uint32_t taddr_row, const float* b3, int lo, int hi, float u, float* logits_row) {
    float mx = -INFINITY;
    for (int c = lo & ~15; c < hi; c += 16) {
        float v[16];
        tmem_ld16(taddr_row + c, v);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int col = c + j;
            if (col >= lo && col < hi) {
                const float l = v[j] + b3[col];
                if (logits_row) logits_row[col] = l;
                mx = fmaxf(mx, l);
            }
        }
    }
    float s = 0.0f;
    for (int c = lo & ~15; c < hi; c += 16) {
        float v[16];
        tmem_ld16(taddr_row + c, v);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int col = c + j;
            if (col >= lo && col < hi) s += __expf(v[j] + b3[col] - mx);
        }
    }
    const float target = u * s;
    float cum = 0.0f;
    int pick = hi - lo - 1;
    bool found = false;
    for (int c = lo & ~15; c < hi; c += 16) {
        float v[16];
        tmem_ld16(taddr_row + c, v);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int col = c + j;
            if (col >= lo && col < hi) {
                cum += __expf(v[j] + b3[col] - mx);
                if (!found && target < cum) { pick = col - lo; found = true; }
            }
        }
    }
    return pick;
}

// f1 masked categorical for a single-head row: unavailable actions are left out of
// the maximum, the sum and the running sum (their probability is exactly 0).  Out of line and
// sweep-based: the unmasked samplers keep their registers; this path is an option, not the headline.
__device__ __noinline__ int sample_head_masked(uint32_t taddr_row, const float* b3, int n_logits, float u, float* logits_row,
                                               const PolicyMask& k, const uint8_t* blob, int agent) {
    unsigned long long av[4] = {0ull, 0ull, 0ull, 0ull};
    auto set = [&](int a) {
        const unsigned long long bit = 1ull << (a & 63);
        const int w = a >> 6;
        av[0] |= w == 0 ? bit : 0ull; av[1] |= w == 1 ? bit : 0ull; av[2] |= w == 2 ? bit : 0ull; av[3] |= w == 3 ? bit : 0ull;
    };
    const float coin = ((const float*)(blob + k.o_coin))[agent];
    const bool room = __popc(((const uint32_t*)(blob + k.o_mask))[agent]) < k.M;
    const int* inv = (const int*)(blob + k.o_inv);
    int enough = 0;
    for (int r = 0; r < k.R; ++r) {
        set(r);  // gather: always
        enough += inv[r * k.NS + agent] >= k.craft_units;
    }
    if (k.craft_mode == EJ_CRAFT_PER_RESOURCE) {
        for (int r = 0; r < k.R; ++r)
            if (inv[r * k.NS + agent] >= k.craft_units) set(k.R + r);
    } else if (enough >= k.craft_distinct) {
        set(k.R);
    }
    if (room) {
        for (int r = 0; r < k.R; ++r) {
            const bool has = inv[r * k.NS + agent] >= 1;
            for (int p = 0; p < k.P; ++p) {
                if (coin >= (float)k.prices[p]) set(k.base_buy + r * k.P + p);
                if (has) set(k.base_sell + r * k.P + p);
            }
        }
    }
    if (k.allow_noop) set(k.A - 1);
    auto ok = [&](int col) {
        const int w = col >> 6;
        const unsigned long long word = w == 0 ? av[0] : w == 1 ? av[1] : w == 2 ? av[2] : av[3];
        return ((word >> (col & 63)) & 1ull) != 0ull;
    };
    float mx = -INFINITY;
    for (int c = 0; c < n_logits; c += 16) {
        float v[16];
        tmem_ld16(taddr_row + c, v);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int col = c + j;
            if (col < n_logits) {
                const float l = v[j] + b3[col];
                if (logits_row) logits_row[col] = l;
                if (ok(col)) mx = fmaxf(mx, l);
            }
        }
    }
    float s = 0.0f;
    for (int c = 0; c < n_logits; c += 16) {
        float v[16];
        tmem_ld16(taddr_row + c, v);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int col = c + j;
            if (col < n_logits && ok(col)) s += __expf(v[j] + b3[col] - mx);
        }
    }
    const float target = u * s;
    float cum = 0.0f;
    int pick = -1, last_ok = 0;
    for (int c = 0; c < n_logits; c += 16) {
        float v[16];
        tmem_ld16(taddr_row + c, v);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int col = c + j;
            if (col < n_logits && ok(col)) {
                cum += __expf(v[j] + b3[col] - mx);
                last_ok = col;
                if (pick < 0 && target < cum) pick = col;
            }
        }
    }
    return pick >= 0 ? pick : last_ok;
}

__device__ __forceinline__ void group_sync(int grp) { asm volatile("bar.sync %0, %1;\n" ::"r"(grp + 1), "r"(PTILE) : "memory"); }

// 1-D TMA bulk copy global -> shared, completion on an mbarrier (bytes and both addresses multiples of 16).
__device__ __forceinline__ void tma_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(dst), "l"(src), "r"(bytes),
                 "r"(bar)
                 : "memory");
}

__global__ void __launch_bounds__(PGROUPS* PTILE, 1) ej_policy_kernel(const __grid_constant__ PolicyLaunch pl) {
    const bool second = (int)blockIdx.x >= pl.split;
    const PolicyArgs& a = second ? pl.job[1] : pl.job[0];
    const int bid = second ? (int)blockIdx.x - pl.split : (int)blockIdx.x, nblk = second ? (int)gridDim.x - pl.split : pl.split;
    extern __shared__ __align__(128) uint8_t psm[];
    __shared__ __align__(8) unsigned long long mbar_mma[PGROUPS], mbar_tma[PGROUPS];
    __shared__ uint32_t tmem_slot;
    const int tid = threadIdx.x, warp = tid >> 5, grp = tid >> 7, gtid = tid & (PTILE - 1);
    const PolicyNet& n = a.net;
    uint8_t* A = psm + a.smem_group + grp * a.group_bytes;
    const float* stage = reinterpret_cast<const float*>(A + a.stage_off);
    const float* b1 = reinterpret_cast<const float*>(psm + a.smem_bias);
    const float* b2 = b1 + PH;
    const float* b3 = b2 + PH;

    // ---- one-time setup: weights to shared memory (once per SM), mbarriers, TMEM ----
    {
        const uint4* src = reinterpret_cast<const uint4*>(n.blob);
        uint4* dst = reinterpret_cast<uint4*>(psm + a.smem_W1);  // W1 | W2 | W3 | biases are contiguous in both
        for (int i = tid; i < n.blob_bytes / 16; i += PGROUPS * PTILE) dst[i] = src[i];
    }
    if (tid == 0) {
        for (int g = 0; g < PGROUPS; ++g) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(smem_u32(&mbar_mma[g])) : "memory");
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(smem_u32(&mbar_tma[g])) : "memory");
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(&tmem_slot)), "r"(P_TMEM_ALLOC) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");  // weights were written by the generic proxy
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const uint32_t tmem_base = tmem_slot;
    const uint32_t tmem = tmem_base + (uint32_t)(grp * a.tmem_cols);           // this group's columns
    const uint32_t taddr_row = tmem + ((uint32_t)((warp & 3) * 32) << 16);     // this warp's 32 lanes
    const uint32_t bar = smem_u32(&mbar_mma[grp]), tbar = smem_u32(&mbar_tma[grp]);
    const uint32_t a_addr = smem_u32(A), stage_addr = smem_u32(stage), w1_addr = smem_u32(psm + a.smem_W1),
                   w2_addr = smem_u32(psm + a.smem_W2), w3_addr = smem_u32(psm + a.smem_W3);
    uint32_t phase = 0, tphase = 0;

    const int n_tiles = (a.rows + PTILE - 1) / PTILE;
    const int tile_step = nblk * a.groups;
    // a tile's rows are contiguous in global memory; TMA needs 16-byte multiples
    auto tile_rows = [&](int tile) { const int left = a.rows - tile * PTILE; return left < PTILE ? left : PTILE; };
    auto tile_bytes = [&](int tile) { return (uint32_t)(tile_rows(tile) * a.row_stride * 4); };
    auto tile_src = [&](int tile) { return a.obs + (size_t)tile * PTILE * a.row_stride; };
    auto tma_ok = [&](int tile) { return ((reinterpret_cast<uintptr_t>(tile_src(tile)) | tile_bytes(tile)) & 15u) == 0; };
    int tile = grp < a.groups ? bid * a.groups + grp : n_tiles;  // surplus groups idle
    if (tile < n_tiles && gtid == 0 && tma_ok(tile)) tma_load_1d(stage_addr, tile_src(tile), tile_bytes(tile), tbar);

    for (; tile < n_tiles; tile += tile_step) {
        const int row0 = tile * PTILE, nrows = tile_rows(tile);
        // ---- observation tile (fp32, staged) -> bf16 A operand (K1p columns, zero padded) ----
        if (tma_ok(tile)) {
            mbar_wait(tbar, tphase);
            tphase ^= 1;
        } else {  // unaligned tile: plain coalesced copy by the group
            float* st = const_cast<float*>(stage);
            const float* src = tile_src(tile);
            for (int i = gtid; i < nrows * a.row_stride; i += PTILE) st[i] = src[i];
            group_sync(grp);
        }
        {
            const float* my = stage + gtid * a.row_stride;
            for (int kc = 0; kc < n.K1p / 8; ++kc) {
                uint32_t w[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int k = kc * 8 + 2 * j;
                    const float v0 = (gtid < nrows && k < n.D_in) ? my[k] : 0.0f;
                    const float v1 = (gtid < nrows && k + 1 < n.D_in) ? my[k + 1] : 0.0f;
                    const __nv_bfloat162 h = __floats2bfloat162_rn(v0, v1);
                    w[j] = *reinterpret_cast<const uint32_t*>(&h);
                }
                *reinterpret_cast<uint4*>(A + op_off(gtid, kc * 8, n.K1p)) = make_uint4(w[0], w[1], w[2], w[3]);
            }
        }
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        group_sync(grp);
        if (gtid == 0) {
            issue_layer(a_addr, w1_addr, n.K1p, PH, tmem, bar);
            const int next = tile + tile_step;  // the staging buffer is free: prefetch the group's next tile
            if (next < n_tiles && tma_ok(next)) tma_load_1d(stage_addr, tile_src(next), tile_bytes(next), tbar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
        hidden_epilogue(taddr_row, b1, A, gtid);
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        group_sync(grp);
        if (gtid == 0) issue_layer(a_addr, w2_addr, PH, PH, tmem, bar);
        mbar_wait(bar, phase);
        phase ^= 1;
        hidden_epilogue(taddr_row, b2, A, gtid);
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        group_sync(grp);
        if (gtid == 0) issue_layer(a_addr, w3_addr, PH, n.Op, tmem, bar);
        mbar_wait(bar, phase);
        phase ^= 1;
        asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");

        // ---- logits -> softmax -> inverse-CDF sample per head (G33) ----
        const int row = row0 + gtid;
        const bool live = gtid < nrows;
        const int env = live ? row / a.rows_per_env : 0;
        const int agent = a.fixed_agent >= 0 ? a.fixed_agent : row - env * a.rows_per_env;
        const int t = live ? *reinterpret_cast<const int*>(a.state + (size_t)env * a.blob_stride) : 0;
        uint32_t x[4] = {0, 0, 0, 0};
        for (int h = 0; h < n.n_heads; ++h) {
            if ((h & 3) == 0)
                philox4x32_10(a.env_id_base + (uint32_t)env, (uint32_t)agent, (uint32_t)t, a.stream_base + (uint32_t)(h >> 2), a.seed_lo,
                              a.seed_hi, x[0], x[1], x[2], x[3]);
            const uint32_t xw = (h & 3) == 0 ? x[0] : (h & 3) == 1 ? x[1] : (h & 3) == 2 ? x[2] : x[3];
            const float u = u01(xw);
            const int lo = h * n.head, hi = lo + n.head;
            float* lrow = (a.logits && live) ? a.logits + (size_t)row * n.n_out : nullptr;
            int pick;
            if (a.mask.on) {  // f1: single-head population job (uniform over the CTA)
                pick = sample_head_masked(taddr_row, b3, n.n_out, u, lrow, a.mask, a.state + (size_t)env * a.blob_stride, agent);
            } else
            switch (n.nch) {
                case 1: pick = sample_head<1>(taddr_row, b3, lo, hi, n.Op, u, lrow); break;
                case 2: pick = sample_head<2>(taddr_row, b3, lo, hi, n.Op, u, lrow); break;
                case 3: pick = sample_head<3>(taddr_row, b3, lo, hi, n.Op, u, lrow); break;
                case 4: pick = sample_head<4>(taddr_row, b3, lo, hi, n.Op, u, lrow); break;
                case 5: pick = sample_head<5>(taddr_row, b3, lo, hi, n.Op, u, lrow); break;
                default: pick = sample_head_sweeps(taddr_row, b3, lo, hi, u, lrow); break;
            }
            if (live) a.actions[(size_t)row * n.n_heads + h] = pick;
        }
        // the next tile's MMAs overwrite these TMEM columns and the A tile
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        group_sync(grp);
    }

    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem_base), "r"(P_TMEM_ALLOC) : "memory");
}

}  // namespace
