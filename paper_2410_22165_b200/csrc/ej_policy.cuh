// ej_policy.cuh -- a12 of the hot path (BASELINE.json configs[4]): forward pass of the shared
// population policy MLP and of the government MLP (obs -> 128 -> 128 -> logits, tanh; P:240,
// Table 2) on the 5th-generation tensor cores, followed by categorical sampling with
// the counter-based Philox of G30 (G33).
//
// Groups of 128 threads work on tiles of 128 observation rows (thread i = row i = TMEM lane i).  The three weight
// matrices stay resident in shared memory in the canonical K-major no-swizzle UMMA layout (8-row x 16-byte core
// matrices); the activation tile is rebuilt in the same layout between layers.  Each layer is a chain of
// tcgen05.mma (M=128, N=128|Op, K=16) issued by one thread, accumulating in TMEM; completion comes back through
// tcgen05.commit on an mbarrier; the epilogue reads its row with tcgen05.ld, adds the bias, applies tanh, rounds
// to bf16 and writes the next layer's A operand.  One CTA per SM holds the weights once and runs two such groups;
// every group keeps two tiles in flight so that one tile's epilogue overlaps the other's MMAs (see ej_policy_kernel).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int PH = 128;        // hidden width (B:configs[4]: 128 -> 128)
constexpr int PTILE = 128;     // rows per tile = UMMA M
constexpr int P_TMEM_ALLOC = 512;  // whole TMEM of the SM (one CTA per SM); group g uses columns [g * tmem_cols, ...)
constexpr int P_THREADS = 2 * 128 + 2 * 32;  // two row groups + one MMA-issuer warp per group
constexpr int PGROUPS = 2;         // 128-thread groups per CTA (a job may use fewer); every group keeps two tiles in flight

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
    int o_episode;           // byte offset of the episode index in a blob (f4: part of the Philox counter)
    uint32_t env_id_base, seed_lo, seed_hi;
    uint32_t stream_base;    // Philox stream of head 0 (population 0, government 1); head h uses word h % 4 of stream + h / 4
    int32_t* actions;        // [rows][n_heads]
    float* logits;           // [rows][n_out] or null
    int smem_W1, smem_W2, smem_W3, smem_bias;  // byte offsets in dynamic shared memory (shared by both groups)
    int smem_group, slot_bytes, stage_off;      // slot s of group g: operand buffer at smem_group + (2 g + s) * slot_bytes, fp32 rows at + stage_off
    int groups, tmem_cols;   // active groups of this job (<= PGROUPS) and TMEM columns per slot (128 or 256)
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

// Issue one layer: D[128 x n] (+)= A[128 x kp] * W[n x kp]^T, then commit to the mbarrier.  The descriptors of
// successive K steps differ in the start-address field only (+256 B = +16 in units of 16 B): one add per step.
__device__ __forceinline__ void issue_layer(uint32_t a_addr, uint32_t w_addr, int kp, int n, uint32_t tmem_d, uint32_t bar) {
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const uint32_t idesc = umma_idesc(n);
    const uint32_t sbo = (uint32_t)kp * 16u;  // (kp / 8) core matrices of 128 B per 8-row group
    uint64_t da = umma_desc(a_addr, 128, sbo), db = umma_desc(w_addr, 128, sbo);
    umma_bf16(tmem_d, da, db, idesc, 0u);
#pragma unroll 1
    for (int k = 1; k < kp / 16; ++k) {
        da += 16u;
        db += 16u;
        umma_bf16(tmem_d, da, db, idesc, 1u);
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

__device__ __forceinline__ void tmem_ld32_nowait(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];\n"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
          "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
          "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
}

// Hidden-layer epilogue: this thread's accumulator row -> +bias -> tanh -> bf16 -> A operand (kp = 128).
// Out of line: compiled on its own, ptxas keeps the order written here; inlined into the kernel it paired every
// tanh with its pack.
template <int OFF>
__device__ __forceinline__ void tmem_ld32_into(uint32_t taddr, float (&r)[PH]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];\n"
        : "=f"(r[OFF + 0]), "=f"(r[OFF + 1]), "=f"(r[OFF + 2]), "=f"(r[OFF + 3]), "=f"(r[OFF + 4]), "=f"(r[OFF + 5]), "=f"(r[OFF + 6]),
          "=f"(r[OFF + 7]), "=f"(r[OFF + 8]), "=f"(r[OFF + 9]), "=f"(r[OFF + 10]), "=f"(r[OFF + 11]), "=f"(r[OFF + 12]),
          "=f"(r[OFF + 13]), "=f"(r[OFF + 14]), "=f"(r[OFF + 15]), "=f"(r[OFF + 16]), "=f"(r[OFF + 17]), "=f"(r[OFF + 18]),
          "=f"(r[OFF + 19]), "=f"(r[OFF + 20]), "=f"(r[OFF + 21]), "=f"(r[OFF + 22]), "=f"(r[OFF + 23]), "=f"(r[OFF + 24]),
          "=f"(r[OFF + 25]), "=f"(r[OFF + 26]), "=f"(r[OFF + 27]), "=f"(r[OFF + 28]), "=f"(r[OFF + 29]), "=f"(r[OFF + 30]),
          "=f"(r[OFF + 31])
        : "r"(taddr)
        : "memory");
}
// volatile forms: the order of these statements in the source is the order ptxas keeps
__device__ __forceinline__ float tanh_v(float x) { float y; asm volatile("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fadd_v(float a, float b) { float y; asm volatile("add.f32 %0, %1, %2;" : "=f"(y) : "f"(a), "f"(b)); return y; }
__device__ __forceinline__ uint32_t pack_v(float lo, float hi) {  // bf16x2, round to nearest even: lo in bits 0..15
    uint32_t w;
    asm volatile("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(w) : "f"(hi), "f"(lo));
    return w;
}
// The row as ONE software pipeline over its 128 columns: in every slot a tanh (special-function unit: one warp
// instruction per 8 cycles), the bias add of the element 32 columns ahead, and the packing of a pair whose tanh was
// issued 8 slots (64+ cycles) ago, so that the unit is fed back to back across the whole row while the adds, packs and
// stores fill its shadow.  Done chunk by chunk (adds, 32 tanh, packs, then the next chunk) the unit idled during every
// chunk's adds and packs: 4,700 cycles per tile for the two hidden layers against 2 x 1,024 of pure tanh issue.
__device__ __noinline__ void hidden_epilogue(uint32_t taddr_row, const float* bias, uint8_t* A, int row) {
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    float x[PH];
    tmem_ld32_into<0>(taddr_row, x);
    tmem_ld32_into<32>(taddr_row + 32, x);
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
    tmem_ld32_into<64>(taddr_row + 64, x);
    tmem_ld32_into<96>(taddr_row + 96, x);
#pragma unroll
    for (int g = 0; g < 8; ++g) {  // prologue: bias of the first 32 columns
        const float4 b4 = *reinterpret_cast<const float4*>(bias + g * 4);
        x[4 * g] = fadd_v(x[4 * g], b4.x);
        x[4 * g + 1] = fadd_v(x[4 * g + 1], b4.y);
        x[4 * g + 2] = fadd_v(x[4 * g + 2], b4.z);
        x[4 * g + 3] = fadd_v(x[4 * g + 3], b4.w);
    }
    uint32_t w[4];
    float4 b4 = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int k = 0; k < PH; ++k) {
        x[k] = tanh_v(x[k]);
        if (k + 32 < PH) {
            if (k + 32 == 64) asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");  // columns 64..127 have arrived long ago
            if ((k & 3) == 0) b4 = *reinterpret_cast<const float4*>(bias + k + 32);
            x[k + 32] = fadd_v(x[k + 32], (k & 3) == 0 ? b4.x : (k & 3) == 1 ? b4.y : (k & 3) == 2 ? b4.z : b4.w);
        }
        const int j = k - 9;  // pair (j, j + 1): the younger tanh was issued 8 slots ago
        if (j >= 0 && (j & 1) == 0) {
            w[(j >> 1) & 3] = pack_v(x[j], x[j + 1]);
            if ((j & 7) == 6) *reinterpret_cast<uint4*>(A + op_off(row, j - 6, PH)) = make_uint4(w[0], w[1], w[2], w[3]);
        }
    }
#pragma unroll
    for (int j = PH - 8; j < PH; j += 2) w[(j >> 1) & 3] = pack_v(x[j], x[j + 1]);  // the pairs of the last 8 slots
    *reinterpret_cast<uint4*>(A + op_off(row, PH - 8, PH)) = make_uint4(w[0], w[1], w[2], w[3]);
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

__device__ __forceinline__ float ex2_fast(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// The population head when its width NL is a compile-time constant (one head, columns 0 .. NL-1): the row of
// logits is read once, and every later pass (bias, maximum, exponentials, sum, cumulative count) touches exactly
// the NL live columns -- about 8 instructions per logit where the general window sampler spends 17.
template <int NL>
__device__ __forceinline__ int sample_single_head(uint32_t taddr_row, const float* b3, float u, float* logits_row) {
    constexpr int NCH = (NL + 15) / 16;
    float l[NCH * 16];
    load_window<0, NCH>(taddr_row, 0, NCH * 16, l);
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
    float m4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};  // four running maxima: short dependence chains
#pragma unroll
    for (int q = 0; q < (NL + 3) / 4; ++q) {
        const float4 b = *reinterpret_cast<const float4*>(b3 + 4 * q);  // b3 is padded to a multiple of 16 floats
        const float bb[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (4 * q + j < NL) {
                l[4 * q + j] += bb[j];
                m4[j] = fmaxf(m4[j], l[4 * q + j]);
            }
        }
    }
    const float mx = fmaxf(fmaxf(m4[0], m4[1]), fmaxf(m4[2], m4[3]));
    if (logits_row) {
#pragma unroll
        for (int k = 0; k < NL; ++k) logits_row[k] = l[k];
    }
    const float mneg = -mx * 1.4426950408889634f;
#pragma unroll
    for (int k = 0; k < NL; ++k) l[k] = ex2_fast(__fmaf_rn(l[k], 1.4426950408889634f, mneg));  // exp(l - max)
    // running sums in the order of the definition (left to right, never reassociated); the total is the last one,
    // and the sampled index = number of running sums <= u * total: 65 independent compares, no second chain
#pragma unroll
    for (int k = 1; k < NL; ++k) l[k] += l[k - 1];
    const float target = u * l[NL - 1];
    int below = 0;
#pragma unroll
    for (int k = 0; k < NL; ++k) below += (l[k] <= target) ? 1 : 0;
    return below > NL - 1 ? NL - 1 : below;
}

// Several equal heads whose count and width are compile-time constants (the government's B = 7 brackets of L = 21
// rate levels): head H covers the columns [H * HEAD, (H + 1) * HEAD); its 16-column chunks and every register
// index are known at compile time, so each head costs what sample_single_head costs per logit.  The general window
// sampler (runtime bounds, masked padding columns, exp2f) made a government tile several times as expensive as a
// population tile, and the few government CTAs the tail of the whole launch.
template <int H, int NH, int HEAD>
struct HeadSampler {
    template <class PH_>
    __device__ __forceinline__ static void run(uint32_t taddr_row, const float* b3, float* logits_row, int32_t* out, bool live, PH_&& next_u) {
        constexpr int LO = H * HEAD, HI = LO + HEAD, C0 = LO & ~15, NCH = (HI - C0 + 15) / 16;
        float l[NCH * 16];
        load_window<0, NCH>(taddr_row, C0, C0 + NCH * 16, l);
        const float u = next_u(H);
        asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
        float m4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
        for (int k = LO - C0; k < HI - C0; ++k) {
            l[k] += b3[C0 + k];
            m4[k & 3] = fmaxf(m4[k & 3], l[k]);
        }
        const float mx = fmaxf(fmaxf(m4[0], m4[1]), fmaxf(m4[2], m4[3]));
        if (logits_row) {
#pragma unroll
            for (int k = LO - C0; k < HI - C0; ++k) logits_row[C0 + k] = l[k];
        }
        const float mneg = -mx * 1.4426950408889634f;
#pragma unroll
        for (int k = LO - C0; k < HI - C0; ++k) l[k] = ex2_fast(__fmaf_rn(l[k], 1.4426950408889634f, mneg));
#pragma unroll
        for (int k = LO - C0 + 1; k < HI - C0; ++k) l[k] += l[k - 1];  // running sums, left to right
        const float target = u * l[HI - C0 - 1];
        int below = 0;
#pragma unroll
        for (int k = LO - C0; k < HI - C0; ++k) below += (l[k] <= target) ? 1 : 0;
        if (live) out[H] = below > HEAD - 1 ? HEAD - 1 : below;
        if constexpr (H + 1 < NH) HeadSampler<H + 1, NH, HEAD>::run(taddr_row, b3, logits_row, out, live, next_u);
    }
};

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

// The kernel.  A CTA holds the three weight matrices once and runs PGROUPS groups of 128 threads (thread = row =
// TMEM lane).  Every group keeps TWO tiles in flight (slots 0 and 1: own operand buffer, own TMEM accumulator
// columns, own mbarriers) and works through them phase by phase -- operand build, tanh epilogue 1, tanh epilogue 2,
// sampling -- first for slot 0, then for slot 1: while the threads run one slot's epilogue on the special-function
// unit, the tensor cores run the other slot's MMAs, so a group never sits on an MMA wait (the first version ran one
// tile per group and three groups in step: 45 % of a tile's time was operand builds and MMA waits with the
// special-function unit idle, profiles/r2d).  A slot's buffer holds, in turn, the fp32 observation rows (1-D TMA bulk
// copy, issued as soon as the slot's last MMA is done, so it lands under the sampling), the layer-1 operand built
// from them (beside the rows), then the hidden activations (over both).
__global__ void __launch_bounds__(P_THREADS, 1) ej_policy_kernel(const __grid_constant__ PolicyLaunch pl) {
    const bool second = (int)blockIdx.x >= pl.split;
    const PolicyArgs& a = second ? pl.job[1] : pl.job[0];
    const int bid = second ? (int)blockIdx.x - pl.split : (int)blockIdx.x, nblk = second ? (int)gridDim.x - pl.split : pl.split;
    extern __shared__ __align__(128) uint8_t psm[];
    __shared__ __align__(8) unsigned long long mbar_mma[PGROUPS][2], mbar_tma[PGROUPS][2], mbar_rdy[PGROUPS][2], mbar_w;
    __shared__ uint32_t tmem_slot;
    const int tid = threadIdx.x, warp = tid >> 5, gtid = tid & (PTILE - 1);
    const bool issuer = tid >= PGROUPS * PTILE;                       // warps 8, 9: MMA issuers of groups 0, 1
    const int grp = issuer ? (tid - PGROUPS * PTILE) >> 5 : tid >> 7;
    const PolicyNet& n = a.net;
    const float* b1 = reinterpret_cast<const float*>(psm + a.smem_bias);
    const float* b2 = b1 + PH;
    const float* b3 = b2 + PH;

    // ---- one-time setup: weights to shared memory (once per SM, one TMA bulk copy), mbarriers, TMEM ----
    if (tid == 0) {
        for (int g = 0; g < PGROUPS; ++g)
            for (int sl = 0; sl < 2; ++sl) {
                asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(smem_u32(&mbar_mma[g][sl])) : "memory");
                asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(smem_u32(&mbar_tma[g][sl])) : "memory");
                asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(&mbar_rdy[g][sl])), "r"(PTILE) : "memory");
            }
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(smem_u32(&mbar_w)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        tma_load_1d(smem_u32(psm + a.smem_W1), n.blob, (uint32_t)n.blob_bytes, smem_u32(&mbar_w));  // W1 | W2 | W3 | biases, contiguous in both
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(&tmem_slot)), "r"(P_TMEM_ALLOC) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    mbar_wait(smem_u32(&mbar_w), 0);  // the weights have landed (async proxy: visible to the MMAs and, after this wait, to every thread)
    const uint32_t tmem_base = tmem_slot;
    const uint32_t w1_addr = smem_u32(psm + a.smem_W1), w2_addr = smem_u32(psm + a.smem_W2), w3_addr = smem_u32(psm + a.smem_W3);

    const int n_tiles = (a.rows + PTILE - 1) / PTILE;
    const int tile_step = nblk * a.groups;
    // a tile's rows are contiguous in global memory; TMA needs 16-byte multiples
    auto tile_rows = [&](int tile) { const int left = a.rows - tile * PTILE; return left < PTILE ? left : PTILE; };
    auto tile_bytes = [&](int tile) { return (uint32_t)(tile_rows(tile) * a.row_stride * 4); };
    auto tile_src = [&](int tile) { return a.obs + (size_t)tile * PTILE * a.row_stride; };
    auto tma_ok = [&](int tile) { return ((reinterpret_cast<uintptr_t>(tile_src(tile)) | tile_bytes(tile)) & 15u) == 0; };

    // per-slot state of this group
    uint8_t* const gbase = psm + a.smem_group + grp * (2 * a.slot_bytes);
    int tile[2];
    int t_env[2] = {0, 0}, ep_env[2] = {0, 0};  // clock and episode of the row's env (Philox counter), fetched while the slot's operand is built
    uint32_t ph_mma[2] = {0u, 0u}, ph_tma[2] = {0u, 0u};
    auto slotA = [&](int sl) { return gbase + sl * a.slot_bytes; };
    auto slotStage = [&](int sl) { return reinterpret_cast<float*>(gbase + sl * a.slot_bytes + a.stage_off); };
    auto slotTmem = [&](int sl) { return tmem_base + (uint32_t)((grp * 2 + sl) * a.tmem_cols); };
    auto rowTmem = [&](int sl) { return slotTmem(sl) + ((uint32_t)((warp & 3) * 32) << 16); };  // this warp's 32 lanes
    auto barM = [&](int sl) { return smem_u32(&mbar_mma[grp][sl]); };
    auto barT = [&](int sl) { return smem_u32(&mbar_tma[grp][sl]); };
    const int first = grp < a.groups ? bid * a.groups + grp : n_tiles;  // surplus groups idle
    tile[0] = first;
    tile[1] = first < n_tiles ? first + tile_step : n_tiles;
    auto barR = [&](int sl) { return smem_u32(&mbar_rdy[grp][sl]); };
    if (issuer) {
        // MMA-issuer warp of group `grp`: one lane waits for "operand ready" (all 128 rows of the group have written and
        // fenced their part) and issues the layer's MMAs, in the order in which the group produces operands.  The row
        // threads never wait for the tensor pipe to accept an instruction; they only wait for results.
        if ((tid & 31) == 0) {
            uint32_t ph_rdy[2] = {0u, 0u};
            while (tile[0] < n_tiles) {
#pragma unroll 1
                for (int stage_i = 0; stage_i < 3; ++stage_i) {
#pragma unroll 1
                    for (int sl = 0; sl < 2; ++sl) {
                        if (tile[sl] >= n_tiles) break;
                        mbar_wait(barR(sl), ph_rdy[sl]);
                        ph_rdy[sl] ^= 1u;
                        const uint32_t a_addr = smem_u32(slotA(sl));
                        if (stage_i == 0) issue_layer(a_addr, w1_addr, n.K1p, PH, slotTmem(sl), barM(sl));
                        else if (stage_i == 1) issue_layer(a_addr, w2_addr, PH, PH, slotTmem(sl), barM(sl));
                        else issue_layer(a_addr, w3_addr, PH, n.Op, slotTmem(sl), barM(sl));
                    }
                }
                tile[0] += 2 * tile_step;
                tile[1] += 2 * tile_step;
            }
        }
        tile[0] = tile[1] = n_tiles;  // skip the row-group code below
    }
#pragma unroll
    for (int sl = 0; sl < 2; ++sl)
        if (tile[sl] < n_tiles && gtid == 0 && tma_ok(tile[sl])) tma_load_1d(smem_u32(slotStage(sl)), tile_src(tile[sl]), tile_bytes(tile[sl]), barT(sl));

    while (tile[0] < n_tiles) {
        // ---- observation rows (fp32, staged) -> bf16 layer-1 operand (K1p columns, zero padded); layer-1 MMAs ----
#pragma unroll 1
        for (int sl = 0; sl < 2; ++sl) {
            if (tile[sl] >= n_tiles) break;
            const int nrows = tile_rows(tile[sl]);
            uint8_t* A = slotA(sl);
            float* stage = slotStage(sl);
            if (tma_ok(tile[sl])) {
                mbar_wait(barT(sl), ph_tma[sl]);
                ph_tma[sl] ^= 1u;
            } else {  // unaligned tile: plain coalesced copy by the group
                const float* src = tile_src(tile[sl]);
                for (int i = gtid; i < nrows * a.row_stride; i += PTILE) stage[i] = src[i];
                group_sync(grp);
            }
            {   // the sampler's Philox counter needs the env's clock: a global load, issued a whole tile ahead of its use
                const int row = tile[sl] * PTILE + gtid;
                const uint8_t* blob = a.state + (size_t)(row / a.rows_per_env) * a.blob_stride;
                t_env[sl] = gtid < nrows ? *reinterpret_cast<const int*>(blob) : 0;
                ep_env[sl] = gtid < nrows ? *reinterpret_cast<const int*>(blob + a.o_episode) : 0;
            }
            const float* my = stage + gtid * a.row_stride;
            const bool in_tile = gtid < nrows;
            for (int k0 = 0; k0 < n.K1p; k0 += 48) {  // 48 columns at a time: all loads in flight before the first conversion
                float v[48];
#pragma unroll
                for (int j = 0; j < 48; ++j) v[j] = (in_tile && k0 + j < n.D_in) ? my[k0 + j] : 0.0f;  // zero padding, rows beyond the tile
#pragma unroll
                for (int c8 = 0; c8 < 6; ++c8) {
                    if (k0 + c8 * 8 < n.K1p) {
                        uint32_t w[4];
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const __nv_bfloat162 h = __floats2bfloat162_rn(v[c8 * 8 + 2 * j], v[c8 * 8 + 2 * j + 1]);
                            w[j] = *reinterpret_cast<const uint32_t*>(&h);
                        }
                        *reinterpret_cast<uint4*>(A + op_off(gtid, k0 + c8 * 8, n.K1p)) = make_uint4(w[0], w[1], w[2], w[3]);
                    }
                }
            }
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
            // operand written and fenced; this thread has also finished sampling the slot's previous tile (TMEM columns reused)
            asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(barR(sl)) : "memory");
        }
        // ---- hidden layers: tanh epilogue of one slot under the MMAs of the other ----
#pragma unroll 1
        for (int layer = 0; layer < 2; ++layer) {
#pragma unroll 1
            for (int sl = 0; sl < 2; ++sl) {
                if (tile[sl] >= n_tiles) break;
                uint8_t* A = slotA(sl);
                mbar_wait(barM(sl), ph_mma[sl]);
                ph_mma[sl] ^= 1u;
                hidden_epilogue(rowTmem(sl), layer == 0 ? b1 : b2, A, gtid);
                asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
                asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
                asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(barR(sl)) : "memory");
            }
        }
        // ---- logits -> softmax -> inverse-CDF sample per head (G33) ----
#pragma unroll 1
        for (int sl = 0; sl < 2; ++sl) {
            if (tile[sl] >= n_tiles) break;
            const int cur = tile[sl], nrows = tile_rows(cur);
            const uint32_t taddr_row = rowTmem(sl);
            mbar_wait(barM(sl), ph_mma[sl]);
            ph_mma[sl] ^= 1u;
            asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
            // the slot's operand buffer is free: fetch the observation rows of its next tile under the sampling
            tile[sl] = cur + 2 * tile_step;
            if (tile[sl] < n_tiles && gtid == 0 && tma_ok(tile[sl]))
                tma_load_1d(smem_u32(slotStage(sl)), tile_src(tile[sl]), tile_bytes(tile[sl]), barT(sl));
            const int row = cur * PTILE + gtid;
            const bool live = gtid < nrows;
            const int env = live ? row / a.rows_per_env : 0;
            const int agent = a.fixed_agent >= 0 ? a.fixed_agent : row - env * a.rows_per_env;
            const int t = t_env[sl];
            const uint32_t ep_bits = (uint32_t)ep_env[sl] << 8;  // G44
            uint32_t x[4] = {0, 0, 0, 0};
            if (!a.mask.on && n.n_heads == 7 && n.head == 21) {  // the government's 7 brackets x 21 levels
                float* lrow = (a.logits && live) ? a.logits + (size_t)row * n.n_out : nullptr;
                auto next_u = [&](int h) {
                    if ((h & 3) == 0)
                        philox4x32_10(a.env_id_base + (uint32_t)env, (uint32_t)agent, (uint32_t)t, (a.stream_base + (uint32_t)(h >> 2)) | ep_bits, a.seed_lo,
                                      a.seed_hi, x[0], x[1], x[2], x[3]);
                    return u01((h & 3) == 0 ? x[0] : (h & 3) == 1 ? x[1] : (h & 3) == 2 ? x[2] : x[3]);
                };
                HeadSampler<0, 7, 21>::run(taddr_row, b3, lrow, a.actions + (size_t)row * 7, live, next_u);
            } else
            for (int h = 0; h < n.n_heads; ++h) {
                if ((h & 3) == 0)
                    philox4x32_10(a.env_id_base + (uint32_t)env, (uint32_t)agent, (uint32_t)t, (a.stream_base + (uint32_t)(h >> 2)) | ep_bits, a.seed_lo,
                                  a.seed_hi, x[0], x[1], x[2], x[3]);
                const uint32_t xw = (h & 3) == 0 ? x[0] : (h & 3) == 1 ? x[1] : (h & 3) == 2 ? x[2] : x[3];
                const float u = u01(xw);
                const int lo = h * n.head, hi = lo + n.head;
                float* lrow = (a.logits && live) ? a.logits + (size_t)row * n.n_out : nullptr;
                int pick;
                if (a.mask.on) {  // f1: single-head population job (uniform over the CTA)
                    pick = sample_head_masked(taddr_row, b3, n.n_out, u, lrow, a.mask, a.state + (size_t)env * a.blob_stride, agent);
                } else if (n.n_heads == 1 && n.head == 65) {  // R = 3 (BASELINE.json configs[4]): 3 + 1 + 60 + 1 actions
                    pick = sample_single_head<65>(taddr_row, b3, u, lrow);
                } else if (n.n_heads == 1 && n.head == 44) {  // R = 2
                    pick = sample_single_head<44>(taddr_row, b3, u, lrow);
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
            // the slot's next layer-1 MMAs overwrite these TMEM columns: ordered by the fence + group barrier of the next build
            asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        }
    }

    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem_base), "r"(P_TMEM_ALLOC) : "memory");
}

}  // namespace
