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
// to bf16 and writes the next layer's A operand.  Two CTAs per SM overlap one CTA's epilogue
// with the other's MMAs.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int PH = 128;        // hidden width (B:configs[4]: 128 -> 128)
constexpr int PTILE = 128;     // rows per tile = UMMA M
constexpr int P_TMEM_COLS = 256;

struct PolicyNet {
    const uint8_t* blob;   // device: W1 | W2 | W3 (canonical bf16) | b1 | b2 | b3 (f32)
    int D_in, K1p;         // input width and its multiple-of-16 padding
    int n_out, Op;         // logits and their multiple-of-16 padding (<= 256)
    int n_heads, head;     // categorical heads of `head` logits each (n_out = n_heads * head)
    int w1_bytes, w2_bytes, w3_bytes, blob_bytes;
    uint32_t recipK1p;     // ceil(2^32 / K1p)
};

struct PolicyArgs {
    PolicyNet net;
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
    int smem_A, smem_W1, smem_W2, smem_W3, smem_bias;  // byte offsets in dynamic shared memory
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

// Hidden-layer epilogue: this thread's accumulator row -> +bias -> tanh -> bf16 -> A operand (kp = 128).
__device__ __forceinline__ void hidden_epilogue(uint32_t taddr_row, const float* bias, uint8_t* A, int row) {
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
#pragma unroll 4
    for (int c = 0; c < PH; c += 8) {
        float v[8];
        tmem_ld8(taddr_row + c, v);
        uint32_t w[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float a0 = tanh_fast(v[2 * j] + bias[c + 2 * j]), a1 = tanh_fast(v[2 * j + 1] + bias[c + 2 * j + 1]);
            const __nv_bfloat162 h = __floats2bfloat162_rn(a0, a1);
            w[j] = *reinterpret_cast<const uint32_t*>(&h);
        }
        *reinterpret_cast<uint4*>(A + op_off(row, c, PH)) = make_uint4(w[0], w[1], w[2], w[3]);
    }
}

__global__ void __launch_bounds__(PTILE, 2) ej_policy_kernel(const __grid_constant__ PolicyArgs a) {
    extern __shared__ __align__(128) uint8_t psm[];
    __shared__ __align__(8) unsigned long long mbar;
    __shared__ uint32_t tmem_slot;
    const int tid = threadIdx.x, warp = tid >> 5;
    const PolicyNet& n = a.net;
    uint8_t* A = psm + a.smem_A;
    const float* b1 = reinterpret_cast<const float*>(psm + a.smem_bias);
    const float* b2 = b1 + PH;
    const float* b3 = b2 + PH;

    // ---- one-time setup: weights to shared memory, mbarrier, TMEM ----
    {
        const uint4* src = reinterpret_cast<const uint4*>(n.blob);
        uint4* dst = reinterpret_cast<uint4*>(psm + a.smem_W1);  // W1 | W2 | W3 | biases are contiguous in both
        for (int i = tid; i < n.blob_bytes / 16; i += PTILE) dst[i] = src[i];
    }
    const uint32_t bar = smem_u32(&mbar);
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(bar) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(&tmem_slot)), "r"(P_TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");  // weights were written by the generic proxy
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const uint32_t tmem = tmem_slot;
    const uint32_t taddr_row = tmem + ((uint32_t)(warp * 32) << 16);  // this warp's 32 lanes
    const uint32_t a_addr = smem_u32(A), w1_addr = smem_u32(psm + a.smem_W1), w2_addr = smem_u32(psm + a.smem_W2),
                   w3_addr = smem_u32(psm + a.smem_W3);
    uint32_t phase = 0;

    const int n_tiles = (a.rows + PTILE - 1) / PTILE;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int row0 = tile * PTILE;
        // ---- observation tile -> bf16 A operand (K1p columns, zero padded) ----
        for (int idx = tid; idx < PTILE * n.K1p; idx += PTILE) {
            const int r = (int)__umulhi((uint32_t)idx, n.recipK1p), k = idx - r * n.K1p;
            float v = 0.0f;
            if (k < n.D_in && row0 + r < a.rows) v = a.obs[(size_t)(row0 + r) * a.row_stride + k];
            *reinterpret_cast<__nv_bfloat16*>(A + op_off(r, k, n.K1p)) = __float2bfloat16_rn(v);
        }
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        __syncthreads();
        if (tid == 0) issue_layer(a_addr, w1_addr, n.K1p, PH, tmem, bar);
        mbar_wait(bar, phase);
        phase ^= 1;
        hidden_epilogue(taddr_row, b1, A, tid);
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        __syncthreads();
        if (tid == 0) issue_layer(a_addr, w2_addr, PH, PH, tmem, bar);
        mbar_wait(bar, phase);
        phase ^= 1;
        hidden_epilogue(taddr_row, b2, A, tid);
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        __syncthreads();
        if (tid == 0) issue_layer(a_addr, w3_addr, PH, n.Op, tmem, bar);
        mbar_wait(bar, phase);
        phase ^= 1;
        asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");

        // ---- logits -> softmax -> inverse-CDF sample per head (G33) ----
        const int row = row0 + tid;
        const bool live = row < a.rows;
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
            // pass 1: running maximum and sum of exp (online softmax), fp32
            float mx = -INFINITY, s = 0.0f;
            for (int c = lo & ~7; c < hi; c += 8) {
                float v[8];
                tmem_ld8(taddr_row + c, v);
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int col = c + j;
                    if (col >= lo && col < hi) {
                        const float l = v[j] + b3[col];
                        if (a.logits && live) a.logits[(size_t)row * n.n_out + col] = l;
                        if (l > mx) { s = s * __expf(mx - l) + 1.0f; mx = l; }
                        else s += __expf(l - mx);
                    }
                }
            }
            // pass 2: first index whose cumulative weight exceeds u * s (last index otherwise)
            const float target = u * s;
            float cum = 0.0f;
            int pick = n.head - 1;
            bool found = false;
            for (int c = lo & ~7; c < hi; c += 8) {
                float v[8];
                tmem_ld8(taddr_row + c, v);
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int col = c + j;
                    if (col >= lo && col < hi) {
                        cum += __expf(v[j] + b3[col] - mx);
                        if (!found && target < cum) { pick = col - lo; found = true; }
                    }
                }
            }
            if (live) a.actions[(size_t)row * n.n_heads + h] = pick;
        }
        // the next tile's MMAs overwrite these TMEM columns and the A tile
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        __syncthreads();
    }

    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem), "r"(P_TMEM_COLS) : "memory");
}

}  // namespace
