// econojax.cu -- C ABI (include/econojax.h) of the batched EconoJax environment step: parameter
// validation, shared-memory layout, kernel launches, canonical state dump.  The kernels are in
// ej_device.cuh.  Everything on the step path runs on the device; this file only marshals.
#include <cuda_runtime.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <map>
#include <mutex>
#include <new>
#include <type_traits>
#include <utility>
#include <vector>

#include "ej_device.cuh"
#include "ej_policy.cuh"

namespace {

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
char g_create_err[256] = "";

int align16(int x) { return (x + 15) & ~15; }

}  // namespace

// Scratch of ej_rollout_noalloc: the state blobs the reset and step kernels work on, which every other entry point
// keeps in memory that ej_create allocates.  File scope, fixed size: every GPU that loads the library holds these
// EJ_NOALLOC_SCRATCH_BYTES until the process exits.  In HOST code this name is a stand-in, not a device address: the
// kernels are given the pointer that cudaGetSymbolAddress returns (noalloc_scratch_ptr below).
static __device__ __align__(256) unsigned char g_noalloc_scratch[EJ_NOALLOC_SCRATCH_BYTES];

struct ej_env {
    DevCfg c;
    ej_params p;
    uint8_t* d_state = nullptr;
    uint32_t* d_cdf = nullptr;
    cudaStream_t stream = 0;
    bool was_reset = false;
    bool masking = false;  // f1: generator-drawn actions respect the action mask
    int64_t launches = 0;
    char err[256] = "";
    // staging for ej_step_host
    int32_t *d_act = nullptr, *d_gov = nullptr;
    float *d_obs = nullptr, *d_rew = nullptr;
    uint8_t* d_done = nullptr;
    // staging for ej_step_host_factored: one allocation, byte offsets of its sections
    uint8_t* d_fx = nullptr;
    size_t fx_act = 0, fx_gov = 0, fx_priv = 0, fx_shared = 0, fx_govrow = 0, fx_rew = 0, fx_done = 0;
    // a12: installed policies and the buffers the policy-driven rollout chains through
    bool has_policy = false;
    PolicyNet pop_net{}, gov_net{};
    uint8_t *d_pop_blob = nullptr, *d_gov_blob = nullptr;
    float* d_pobs = nullptr;
    int32_t *d_pact = nullptr, *d_pgov = nullptr;
    int n_sms = 148;
    // the step kernel variant of this handle's shape (CTA size, array stride, specialised R / P)
    void (*step_fn)(const DevCfg, uint8_t*, const StepIO) = nullptr;
    void (*step_fn_fx)(const DevCfg, uint8_t*, const StepIO) = nullptr;  // f2: factored observations
    void (*step_fn_ar)(const DevCfg, uint8_t*, const StepIO) = nullptr;  // f4: auto-resetting rollouts
    int step_RT = 0, step_PT = 0, step_pf = 0;
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

// Kernel variants: CTA size NPAD (a power of two >= N) and stride NS of the per-agent arrays:
// NPAD itself, or the tighter 13/16 NPAD when N fits (N = 100: 104 instead of 128, which is what
// brings the headline shape from 7 to 8 resident CTAs per SM).
constexpr int tight_stride(int npad) { return npad >= 64 ? npad / 16 * 13 : npad; }

template <int NPAD, typename F>
int for_stride(int ns, F&& f) {
    if (ns == NPAD) return f(std::integral_constant<int, NPAD>(), std::integral_constant<int, NPAD>());
    return f(std::integral_constant<int, NPAD>(), std::integral_constant<int, tight_stride(NPAD)>());
}

template <typename F>
int for_variant(int Npad, int ns, F&& f) {
#ifdef EJ_DEV_ONLY_128  // development builds: only the N = 65..128 variants (build time)
    return for_stride<128>(ns, f);
#endif
    switch (Npad) {
        case 32: return for_stride<32>(ns, f);
        case 64: return for_stride<64>(ns, f);
        case 128: return for_stride<128>(ns, f);
        case 256: return for_stride<256>(ns, f);
        case 512: return for_stride<512>(ns, f);
        default: return for_stride<1024>(ns, f);
    }
}

// Shapes with a fully specialised step kernel (R, P, N, B and the paper's mechanics as compile-time constants, 16-bit
// order-pool words): BASELINE.json's N = 100 shapes and the paper's section-5 shape r = 4.  select_step_kernel
// instantiates exactly these.
bool is_paper_shape(const DevCfg& c) {
    const bool paper = c.M == 15 && c.Mp_log2 == 4 && c.K == 0 && c.craft_mode == EJ_CRAFT_SINGLE && c.craft_units == 2 &&
                       c.craft_distinct == 2 && c.allow_noop == 1 && c.expiry <= 31;
    if (!paper || c.N != 100 || c.Npad != 128 || c.N4 != tight_stride(128)) return false;
    return (c.P == 10 && c.B == 7 && (c.R == 2 || c.R == 3 || c.R == 6)) || (c.P == 3 && c.B == 3 && c.R == 4);
}

// Shared-memory layout: the NP-only sections come from Lay<NP> (compile-time constants shared
// with the kernels); the R-, P-, M-dependent sections are placed here.
void build_layout(DevCfg& c, bool allow_pool16 = true) {
    const int NP = c.N4, R = c.R, nl = c.n_levels;  // NP: stride of the per-agent arrays
    for_variant(c.Npad, NP, [&](auto, auto ns) {
        using L = Lay<decltype(ns)::value>;
        c.o_key = L::key; c.o_cslot = L::cslot; c.o_anext = L::anext; c.o_cinfo = L::anext; c.o_credit = L::credit;
        c.o_sale = L::sale; c.o_resq = L::resq; c.o_shrow = L::shrow; c.o_govrow = L::govrow; c.o_misc = L::misc;
        c.o_blob = L::blob;
        c.o_coin = L::coin; c.o_labor = L::labor; c.o_income = L::income; c.o_SC = L::SC; c.o_esc_coin = L::esc_coin;
        c.o_mask = L::mask; c.o_cf = L::cf; c.o_inv = L::inv;
        return 0;
    });
    int o = c.o_inv;  // blob-relative
    auto take = [&](int bytes) { const int at = o; o = align16(o + bytes); return at; };
    take(R * NP * 4);
    c.o_esc_res = take(R * NP * 4);
    c.o_SG = take(R * NP * 4);
    c.o_head = take(nl * 2);
    c.o_tail = take(nl * 2);
    c.o_cnt = take(2 * nl * 4);
    c.pool16 = (allow_pool16 && is_paper_shape(c)) ? 1 : 0;
    c.o_pool = take((c.N << c.Mp_log2) * (c.pool16 ? 2 : 4));
    c.o_spl = o;  // bucket bounds of the block-wide sort (hints), sized by the kernel variant
    o += for_variant(c.Npad, NP, [&](auto, auto ns) { return Lay<decltype(ns)::value>::spl_bytes; });
    c.blob_bytes = o;
    // runtime scratch (absolute offsets; zeroed at kernel start up to the staging tile)
    o = c.o_blob + c.blob_bytes;
    c.o_scratch1 = o;
    c.o_ahead = take(nl * 4);
    c.o_cdf = take(c.A * 4);
    if (c.K) {  // book-cap path: key bins of this step's candidates, per book and per level
        c.o_bbh = take(2 * R * BOOK_BINS * 4);
        c.o_bbc = take(2 * R * BOOK_BINS * 4);
        c.o_lbh = take(nl * LEVEL_BINS * 4);
        c.o_lmask = take(nl * 4);
    } else {
        c.o_bbh = c.o_bbc = c.o_lbh = c.o_lmask = c.o_ahead;  // unused
    }
    // staging tile of the population observation rows (not zeroed); the matched-order lists
    // mb | ma alias its head (written after the previous step's bulk store has been read,
    // consumed before the rows are staged)
    // bucket keys of labor and income (block-wide sort of CTAs of 512 / 1024 threads): live between the end of the
    // state update and the statistics of the same step
    const int bk2 = for_variant(c.Npad, NP, [&](auto, auto ns) {
        using L = Lay<decltype(ns)::value>;
        return L::bk_metrics > 1 ? (L::bk_metrics - 1) * L::bk_warps * L::bk_cap * 4 : 0;
    });
    c.o_stage = o;
    c.stage_obs = 0;
    const int lists = 2 * R * NP * 4;
    if ((c.N * c.D_pop) % 4 == 0 && c.N * c.D_pop * 4 >= lists && o + c.N * c.D_pop * 4 <= 100 * 1024) {
        c.o_bk2 = bk2 ? take(bk2) : c.o_ahead;  // the staging tile is being written while these keys are live
        c.o_stage = o;
        c.stage_obs = 1;
        c.stage_alias_bytes = lists;
        c.o_mb = o;
        c.o_ma = o + R * NP * 4;
        take(c.N * c.D_pop * 4);
    } else {
        // matched-order lists, and over the same bytes the per-warp row buffers of the unstaged observation path (the
        // lists are consumed when the trades settle, the rows are written after the state is final)
        const int rowbuf = c.n_warps * 8 * c.D_pop * 4;
        int region = lists > rowbuf ? lists : rowbuf;
        if (bk2 > region) region = bk2;  // the same bytes hold the bucket keys of labor and income in between
        c.o_mb = take(region);
        c.o_bk2 = c.o_mb;
        c.o_ma = c.o_mb + R * NP * 4;
        c.o_rowbuf = c.o_mb;
        c.o_stage = o;
    }
    c.smem_bytes = o;
}

// Shape-specialised step kernels: resource and price counts as compile-time constants remove
// the loop and index overhead of the R- and P-loops (-12 % at the headline shape).  Instantiated
// for the CTA sizes and shapes of BASELINE.json's configs; every other shape runs the generic one.
template <int MT, int NS>
void select_step_kernel(ej_env* h) {
    const DevCfg& c = h->c;
    h->step_fn = ej_step_kernel<MT, NS, 0, 0, 0, 0, 0>;
    h->step_fn_ar = ej_step_kernel<MT, NS, 0, 0, 0, 0, 0, 0, 1>;
    h->step_fn_fx = nullptr;  // f2 variants exist for CTAs of up to 256 threads (build time)
    if constexpr (MT <= 256) h->step_fn_fx = ej_step_kernel<MT, NS, 0, 0, 0, 0, 0, 1>;
    h->step_RT = h->step_PT = 0;
    h->step_pf = 0;
    // pf = 1 also fixes the paper's mechanics (Table 2; PF in ej_device.cuh)
    auto pick = [&](auto rt, auto pt, auto nt, auto bt, auto pf) {
        constexpr int RT = decltype(rt)::value, PT = decltype(pt)::value, NT = decltype(nt)::value, BT = decltype(bt)::value;
        constexpr int PF = decltype(pf)::value;
        const bool paper = c.pool16 == 1 && c.stage_obs == 1;
        bool lay_ok = true;
        if constexpr (PF == 1) {  // the kernel's compile-time layout must be the one build_layout() made
            using S = StaticLay<NS, RT, PT, NT>;
            lay_ok = c.o_esc_res == S::esc_res && c.o_SG == S::SG && c.o_head == S::head && c.o_tail == S::tail && c.o_cnt == S::cnt &&
                     c.o_pool == S::pool && c.o_spl == S::spl && c.blob_bytes == S::blob_bytes && c.o_ahead == S::ahead && c.o_cdf == S::cdf &&
                     c.o_stage == S::stage && c.o_mb == S::mb && c.o_ma == S::ma;
        }
        if (c.R == RT && c.P == PT && (NT == 0 || (c.N == NT && c.B == BT)) && (PF == 0 || (paper && lay_ok))) {
            h->step_fn = ej_step_kernel<MT, NS, RT, PT, NT, BT, PF>;
            h->step_fn_ar = ej_step_kernel<MT, NS, RT, PT, NT, BT, PF, 0, 1>;
            h->step_pf = PF;
            // f2: the factored variant must read the same (16-bit) order pool as the dense one
            if constexpr (PF == 1) h->step_fn_fx = ej_step_kernel<MT, NS, RT, PT, NT, BT, PF, 1>;
            h->step_RT = RT; h->step_PT = PT;
        }
    };
    using I0 = std::integral_constant<int, 0>;
    using I1 = std::integral_constant<int, 1>;
    using I2 = std::integral_constant<int, 2>;
    using I7 = std::integral_constant<int, 7>;
    using I10 = std::integral_constant<int, 10>;
    if constexpr (MT == 128) {
        // BASELINE.json's N = 100 shapes: R, P, N, B and the mechanics are compile-time constants
        if constexpr (NS == tight_stride(128)) {
            using I100 = std::integral_constant<int, 100>;
            pick(I2(), I10(), I100(), I7(), I1());
#ifndef EJ_DEV_ONLY_128
            pick(std::integral_constant<int, 3>(), I10(), I100(), I7(), I1());
            pick(std::integral_constant<int, 6>(), I10(), I100(), I7(), I1());
            // f3, the paper's section-5 shapes: prices {3,6,9}, 3 brackets; r = 4 keeps Table 2's mechanics
            // (R_d = floor(log2 4) = 2), r = 12 has R_d = 3 and gets R and P only
            pick(std::integral_constant<int, 4>(), std::integral_constant<int, 3>(), I100(), std::integral_constant<int, 3>(), I1());
#endif
        }
#ifndef EJ_DEV_ONLY_128
        if (h->step_RT == 0) pick(I2(), std::integral_constant<int, 5>(), I0(), I0(), I0());
        if (h->step_RT == 0) pick(std::integral_constant<int, 12>(), std::integral_constant<int, 3>(), I0(), I0(), I0());
#endif
    }
    if constexpr (MT == 1024 && NS == 1024) {
        // configs[3]: N = 1000 with a book cap (mechanics stay runtime)
        pick(I2(), I10(), std::integral_constant<int, 1000>(), I7(), I0());
    }
}

bool misaligned16(const void* p) { return ((uintptr_t)p & 15u) != 0; }
bool misaligned4(const void* p) { return ((uintptr_t)p & 3u) != 0; }

int launch_step(ej_env* h, const StepIO& io) {
    const DevCfg& c = h->c;
    // the kernels move observation tiles with 16-byte bulk copies and everything else with 32-bit accesses
    if (misaligned16(io.obs) || misaligned16(io.obs_priv) || misaligned16(io.obs_shared) || misaligned16(io.obs_gov))
        return fail(h, EJ_ERR_PARAM, "bad field: %s", "observation pointer (must be 16-byte aligned)");
    if (misaligned4(io.actions) || misaligned4(io.gov_actions) || misaligned4(io.rew) || misaligned4(io.actions_out) || misaligned4(io.gov_out))
        return fail(h, EJ_ERR_PARAM, "bad field: %s", "actions / rewards pointer (must be 4-byte aligned)");
    int smem = c.smem_bytes;
    if (io.obs_priv && h->step_pf) {
        // f2 on the shape-specialised kernels: the staged tile holds the 3R + 4 private columns only, so the launch asks
        // for what that tile (or the matched-order lists under it) needs: 10 instead of 9 CTAs fit an SM at the headline shape
        const int lists = 2 * c.R * c.N4 * 4, tile = align16(c.N * (3 * c.R + 4) * 4);
        smem = c.o_stage + (lists > tile ? lists : tile);
    }
    (io.obs_priv ? h->step_fn_fx : io.auto_reset ? h->step_fn_ar : h->step_fn)<<<c.E, c.Npad, smem, h->stream>>>(c, h->d_state, io);
    h->launches++;
    EJ_CUDA(h, cudaGetLastError(), "ej_step_kernel launch");
    return EJ_OK;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel FUNCTION, and handles of different shapes
// share functions (the generic step kernel, reset, observe, the policy kernel): the attribute is only ever
// raised, to the largest request any live or past handle of this process has made for that function.
std::mutex g_smem_mu;
std::map<std::pair<int, const void*>, int> g_smem_max;  // (device, function) -> bytes
cudaError_t raise_smem_attr(const void* fn, int bytes) {
    std::lock_guard<std::mutex> lock(g_smem_mu);
    int dev = 0;
    cudaGetDevice(&dev);
    int& cur = g_smem_max[std::make_pair(dev, fn)];
    if (bytes <= cur) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) cur = bytes;
    return e;
}

int set_smem_attr(ej_env* h) {
    const DevCfg& c = h->c;
    return for_variant(c.Npad, c.N4, [&](auto mt, auto ns) {
        constexpr int MT = decltype(mt)::value, NS = decltype(ns)::value;
        select_step_kernel<MT, NS>(h);
        EJ_CUDA(h, raise_smem_attr((const void*)h->step_fn, c.smem_bytes), "smem attr (step)");
        EJ_CUDA(h, raise_smem_attr((const void*)h->step_fn_ar, c.smem_bytes), "smem attr (step, auto-reset)");
        if (h->step_fn_fx) EJ_CUDA(h, raise_smem_attr((const void*)h->step_fn_fx, c.smem_bytes), "smem attr (step, factored)");
        EJ_CUDA(h, raise_smem_attr((const void*)ej_observe_kernel<MT, NS>, c.smem_bytes), "smem attr (observe)");
        EJ_CUDA(h, raise_smem_attr((const void*)ej_reset_kernel<MT, NS>, c.smem_bytes), "smem attr (reset)");
        return EJ_OK;
    });
}

size_t state_words(const DevCfg& c) {
    const size_t N = c.N, R = c.R, B = c.B, cap = (size_t)c.N * c.M;
    return 13 + B + R + N * (6 + 3 * R) + 2 * R * (1 + 3 * cap) + 1;  // last word: episode index (f4)
}

int32_t f2w(float f) { int32_t w; memcpy(&w, &f, 4); return w; }
float w2f(int32_t w) { float f; memcpy(&f, &w, 4); return f; }

// ---- a12: policy networks ----
int align128(int x) { return (x + 127) & ~127; }

// Dynamic shared memory of ej_policy_kernel: weights once, then two slots per group.  A slot's buffer holds the
// layer-1 operand (128 x K1p bf16) with the fp32 observation rows beside it, later the hidden activations (128 x 128 bf16).
int policy_stage_off(const PolicyNet& n) { return align128(PTILE * n.K1p * 2); }
int policy_slot_bytes(const PolicyNet& n, int row_stride) {
    const int a_cols = n.K1p > PH ? n.K1p : PH;
    const int hidden = PTILE * a_cols * 2, first = policy_stage_off(n) + align16(PTILE * row_stride * 4);
    return align128(hidden > first ? hidden : first);
}
int policy_tmem_cols(const PolicyNet& n) { return n.Op > 128 ? 256 : 128; }
int policy_groups(const PolicyNet& n, int row_stride) {
    int g = P_TMEM_ALLOC / (2 * policy_tmem_cols(n));
    const int fit = (227 * 1024 - align128(n.blob_bytes)) / (2 * policy_slot_bytes(n, row_stride));
    if (g > fit) g = fit;
    return g > PGROUPS ? PGROUPS : g;
}
int policy_smem_bytes(const PolicyNet& n, int row_stride) {
    return align128(n.blob_bytes) + policy_groups(n, row_stride) * 2 * policy_slot_bytes(n, row_stride);
}

// Repack a row-major [rows][cols] bf16 matrix into the canonical K-major no-swizzle UMMA layout
// with rows_p x cols_p extent (zero padded): element (r, k) at (r%8)*16 + (r/8)*cols_p*16 + (k/8)*128 + (k%8)*2.
void pack_operand(const uint16_t* w, int rows, int cols, int rows_p, int cols_p, uint8_t* dst) {
    memset(dst, 0, (size_t)rows_p * cols_p * 2);
    for (int r = 0; r < rows; ++r)
        for (int k = 0; k < cols; ++k) {
            const size_t off = (size_t)(r & 7) * 16 + (size_t)(r >> 3) * cols_p * 16 + (size_t)(k >> 3) * 128 + (size_t)(k & 7) * 2;
            memcpy(dst + off, &w[(size_t)r * cols + k], 2);
        }
}

int build_net(ej_env* h, const ej_mlp* m, const char* which, int in_dim, int n_heads, int head, PolicyNet& net, uint8_t** d_blob) {
    if (m->struct_size != sizeof(ej_mlp)) return fail(h, EJ_ERR_PARAM, "bad field: %s.struct_size", which);
    if (m->hidden != PH) return fail(h, EJ_ERR_PARAM, "bad field: %s.hidden (must be 128)", which);
    if (m->in_dim != in_dim) return fail(h, EJ_ERR_PARAM, "bad field: %s.in_dim", which);
    if (m->out_dim != n_heads * head || m->out_dim > 256) return fail(h, EJ_ERR_PARAM, "bad field: %s.out_dim", which);
    if (!m->w1 || !m->w2 || !m->w3 || !m->b1 || !m->b2 || !m->b3) return fail(h, EJ_ERR_PARAM, "bad field: %s weights", which);
    net.D_in = in_dim;
    net.K1p = (in_dim + 15) & ~15;
    net.n_out = m->out_dim;
    net.Op = (m->out_dim + 15) & ~15;
    net.n_heads = n_heads;
    net.head = head;
    net.w1_bytes = PH * net.K1p * 2;
    net.w2_bytes = PH * PH * 2;
    net.w3_bytes = net.Op * PH * 2;
    const int bias_bytes = align16((PH + PH + net.Op) * 4);
    net.blob_bytes = net.w1_bytes + net.w2_bytes + net.w3_bytes + bias_bytes;
    net.recipK1p = (uint32_t)((0x100000000ull + net.K1p - 1) / net.K1p);
    net.nch = 0;
    for (int hh = 0; hh < n_heads; ++hh) {
        const int span = ((hh * head + head - 1) >> 4) - ((hh * head) >> 4) + 1;
        if (span > net.nch) net.nch = span;
    }
    if (policy_groups(net, in_dim + 3) < 1) return fail(h, EJ_ERR_PARAM, "bad field: %s (network does not fit in shared memory)", which);
    std::vector<uint8_t> blob(net.blob_bytes, 0);
    pack_operand(m->w1, PH, in_dim, PH, net.K1p, blob.data());
    pack_operand(m->w2, PH, PH, PH, PH, blob.data() + net.w1_bytes);
    pack_operand(m->w3, m->out_dim, PH, net.Op, PH, blob.data() + net.w1_bytes + net.w2_bytes);
    float* b = (float*)(blob.data() + net.w1_bytes + net.w2_bytes + net.w3_bytes);
    memcpy(b, m->b1, PH * 4);
    memcpy(b + PH, m->b2, PH * 4);
    memcpy(b + 2 * PH, m->b3, (size_t)m->out_dim * 4);
    if (*d_blob) { cudaFree(*d_blob); *d_blob = nullptr; }
    if (cudaMalloc(d_blob, blob.size()) != cudaSuccess) { cudaGetLastError(); return fail(h, EJ_ERR_NOMEM, "%s", "policy allocation failed"); }
    EJ_CUDA(h, cudaMemcpy(*d_blob, blob.data(), blob.size(), cudaMemcpyHostToDevice), "policy upload");
    net.blob = *d_blob;
    return EJ_OK;
}

void fill_job(ej_env* h, PolicyArgs& a, const PolicyNet& net, const float* obs, int row_stride, int rows, int rows_per_env,
              int fixed_agent, uint32_t stream_base, int32_t* actions, float* logits) {
    const DevCfg& c = h->c;
    memset(&a, 0, sizeof(a));
    a.net = net;
    a.obs = obs; a.row_stride = row_stride; a.rows = rows; a.rows_per_env = rows_per_env; a.fixed_agent = fixed_agent;
    a.state = h->d_state; a.blob_stride = c.blob_bytes; a.o_episode = (int)offsetof(EnvHdr, episode);
    a.env_id_base = c.env_id_base; a.seed_lo = c.seed_lo; a.seed_hi = c.seed_hi; a.stream_base = stream_base;
    a.actions = actions; a.logits = logits;
    a.smem_W1 = 0;
    a.smem_W2 = a.smem_W1 + net.w1_bytes;
    a.smem_W3 = a.smem_W2 + net.w2_bytes;
    a.smem_bias = a.smem_W3 + net.w3_bytes;
    a.smem_group = align128(net.blob_bytes);
    a.slot_bytes = policy_slot_bytes(net, row_stride);
    a.stage_off = policy_stage_off(net);
    a.groups = policy_groups(net, row_stride);
    a.tmem_cols = policy_tmem_cols(net);
}

int ctas_for(const PolicyArgs& a, int cap) {
    const int tiles = (a.rows + PTILE - 1) / PTILE;
    const int want = (tiles + a.groups - 1) / a.groups;
    return want < cap ? want : cap;
}

// Population and (optionally) government policy in ONE launch: the government's few tiles get
// their own CTAs next to the population's, so they cost no extra launch and no extra latency.
int launch_policy(ej_env* h, const float* obs, int32_t* actions, int32_t* gov_actions, float* pop_logits, float* gov_logits) {
    const DevCfg& c = h->c;
    PolicyLaunch pl;
    memset(&pl, 0, sizeof(pl));
    fill_job(h, pl.job[0], h->pop_net, obs, c.D_pop, c.E * c.N, c.N, -1, 0u, actions, pop_logits);
    if (h->masking) {  // f1: the population head samples among the available actions
        PolicyMask& k = pl.job[0].mask;
        k.on = 1;
        k.o_coin = c.o_coin; k.o_mask = c.o_mask; k.o_inv = c.o_inv; k.NS = c.N4;
        k.R = c.R; k.P = c.P; k.M = c.M; k.craft_mode = c.craft_mode; k.craft_units = c.craft_units;
        k.craft_distinct = c.craft_distinct; k.base_buy = c.base_buy; k.base_sell = c.base_sell; k.A = c.A;
        k.allow_noop = c.allow_noop;
        for (int i = 0; i < EJ_MAX_PRICES; ++i) k.prices[i] = c.prices[i];
    }
    int smem = policy_smem_bytes(h->pop_net, c.D_pop), gov_ctas = 0;
    if (gov_actions) {
        fill_job(h, pl.job[1], h->gov_net, obs + c.gov_obs_offset, c.D_gov_pad, c.E, 1, c.N, 1u, gov_actions, gov_logits);
        // a government tile costs several population tiles (one categorical per bracket): two tiles per CTA, both in
        // flight at once, end well before the population CTAs do and take fewer SMs away from them than one tile each
        const int gov_tiles = (c.E + PTILE - 1) / PTILE;
        gov_ctas = ctas_for(pl.job[1], (gov_tiles + 1) / 2);
        const int sg = policy_smem_bytes(h->gov_net, c.D_gov_pad);
        if (sg > smem) smem = sg;
    }
    pl.split = ctas_for(pl.job[0], h->n_sms - gov_ctas);
    ej_policy_kernel<<<pl.split + gov_ctas, P_THREADS, smem, h->stream>>>(pl);
    h->launches++;
    EJ_CUDA(h, cudaGetLastError(), "ej_policy_kernel launch");
    return EJ_OK;
}

int launch_step(ej_env* h, const StepIO& io);

// ej_rollout in policy mode: per step, policy kernels (population, government) on the current
// observation, then one step of the env kernel.  Observations and actions chain through the
// caller's rings when given, else through library-owned buffers.
int rollout_with_policy(ej_env* h, int T, const ej_rollout_io* rio, const StepIO& base) {
    const DevCfg& c = h->c;
    const size_t EN = (size_t)c.E * c.N, EB = (size_t)c.E * c.B;
    const int depth = base.ring_depth;
    float* pl_ring = rio ? rio->pop_logits_ring : nullptr;
    float* gl_ring = rio ? rio->gov_logits_ring : nullptr;
    // observation of the current state
    int rc = for_variant(c.Npad, c.N4, [&](auto mt, auto ns) {
        constexpr int MT = decltype(mt)::value, NS = decltype(ns)::value;
        ej_observe_kernel<MT, NS><<<c.E, c.Npad, c.smem_bytes, h->stream>>>(c, h->d_state, h->d_pobs);
        h->launches++;
        EJ_CUDA(h, cudaGetLastError(), "ej_observe_kernel launch");
        return EJ_OK;
    });
    if (rc != EJ_OK) return rc;
    const float* cur_obs = h->d_pobs;
    for (int s = 0; s < T; ++s) {
        const int slot = s % depth;
        int32_t* act = base.actions_out ? base.actions_out + slot * EN : h->d_pact;
        int32_t* gov = base.gov_out ? base.gov_out + slot * EB : h->d_pgov;
        const bool gov_supplied = base.gov_actions != nullptr;
        rc = launch_policy(h, cur_obs, act, gov_supplied ? nullptr : gov, pl_ring ? pl_ring + (size_t)slot * EN * c.A : nullptr,
                           gl_ring ? gl_ring + (size_t)slot * c.E * c.B * c.L : nullptr);
        if (rc != EJ_OK) return rc;
        if (gov_supplied) gov = const_cast<int32_t*>(base.gov_actions + (size_t)s * EB);
        StepIO io;
        memset(&io, 0, sizeof(io));
        io.cdf = base.cdf; io.n_steps = 1; io.ring_depth = 1; io.auto_reset = base.auto_reset;
        io.actions = act; io.gov_actions = gov;
        io.obs = base.obs ? base.obs + (size_t)slot * c.obs_floats : h->d_pobs;
        io.rew = base.rew ? base.rew + (size_t)slot * (EN + c.E) : nullptr;
        io.done = base.done ? base.done + (size_t)slot * c.E : nullptr;
        rc = launch_step(h, io);
        if (rc != EJ_OK) return rc;
        cur_obs = io.obs;
    }
    return EJ_OK;
}

// The two halves of ej_create that need no allocation (shared with ej_rollout_noalloc): validation of the shape and
// the parameters, and the device configuration of a handle (constants, shared-memory layout, kernel variant).  Errors
// go to the create-error string (ej_last_error(NULL)).
int check_shape_and_params(int32_t E, int32_t N, int32_t R, const ej_params* p, int* mp_log2_out) {
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
    if (p->skill_init != EJ_SKILL_UNIFORM01 && p->skill_init != EJ_SKILL_PARETO_CLIP && p->skill_init != EJ_SKILL_NORMAL_CLIP)
        return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "skill_init");
    if (p->skill_init == EJ_SKILL_NORMAL_CLIP && !(p->skill_std >= 0.0f && p->skill_clip_lo <= p->skill_clip_hi))
        return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "skill_std / skill_clip_lo / skill_clip_hi");
    if (!(p->skill_growth_rate >= 0.0f)) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "skill_growth_rate");
    if (p->skill_growth_rate > 0.0f && !(p->skill_max > 0.0f)) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "skill_max");
    int mp_log2 = 0;
    while ((1 << mp_log2) < p->max_active_orders) ++mp_log2;
    *mp_log2_out = mp_log2;
    if (((int64_t)N << mp_log2) >= 65535) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "max_active_orders (N * M too large)");
    return EJ_OK;
}

int configure_handle(ej_env* h, int32_t E, int32_t N, int32_t R, const ej_params* p, int mp_log2) {
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
    c.recipP = (65536 + c.P - 1) / c.P;
    c.n_groups = c.K ? 2 * R : c.n_levels;
    c.D_pop = 6 + 8 * R + c.B;
    c.D_gov = 3 * (3 + R) + c.B + 2;
    c.D_gov_pad = (c.D_gov + 3) & ~3;
    c.Npad = 32;
    while (c.Npad < N) c.Npad <<= 1;
    c.N4 = (N <= tight_stride(c.Npad)) ? tight_stride(c.Npad) : c.Npad;  // stride of the per-agent arrays
    c.n_metrics = 3 + R;
    c.n_warps = c.Npad / 32;
    c.shrow_len = 5 * R + c.B + 2;
    c.inv_n = 1.0 / (double)N;
    c.ua = 1.0 - (double)p->eta;
    c.inv_ua = 1.0 / c.ua;
    for (int i = 0; i < c.P; ++i) c.prices[i] = p->prices[i];
    for (int i = 0; i + 1 < c.B; ++i) c.thresholds[i] = p->thresholds[i];
    for (int i = 0; i < c.L; ++i) c.rate_table[i] = p->rate_table[i];
    c.starting_coin = p->starting_coin; c.labor_craft = p->labor_craft; c.labor_gather = p->labor_gather;
    c.labor_trade = p->labor_trade; c.eta = p->eta; c.omega = p->omega; c.craft_scale = p->craft_scale;
    c.clip_lo = p->skill_clip_lo; c.clip_hi = p->skill_clip_hi;
    c.skill_rate = p->skill_growth_rate; c.skill_max = p->skill_max;
    c.skill_mean = p->skill_mean; c.skill_std = p->skill_std;
    c.s_coin = p->obs_scale_coin; c.s_count = p->obs_scale_count; c.s_price = p->obs_scale_price; c.s_labor = p->obs_scale_labor;
    c.env_id_base = p->env_id_base;
    c.gov_obs_offset = ((unsigned long long)E * N * c.D_pop + 3ull) & ~3ull;
    c.obs_floats = c.gov_obs_offset + (unsigned long long)E * c.D_gov_pad;
    build_layout(c);
    if (c.smem_bytes > 227 * 1024) {
        return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "N/R/max_active_orders (state exceeds 227 KB of shared memory)");
    }
    int rc = set_smem_attr(h);
    if (rc == EJ_OK && c.pool16 && !h->step_pf) {  // no kernel for the 16-bit pool words of this layout: plain layout, generic kernel
        build_layout(c, false);
        rc = set_smem_attr(h);
    }
    if (rc != EJ_OK) { memcpy(g_create_err, h->err, 256); return rc; }
    return EJ_OK;
}

}  // namespace

extern "C" {

const char* ej_last_error(const ej_env* h) { return h ? h->err : g_create_err; }

int ej_create(int32_t E, int32_t N, int32_t R, const ej_params* p, ej_env** out) {
    g_create_err[0] = 0;
    if (!out) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "out");
    *out = nullptr;
    int mp_log2 = 0;
    {
        const int vrc = check_shape_and_params(E, N, R, p, &mp_log2);
        if (vrc != EJ_OK) return vrc;
    }

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, EJ_ERR_CUDA, "%s", "no CUDA device: this library has no CPU fallback");
    }
    ej_env* h = new (std::nothrow) ej_env();
    if (!h) return fail(nullptr, EJ_ERR_NOMEM, "%s", "host allocation failed");
    {
        const int crc = configure_handle(h, E, N, R, p, mp_log2);
        if (crc != EJ_OK) { delete h; return crc; }
    }
    DevCfg& c = h->c;
    cudaError_t ce = cudaMalloc(&h->d_state, (size_t)E * c.blob_bytes);
    if (ce == cudaSuccess) ce = cudaMemset(h->d_state, 0, (size_t)E * c.blob_bytes);
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
    cudaFree(h->d_act); cudaFree(h->d_gov); cudaFree(h->d_obs); cudaFree(h->d_rew); cudaFree(h->d_done); cudaFree(h->d_fx);
    cudaFree(h->d_pop_blob); cudaFree(h->d_gov_blob); cudaFree(h->d_pobs); cudaFree(h->d_pact); cudaFree(h->d_pgov);
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
    o->D_priv = 3 * c.R + 4; o->D_shared = 5 * c.R + c.B + 2; o->D_shared_pad = (o->D_shared + 3) & ~3;
    return EJ_OK;
}

int ej_reset(ej_env* h, uint64_t seed) {
    if (!h) return EJ_ERR_PARAM;
    DevCfg& c = h->c;
    c.seed_lo = (uint32_t)(seed & 0xFFFFFFFFull);
    c.seed_hi = (uint32_t)(seed >> 32);
    int rc = for_variant(c.Npad, c.N4, [&](auto mt, auto ns) {
        constexpr int MT = decltype(mt)::value, NS = decltype(ns)::value;
        ej_reset_kernel<MT, NS><<<c.E, c.Npad, c.smem_bytes, h->stream>>>(c, h->d_state);
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
    if (misaligned16(obs_out)) return fail(h, EJ_ERR_PARAM, "bad field: %s", "obs_out (must be 16-byte aligned)");
    const DevCfg& c = h->c;
    return for_variant(c.Npad, c.N4, [&](auto mt, auto ns) {
        constexpr int MT = decltype(mt)::value, NS = decltype(ns)::value;
        ej_observe_kernel<MT, NS><<<c.E, c.Npad, c.smem_bytes, h->stream>>>(c, h->d_state, obs_out);
        h->launches++;
        EJ_CUDA(h, cudaGetLastError(), "ej_observe_kernel launch");
        return EJ_OK;
    });
}

int ej_action_mask(ej_env* h, uint8_t* mask_out) {
    if (!h) return EJ_ERR_PARAM;
    if (!mask_out || ((uintptr_t)mask_out & 3)) return fail(h, EJ_ERR_PARAM, "bad field: %s", "mask_out");
    if (!h->was_reset) return fail(h, EJ_ERR_STATE, "%s", "ej_action_mask before ej_reset / ej_set_state");
    const DevCfg& c = h->c;
    const unsigned long long total = (unsigned long long)c.E * c.N * c.A;
    const unsigned long long words = (total + 3) / 4;
    ej_mask_kernel<<<(unsigned)((words + 255) / 256), 256, 0, h->stream>>>(c, h->d_state, mask_out, total);
    h->launches++;
    EJ_CUDA(h, cudaGetLastError(), "ej_mask_kernel launch");
    return EJ_OK;
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

int ej_step_host_factored(ej_env* h, const int32_t* actions, const int32_t* gov_actions, float* priv_out, float* shared_out,
                          float* gov_obs_out, float* rew_out, uint8_t* done_out) {
    if (!h) return EJ_ERR_PARAM;
    if (!actions) return fail(h, EJ_ERR_PARAM, "bad field: %s", "actions");
    if (!gov_actions) return fail(h, EJ_ERR_PARAM, "bad field: %s", "gov_actions");
    if (!priv_out || !shared_out) return fail(h, EJ_ERR_PARAM, "bad field: %s", "priv_out / shared_out (set both)");
    const DevCfg& c = h->c;
    const size_t EN = (size_t)c.E * c.N, EB = (size_t)c.E * c.B;
    const size_t n_priv = EN * (size_t)(3 * c.R + 4), n_shared = (size_t)c.E * (size_t)((5 * c.R + c.B + 2 + 3) & ~3);
    const size_t n_gov = (size_t)c.E * c.D_gov_pad;
    if (!h->d_fx) {  // one allocation: actions | gov actions | priv | shared | gov rows | rewards | done
        size_t off = 0;
        auto take = [&off](size_t bytes) { const size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
        h->fx_act = take(EN * 4); h->fx_gov = take(EB * 4); h->fx_priv = take(n_priv * 4); h->fx_shared = take(n_shared * 4);
        h->fx_govrow = take(n_gov * 4); h->fx_rew = take((EN + c.E) * 4); h->fx_done = take((size_t)c.E);
        if (cudaMalloc(&h->d_fx, off) != cudaSuccess) { cudaGetLastError(); h->d_fx = nullptr; return fail(h, EJ_ERR_NOMEM, "%s", "staging allocation failed"); }
    }
    uint8_t* const d = h->d_fx;
    EJ_CUDA(h, cudaMemcpyAsync(d + h->fx_act, actions, EN * 4, cudaMemcpyHostToDevice, h->stream), "H2D actions");
    EJ_CUDA(h, cudaMemcpyAsync(d + h->fx_gov, gov_actions, EB * 4, cudaMemcpyHostToDevice, h->stream), "H2D gov_actions");
    ej_rollout_io rio;
    memset(&rio, 0, sizeof(rio));
    rio.struct_size = sizeof(rio); rio.ring_depth = 1;
    rio.actions_in = (const int32_t*)(d + h->fx_act); rio.gov_actions_in = (const int32_t*)(d + h->fx_gov);
    rio.obs_priv_ring = (float*)(d + h->fx_priv); rio.obs_shared_ring = (float*)(d + h->fx_shared);
    rio.obs_gov_ring = gov_obs_out ? (float*)(d + h->fx_govrow) : nullptr;
    rio.rew_ring = rew_out ? (float*)(d + h->fx_rew) : nullptr; rio.done_ring = done_out ? d + h->fx_done : nullptr;
    const int rc = ej_rollout(h, 1, &rio);
    if (rc != EJ_OK) return rc;
    EJ_CUDA(h, cudaMemcpyAsync(priv_out, d + h->fx_priv, n_priv * 4, cudaMemcpyDeviceToHost, h->stream), "D2H private block");
    EJ_CUDA(h, cudaMemcpyAsync(shared_out, d + h->fx_shared, n_shared * 4, cudaMemcpyDeviceToHost, h->stream), "D2H env-wide block");
    if (gov_obs_out) EJ_CUDA(h, cudaMemcpyAsync(gov_obs_out, d + h->fx_govrow, n_gov * 4, cudaMemcpyDeviceToHost, h->stream), "D2H government rows");
    if (rew_out) EJ_CUDA(h, cudaMemcpyAsync(rew_out, d + h->fx_rew, (EN + c.E) * 4, cudaMemcpyDeviceToHost, h->stream), "D2H rewards");
    if (done_out) EJ_CUDA(h, cudaMemcpyAsync(done_out, d + h->fx_done, (size_t)c.E, cudaMemcpyDeviceToHost, h->stream), "D2H done");
    EJ_CUDA(h, cudaStreamSynchronize(h->stream), "ej_step_host_factored sync");
    return EJ_OK;
}

int ej_rollout(ej_env* h, int32_t T, const ej_rollout_io* rio) {
    if (!h) return EJ_ERR_PARAM;
    if (T < 0) return fail(h, EJ_ERR_PARAM, "bad field: %s", "T");
    if (!h->was_reset) return fail(h, EJ_ERR_STATE, "%s", "ej_rollout before ej_reset / ej_set_state");
    if (T == 0) return EJ_OK;
    StepIO io;
    memset(&io, 0, sizeof(io));
    io.cdf = h->d_cdf; io.n_steps = T; io.ring_depth = 1; io.masked = h->masking ? 1 : 0;
    if (rio) {
        if (rio->struct_size != sizeof(ej_rollout_io)) return fail(h, EJ_ERR_PARAM, "bad field: %s", "io.struct_size");
        if (rio->ring_depth < 1) return fail(h, EJ_ERR_PARAM, "bad field: %s", "io.ring_depth");
        // the kernels index rings and action streams with 32-bit element offsets
        const unsigned long long lim = 1ull << 32;
        if ((unsigned long long)rio->ring_depth * h->c.obs_floats >= lim) return fail(h, EJ_ERR_PARAM, "bad field: %s", "io.ring_depth (ring_depth * obs_floats must stay below 2^32)");
        if (rio->actions_in && (unsigned long long)T * h->c.E * h->c.N >= lim) return fail(h, EJ_ERR_PARAM, "bad field: %s", "T (T * E * N must stay below 2^32 with actions_in)");
        io.ring_depth = rio->ring_depth;
        io.actions = rio->actions_in; io.gov_actions = rio->gov_actions_in;
        io.obs = rio->obs_ring; io.rew = rio->rew_ring; io.done = rio->done_ring;
        io.actions_out = rio->actions_ring; io.gov_out = rio->gov_actions_ring;
        io.auto_reset = rio->auto_reset ? 1 : 0;
        if (rio->obs_priv_ring || rio->obs_shared_ring || rio->obs_gov_ring) {  // f2: factored observations
            const DevCfg& c = h->c;
            if (!rio->obs_priv_ring || !rio->obs_shared_ring) return fail(h, EJ_ERR_PARAM, "bad field: %s", "io.obs_priv_ring / io.obs_shared_ring (set both)");
            if (rio->obs_ring) return fail(h, EJ_ERR_PARAM, "bad field: %s", "io.obs_ring (must be NULL with factored observations)");
            if (!h->step_fn_fx || !c.stage_obs || (c.N * (3 * c.R + 4)) % 4 != 0) return fail(h, EJ_ERR_PARAM, "bad field: %s", "io.obs_priv_ring (shape cannot stage factored observations)");
            if (h->has_policy && !rio->actions_in) return fail(h, EJ_ERR_PARAM, "bad field: %s", "io.obs_priv_ring (not available in policy mode)");
            if (rio->auto_reset) return fail(h, EJ_ERR_PARAM, "bad field: %s", "io.auto_reset (not available with factored observations)");
            io.obs_priv = rio->obs_priv_ring; io.obs_shared = rio->obs_shared_ring; io.obs_gov = rio->obs_gov_ring;
        }
    }
    if (h->has_policy && !io.actions) return rollout_with_policy(h, T, rio, io);
    return launch_step(h, io);
}

int ej_set_policy(ej_env* h, const ej_mlp* pop, const ej_mlp* gov) {
    if (!h) return EJ_ERR_PARAM;
    const DevCfg& c = h->c;
    if (!pop && !gov) { h->has_policy = false; return EJ_OK; }
    if (!pop || !gov) return fail(h, EJ_ERR_PARAM, "bad field: %s", "pop / gov (both or neither)");
    EJ_CUDA(h, cudaStreamSynchronize(h->stream), "set_policy sync");
    h->has_policy = false;
    int rc = build_net(h, pop, "pop", c.D_pop, 1, c.A, h->pop_net, &h->d_pop_blob);
    if (rc != EJ_OK) return rc;
    rc = build_net(h, gov, "gov", c.D_gov, c.B, c.L, h->gov_net, &h->d_gov_blob);
    if (rc != EJ_OK) return rc;
    const int sp = policy_smem_bytes(h->pop_net, c.D_pop), sg = policy_smem_bytes(h->gov_net, c.D_gov_pad);
    const int smem = sp > sg ? sp : sg;
    EJ_CUDA(h, raise_smem_attr((const void*)ej_policy_kernel, smem), "smem attr (policy)");
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&h->n_sms, cudaDevAttrMultiProcessorCount, dev);
    if (!h->d_pobs) {
        cudaError_t ce = cudaMalloc(&h->d_pobs, (size_t)c.obs_floats * 4);
        if (ce == cudaSuccess) ce = cudaMalloc(&h->d_pact, (size_t)c.E * c.N * 4);
        if (ce == cudaSuccess) ce = cudaMalloc(&h->d_pgov, (size_t)c.E * c.B * 4);
        if (ce != cudaSuccess) { cudaGetLastError(); return fail(h, EJ_ERR_NOMEM, "%s", "policy buffers allocation failed"); }
    }
    h->has_policy = true;
    return EJ_OK;
}

int ej_policy_act(ej_env* h, const float* obs, int32_t* actions_out, int32_t* gov_actions_out, float* pop_logits_out,
                  float* gov_logits_out) {
    if (!h) return EJ_ERR_PARAM;
    if (!h->has_policy) return fail(h, EJ_ERR_STATE, "%s", "ej_policy_act before ej_set_policy");
    if (!h->was_reset) return fail(h, EJ_ERR_STATE, "%s", "ej_policy_act before ej_reset / ej_set_state");
    if (!obs || !actions_out || !gov_actions_out) return fail(h, EJ_ERR_PARAM, "bad field: %s", "obs / actions_out / gov_actions_out");
    const DevCfg& c = h->c;
    (void)c;
    return launch_policy(h, obs, actions_out, gov_actions_out, pop_logits_out, gov_logits_out);
}

int ej_set_action_masking(ej_env* h, int32_t on) {
    if (!h) return EJ_ERR_PARAM;
    h->masking = on != 0;
    return EJ_OK;
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
        const uint16_t* head = (const uint16_t*)(s + c.o_head); const int* cnt = (const int*)(s + c.o_cnt) + (((const EnvHdr*)s)->t & 1) * c.n_levels;
        const uint32_t* pool32 = (const uint32_t*)(s + c.o_pool);
        const uint16_t* pool16 = (const uint16_t*)(s + c.o_pool);
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
                    int age;
                    uint32_t nxt;
                    if (c.pool16) {  // next (11 bits, 0x7FF = none) | placed_at mod 32
                        const uint32_t pe = pool16[hh];
                        age = (int)(((uint32_t)hd->t - (pe >> 11)) & 31u);
                        nxt = (pe & 0x7FFu) == 0x7FFu ? NIL : (pe & 0x7FFu);
                    } else {         // next (16 bits) | placed_at (16 bits)
                        const uint32_t pe = pool32[hh];
                        age = (int)(((uint32_t)hd->t - (pe >> 16)) & 0xFFFFu);
                        nxt = pe & 0xFFFFu;
                    }
                    if (out < cap) {
                        w[q0 + 3 * out] = c.prices[p];
                        w[q0 + 3 * out + 1] = (int32_t)(hh >> c.Mp_log2);
                        w[q0 + 3 * out + 2] = hd->t - age;
                    }
                    ++out;
                    hh = nxt;
                }
            }
            q = q0 + 3 * (size_t)cap;
        }
        w[q++] = hd->episode;
    }
    return EJ_OK;
}

int ej_set_state(ej_env* h, int32_t env_begin, int32_t env_count, const int32_t* words, size_t n_words) {
    if (!h) return EJ_ERR_PARAM;
    const DevCfg& c = h->c;
    if (env_begin < 0 || env_count < 0 || env_begin + env_count > c.E) return fail(h, EJ_ERR_PARAM, "bad field: %s", "env range");
    const size_t W = state_words(c);
    if (!words || n_words < W * (size_t)env_count) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words / n_words");
    // the dump holds no Philox key and may cover only some envs: the handle must have been reset (with the seed
    // of the run the dump comes from, if that run is to continue draw for draw)
    if (!h->was_reset) return fail(h, EJ_ERR_STATE, "%s", "ej_set_state before ej_reset (reset with the original seed first)");
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
        int* cnt = (int*)(s + c.o_cnt); uint32_t* pool32 = (uint32_t*)(s + c.o_pool); uint16_t* pool16 = (uint16_t*)(s + c.o_pool);
        const int32_t* w = words + (size_t)k * W;
        size_t q = 0;
        hd->t = w[q++];
        hd->t_in_period = hd->t % c.period;
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
        cnt += (hd->t & 1) * c.n_levels;  // the buffer current at clock t
        int best_bid = 0;  // of the resource whose bids were just read
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
                const int l = b * P + p;
                if (c.pool16) {
                    if (hd->t - placed > 31) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words (order older than the expiry)");
                    pool16[slot] = (uint16_t)(0x7FFu | (((uint32_t)placed & 31u) << 11));
                    if (tail[l] != NIL) pool16[tail[l]] = (uint16_t)((pool16[tail[l]] & 0xF800u) | slot);
                } else {
                    pool32[slot] = NIL | (((uint32_t)placed & 0xFFFFu) << 16);
                    if (tail[l] != NIL) pool32[tail[l]] = (pool32[tail[l]] & 0xFFFF0000u) | slot;
                }
                if (tail[l] == NIL) head[l] = (uint16_t)slot;
                tail[l] = (uint16_t)slot;
                cnt[l]++;
                // a resting book is uncrossed (G13): the kernels size their matched-order lists by that
                if ((b & 1) == 0) { if (o == 0 || price > best_bid) best_bid = price; }
                else if (price <= best_bid) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words (crossed book: best bid >= best ask)");
            }
            if ((b & 1) == 0 && n == 0) best_bid = 0;
            q += 3 * (size_t)cap;
        }
        hd->episode = w[q++];
        if (hd->episode < 0 || hd->episode >= (1 << 24)) return fail(h, EJ_ERR_PARAM, "bad field: %s", "words (episode)");
    }
    EJ_CUDA(h, cudaStreamSynchronize(h->stream), "set_state sync");
    EJ_CUDA(h, cudaMemcpy(h->d_state + (size_t)env_begin * c.blob_bytes, blobs.data(), blobs.size(), cudaMemcpyHostToDevice), "set_state copy");
    return EJ_OK;
}

// Device address of g_noalloc_scratch on the CURRENT device, looked up once per device (fixed table, no allocation).
static int noalloc_scratch_ptr(uint8_t** out) {
    static std::mutex mu;
    static uint8_t* ptr_of_device[64] = {nullptr};
    int dev = -1;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaGetDevice");
    if (dev < 0 || dev >= 64) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "current CUDA device (ordinal must be below 64)");
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr_of_device[dev]) {
        void* ptr = nullptr;
        ce = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);  // with device `dev` current: the address is per device
        if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaGetSymbolAddress(g_noalloc_scratch)");
        if (!ptr) return fail(nullptr, EJ_ERR_CUDA, "%s", "cudaGetSymbolAddress returned a null scratch address");
        ptr_of_device[dev] = (uint8_t*)ptr;
    }
    *out = ptr_of_device[dev];
    return EJ_OK;
}

int ej_rollout_noalloc(int32_t E, int32_t N, int32_t R, const ej_params* p, uint64_t seed, int32_t T, const int32_t* actions,
                       const int32_t* gov_actions, float* obs_ring, float* rew_ring, uint8_t* done_ring, void* cuda_stream) {
    g_create_err[0] = 0;
    int mp_log2 = 0;
    int rc = check_shape_and_params(E, N, R, p, &mp_log2);
    if (rc != EJ_OK) return rc;
    if (T < 0) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "T");
    ej_env h;  // on the stack: no handle, no heap
    rc = configure_handle(&h, E, N, R, p, mp_log2);
    if (rc != EJ_OK) return rc;
    const DevCfg& c = h.c;
    const unsigned long long need = (unsigned long long)E * (unsigned long long)c.blob_bytes;
    if (need > (unsigned long long)EJ_NOALLOC_SCRATCH_BYTES) {
        snprintf(g_create_err, sizeof(g_create_err),
                 "bad field: E (ej_rollout_noalloc: %d envs x %d state bytes = %llu bytes exceed the static scratch of %llu bytes; at most %llu envs of this shape)",
                 (int)E, c.blob_bytes, need, (unsigned long long)EJ_NOALLOC_SCRATCH_BYTES,
                 (unsigned long long)EJ_NOALLOC_SCRATCH_BYTES / (unsigned long long)c.blob_bytes);
        return EJ_ERR_PARAM;
    }
    uint8_t* scratch = nullptr;
    rc = noalloc_scratch_ptr(&scratch);  // first call on a device: set-up (make it outside a graph capture)
    if (rc != EJ_OK) return rc;
    if (T == 0) return EJ_OK;            // set-up only
    if (!actions) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "actions");
    if (!gov_actions) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "gov_actions");
    const unsigned long long lim = 1ull << 32;  // the kernels index rings and action streams with 32-bit element offsets
    if ((unsigned long long)T * c.obs_floats >= lim) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "T (T * obs_floats must stay below 2^32)");
    if ((unsigned long long)T * E * N >= lim) return fail(nullptr, EJ_ERR_PARAM, "bad field: %s", "T (T * E * N must stay below 2^32)");
    h.stream = (cudaStream_t)cuda_stream;
    h.d_state = scratch;
    h.c.seed_lo = (uint32_t)(seed & 0xFFFFFFFFull);
    h.c.seed_hi = (uint32_t)(seed >> 32);
    // reset: every byte of the E blobs is rewritten (the kernel builds a blob from zero and stores all of it), so
    // nothing of an earlier call's contents survives into this one
    rc = for_variant(c.Npad, c.N4, [&](auto mt, auto ns) {
        constexpr int MT = decltype(mt)::value, NS = decltype(ns)::value;
        ej_reset_kernel<MT, NS><<<c.E, c.Npad, c.smem_bytes, h.stream>>>(c, h.d_state);
        EJ_CUDA(&h, cudaGetLastError(), "ej_reset_kernel launch");
        return EJ_OK;
    });
    if (rc == EJ_OK) {
        StepIO io;
        memset(&io, 0, sizeof(io));
        io.n_steps = T; io.ring_depth = T;
        io.actions = actions; io.gov_actions = gov_actions;
        io.obs = obs_ring; io.rew = rew_ring; io.done = done_ring;
        rc = launch_step(&h, io);
    }
    if (rc != EJ_OK) memcpy(g_create_err, h.err, 256);
    h.d_state = nullptr;  // the scratch is not the handle's to free
    return rc;
}

}  // extern "C"
