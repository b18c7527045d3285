// hq_linear.cu — half 1 of the hot path: per weight group (128 rows x one
// RHT tile) fetch the Rice stream (A3), decode unary + remainders (A4, §3.3), un-zig-zag and
// un-strip to INT8 lattice points (A5, §4.6), stage them in shared memory in the UMMA
// K-major SWIZZLE_128B layout and contract with the INT8 activations on the tensor core
// (A6, tcgen05.mma kind::i8 -> INT32 in TMEM, §4.8), then rescale per K-tile and accumulate (A7,
// §4.3).  Decoded weights stay on the SM (tensor memory at batch 1, shared memory up to 63 rows); the large-M path
// (from 64 rows) decodes once per call into an operand-layout scratch copy (hq_linear_large.cuh).
#include <string.h>

#include <mutex>
#include <string>

#include "hq_common.cuh"
#include "hq_internal.h"
#include "hq_linear_e8.cuh"
#include "hq_linear_large.cuh"
#include "hq_e8_ceiling.cuh"
#include "hq_gemv_e8.cuh"
#include "hq_generic_fast.cuh"
#include "hq_tc.cuh"

namespace hq {

constexpr uint32_t GEN_UCAP = 24;  // U words per row gathered through shared memory by the generic decoders

// ---------------------------------------------------------------------------------------------
// hq_decode_int8: block per (rb, kt), warp per sub-group, lane per row, straight from global memory
// (parity tool).
// ---------------------------------------------------------------------------------------------
template <int LAT>
__global__ void __launch_bounds__(128)
k_decode_int8(const uint8_t* blob, const uint32_t* group_off, int64_t m, int64_t n_kt, int n, int k0, int k1,
              int8_t* codes, uint16_t* norms) {
    __shared__ uint32_t urows[128 * (GEN_UCAP + 1)];
    int64_t g = blockIdx.x;
    int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    int64_t rb = g / n_kt, kt = g % n_kt, r = rb * 128 + t;
    int rbits = rbits_of(LAT, n, k0, k1), rw_words = (rbits + 31) / 32;
    SubGroup sg = sub_group(blob + 16 * (size_t)group_off[g * 4 + warp], rw_words);
    uint32_t ul = sg.ulen[lane], nw = (ul + 31) >> 5;
    uint32_t* urow = urows + t * (GEN_UCAP + 1);
    gather_u_words(sg.uarea, nw, lane, urow, GEN_UCAP);
    __syncwarp();
    if (r >= m) return;
    if (norms) norms[r * n_kt + kt] = sg.norm[lane];
    int8_t* out = codes + r * (n_kt * n) + kt * n;
    WordsRowU uw{urow, sg.uarea, sg.ulen, nw, GEN_UCAP, lane};
    WordsRowR rw{sg.rarea, lane, rw_words};
    decode_row_generic<LAT>(rw, 0u, uw, 0u, n, k0, k1, [&](int bk, const int* c) {
#pragma unroll
        for (int e = 0; e < LAT; ++e) out[bk * LAT + e] = (int8_t)c[e];
    });
}

void launch_decode_int8(const hq_weight* w, int8_t* codes, uint16_t* norms, cudaStream_t st) {
#define HQ_D(L) \
    k_decode_int8<L><<<(unsigned)w->G, 128, 0, st>>>(w->blob, w->group_off, w->m, w->n_kt, w->n, w->k0, w->k1, codes, norms)
    switch (w->lattice) {
        case LAT_Z: HQ_D(LAT_Z); break;
        case LAT_A2: HQ_D(LAT_A2); break;
        case LAT_D4: HQ_D(LAT_D4); break;
        default: HQ_D(LAT_E8); break;
    }
#undef HQ_D
}

// ---------------------------------------------------------------------------------------------
// Fused decode + INT8 MMA, generic version (any lattice / tile / k):
// CTA = 128 threads = the 128 rows of a row block (warp = sub-group); loops over a range of K-tiles.
//   per K-tile: each thread decodes its row into the A operand tile -> B operand tile (activations)
//   -> fence -> one thread issues n/32 tcgen05.mma -> commit -> everybody reads its accumulator row
//   from TMEM, rescales and accumulates in fp32 registers.
// NB = columns of the MMA (batch rows handled per pass, multiple of 16).
// ---------------------------------------------------------------------------------------------
struct LinearParams {
    const uint8_t* blob;
    const uint32_t* group_off;
    int64_t m, n_kt;
    int n, k0, k1, rbits;
    float inv_A;
    const int8_t* q;    // [B, n_in]
    const float* s_x;   // [B, n_kt]
    int64_t B;
    int n_split;        // K split
    float* partials;    // [n_split, B, m]
    int32_t* acc_i32;   // [n_kt, B, m] or null
};

template <int LAT, int NB>
__global__ void __launch_bounds__(128)
k_linear_generic(LinearParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    // carve: A tile | B tile | U scratch | small
    const int n = p.n;
    const int n_atoms = (n + 127) / 128;
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sA = smem;
    uint8_t* sB = sA + n_atoms * 128 * 128;
    uint32_t* urows = (uint32_t*)(sB + n_atoms * NB * 128);  // [128][GEN_UCAP+1]
    float* s_sx = (float*)(urows + 128 * (GEN_UCAP + 1));    // [NB]
    uint64_t* bar = (uint64_t*)(s_sx + NB);
    uint32_t* tmem_slot = (uint32_t*)(bar + 1);
    uint32_t* lut_s = tmem_slot + 2;                         // [2][256] phase-1 table of the fast row decoders
    uint32_t* scr = lut_s + 512;                             // [128][n/8 + 1] nibble words
    for (int i = threadIdx.x; i < 512; i += 128) lut_s[i] = unary_lut_entry(i & 255, i >> 8);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int64_t n_bt = (p.B + NB - 1) / NB;
    int64_t item = blockIdx.x;
    const int split = (int)(item % p.n_split); item /= p.n_split;
    const int64_t bt = item % n_bt;
    const int64_t rb = item / n_bt;
    const int64_t kt_per = (p.n_kt + p.n_split - 1) / p.n_split;
    const int64_t kt0 = split * kt_per, kt1 = min(p.n_kt, kt0 + kt_per);
    const int64_t b0 = bt * NB;
    const int64_t r = rb * 128 + tid;
    const int rw_words = (p.rbits + 31) / 32;

    constexpr uint32_t TCOLS = NB < 32 ? 32 : NB;
    if (warp == 0) tmem_alloc(tmem_slot, TCOLS);
    if (tid == 0) { mbar_init(bar, 1); mbar_fence_init(); }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const uint32_t idesc = make_idesc_i8(128, NB);
    uint32_t phase = 0;
    uint32_t* urow = urows + tid * (GEN_UCAP + 1);

    float yacc[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) yacc[b] = 0.0f;

    for (int64_t kt = kt0; kt < kt1; ++kt) {
        const int64_t g = rb * p.n_kt + kt;
        SubGroup sg = sub_group(p.blob + 16 * (size_t)p.group_off[g * 4 + warp], rw_words);
        // B operand: NB rows x n K-bytes, 16-byte chunks
        {
            const int chunks_per_row = n / 16;
            for (int v = tid; v < NB * chunks_per_row; v += 128) {
                int bb = v / chunks_per_row, c16 = v % chunks_per_row;
                uint4 val = make_uint4(0, 0, 0, 0);
                if (b0 + bb < p.B) val = __ldg((const uint4*)(p.q + (b0 + bb) * (p.n_kt * n) + kt * n + c16 * 16));
                *(uint4*)(sB + sw128_offset(NB, bb, c16 * 16)) = val;
            }
            if (tid < NB) s_sx[tid] = (b0 + tid < p.B) ? p.s_x[(b0 + tid) * p.n_kt + kt] : 0.0f;
        }
        const uint32_t ul = sg.ulen[lane], nw = (ul + 31) >> 5;
        const float rho = f16_bits_to_f32(sg.norm[lane]);
        gather_u_words(sg.uarea, nw, lane, urow, GEN_UCAP);
        __syncwarp();
        if (r < p.m) {
            // fast row decoder (hq_generic_fast.cuh): codes four per word, natural coordinate order, into the swizzled A tile
            for (uint32_t i = nw; i < GEN_UCAP; ++i) urow[i] = 0u;
            const uint32_t row_a = smem_u32(sA) + (uint32_t)((tid >> 3) * 1024 + (tid & 7) * 128);
            const bool ok = decode_row_fast<LAT>(urow, GEN_UCAP, ul, sg.rarea, lane, n, p.k0, p.k1, smem_u32(lut_s),
                                                 smem_u32(scr + tid * (n / 8 + 1)), [&](int wi, uint32_t v) {
                const int col = 4 * wi;
                sts32(row_a + (uint32_t)((col >> 7) * 128 * 128) + (uint32_t)(((((col & 127) >> 4) ^ (tid & 7)) << 4) | (col & 15)), v);
            });
            if (!ok) {   // a quotient >= 16, a long row, k > 3, D4 at tile 64: the clz walker
                WordsRowU uw{urow, sg.uarea, sg.ulen, nw, GEN_UCAP, lane};
                WordsRowR rw{sg.rarea, lane, rw_words};
                decode_row_generic<LAT>(rw, 0u, uw, 0u, n, p.k0, p.k1, [&](int bk, const int* c) {
#pragma unroll
                    for (int e = 0; e < LAT; ++e) sA[sw128_offset(128, tid, bk * LAT + e)] = (uint8_t)(int8_t)c[e];
                });
            }
        } else {
            for (int j = 0; j < n; j += 16) *(uint4*)(sA + sw128_offset(128, tid, j)) = make_uint4(0, 0, 0, 0);
        }
        fence_proxy_async_smem();
        __syncthreads();
        if (tid == 0) {
            tc_fence_after();
            const uint32_t a0 = smem_u32(sA), bb0 = smem_u32(sB);
            for (int ks = 0; ks < n / 32; ++ks) {
                uint32_t aoff = (uint32_t)((ks >> 2) * 128 * 128 + (ks & 3) * 32);
                uint32_t boff = (uint32_t)((ks >> 2) * NB * 128 + (ks & 3) * 32);
                mma_i8(tmem_base, make_desc_sw128(a0 + aoff), make_desc_sw128(bb0 + boff), idesc, ks > 0);
            }
            mma_commit(bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
        tc_fence_after();
        const float sw = rho * p.inv_A;
#pragma unroll
        for (int c0 = 0; c0 < NB; c0 += 16) {
            uint32_t v[16];
            tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + c0, v);
            tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                int a = (int)v[e];
                if (p.acc_i32 && r < p.m && b0 + c0 + e < p.B) p.acc_i32[(kt * p.B + b0 + c0 + e) * p.m + r] = a;
                yacc[c0 + e] += (sw * s_sx[c0 + e]) * (float)a;
            }
        }
        tc_fence_before();
        __syncthreads();
    }
    if (r < p.m) {
#pragma unroll
        for (int b = 0; b < NB; ++b)
            if (b0 + b < p.B) p.partials[((int64_t)split * p.B + b0 + b) * p.m + r] = yacc[b];
    }
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem_base, TCOLS);
}

// y[b, r] = sum over splits (in order) -> fp32 and bf16
__global__ void k_linear_finalize(const float* partials, int n_split, int64_t B, int64_t m, __nv_bfloat16* y,
                                  int64_t ldy, float* y_f32) {
    griddep_launch();
    griddep_wait();
    int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (idx >= B * m) return;
    float s = 0.0f;
    for (int sp = 0; sp < n_split; ++sp) s += partials[(int64_t)sp * B * m + idx];
    int64_t b = idx / m, r = idx % m;
    if (y) y[b * ldy + r] = __float2bfloat16_rn(s);
    if (y_f32) y_f32[idx] = s;
}

static int generic_split(const hq_ctx* ctx, const hq_weight* w, int64_t B) {
    int NB = B <= 16 ? 16 : 64;
    int64_t n_bt = (B + NB - 1) / NB;
    int64_t items = w->n_rb * n_bt;
    int target = ctx->sm_count * 4;
    int split = 1;
    while (items * split < target && split * 2 <= w->n_kt) split *= 2;
    return split;
}

template <int NB>
static hq_status launch_generic_nb(hq_ctx* ctx, const hq_weight* w, LinearParams& p, cudaStream_t st) {
    int n_atoms = (w->n + 127) / 128;
    int64_t n_bt = (p.B + NB - 1) / NB;
    int64_t grid = w->n_rb * n_bt * p.n_split;
    size_t smem = 1024 + (size_t)n_atoms * 128 * 128 + (size_t)n_atoms * NB * 128 + 128 * (size_t)(GEN_UCAP + 1) * 4 +
                  NB * 4 + 16 + 8 + 8 + 2048 + 128 * (size_t)(w->n / 8 + 1) * 4;
#define HQ_L(L)                                                                                                   \
    do {                                                                                                          \
        HQ_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_linear_generic<L, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        k_linear_generic<L, NB><<<(unsigned)grid, 128, smem, st>>>(p);                                            \
    } while (0)
    switch (w->lattice) {
        case LAT_Z: HQ_L(LAT_Z); break;
        case LAT_A2: HQ_L(LAT_A2); break;
        case LAT_D4: HQ_L(LAT_D4); break;
        default: HQ_L(LAT_E8); break;
    }
#undef HQ_L
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    return HQ_OK;
}

// ---- E8 fast path -----------------------------------------------------------------------------
bool linear_uses_e8_fast(const hq_weight* w) { return w->lattice == LAT_E8 && w->n == 128 && w->k0 <= 3; }

// activation rows from which the decode-once large-M path is used (measured crossover)
constexpr int64_t LG_MIN_B = 64;
struct E8Plan { int NB, BC, NWG, CPS, n_bt, n_split, L, n_items, grid; };
// plan for a group of weights that share n_in (their row blocks are stacked into one item space)
static E8Plan e8_plan(const hq_ctx* ctx, int64_t n_rb_total, int64_t n_kt64, int64_t n_in, int64_t B) {
    E8Plan pl;
    pl.NB = B <= 16 ? 16 : 64;
    pl.BC = B == 1 ? 1 : pl.NB;
    pl.NWG = B == 1 ? 6 : (B <= 16 ? 5 : 3);
    pl.CPS = 1;   // (two half-size CTAs per SM, to overlap launches, measured 2 % slower: DESIGN.md §6.1)
    pl.n_bt = (int)((B + pl.NB - 1) / pl.NB);
    const int n_kt = (int)n_kt64;
    // K split.  Every item end costs a release fence + an arrival atomic per warp and one fp32 partial per row, so
    // items should be long, but the Llama-shaped matrices have too few row blocks to fill 148 x NWG warp groups
    // without splitting K finely.  Measured at batch 1: items of two tiles beat one and four.
    // Never more partial-sum traffic than half of the compressed weight bytes (matters for batch > 1; measured at batch 16).
    int split = n_kt;
    for (int d = 1; d <= n_kt; ++d)
        if (n_kt % d == 0 && n_kt / d <= 2) { split = d; break; }
    const double budget = 0.50 * 0.53 * (double)n_in / (8.0 * (double)B);
    while (split > 1 && (double)split > budget) {   // next smaller divisor
        int d = split - 1;
        while (d > 1 && n_kt % d != 0) --d;
        split = d;
    }
    pl.n_split = split;
    pl.L = n_kt / split;
    pl.n_items = (int)(n_rb_total * pl.n_bt * split);
    const int ctas = ctx->sm_count * pl.CPS;
    pl.grid = pl.n_items < ctas ? pl.n_items : ctas;
    return pl;
}

template <int NB, int BC, int NWG, int CPS>
static hq_status launch_e8_v(hq_ctx* ctx, int k0, E8Params& p, const E8Plan& pl, cudaStream_t st) {
    const size_t smem = e8_smem_bytes<NB, NWG>();
    dim3 grid((unsigned)pl.grid);
#define HQ_LE(KK)                                                                                                   \
    case KK:                                                                                                        \
        HQ_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_linear_e8<KK, NB, BC, NWG, CPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        HQ_CUDA_CHECK(ctx, launch_pdl(k_linear_e8<KK, NB, BC, NWG, CPS>, grid, dim3(NWG * 128), smem, st, p));           \
        break
    switch (k0) {
        HQ_LE(0); HQ_LE(1); HQ_LE(2); HQ_LE(3);
    }
#undef HQ_LE
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    return HQ_OK;
}

// batch 1: k_gemv_e8 (decoded rows through tensor memory, independent warps, activations quantized in-kernel)
// Warp groups per CTA: 5 or 4, whichever wastes fewer tile slots.  The flat partition gives every warp group floor or ceil
// of T / (SMs x NWG) tiles and the launch ends with the slowest one, so its length is ~ ceil(T / (SMs x NWG)) x NWG
// (a tile takes a warp NWG x as long when NWG groups share the SM's issue slots).
constexpr int GV_NWG = 5;   // the largest: sizes the partial-sum slots
static int gv_pick_nwg(const hq_ctx* ctx, int64_t T) {
    const int64_t sm = ctx->sm_count;
    const int64_t c5 = (T + sm * 5 - 1) / (sm * 5) * 5, c4 = (T + sm * 4 - 1) / (sm * 4) * 4;
    return c4 < c5 ? 4 : 5;
}
template <int NWG>
static hq_status launch_gemv(hq_ctx* ctx, int k0, E8Params& p, const E8Plan& pl, cudaStream_t st) {
    const size_t smem = gv_smem_bytes<NWG>(p.n_kt);
    dim3 grid((unsigned)ctx->sm_count);   // flat partition of the items over all warp groups of the device
#define HQ_LG(KK)                                                                                                   \
    case KK:                                                                                                        \
        HQ_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_gemv_e8<KK, NWG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        HQ_CUDA_CHECK(ctx, launch_pdl(k_gemv_e8<KK, NWG>, grid, dim3(NWG * 128), smem, st, p));                      \
        break
    switch (k0) {
        HQ_LG(0); HQ_LG(1); HQ_LG(2); HQ_LG(3);
    }
#undef HQ_LG
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    return HQ_OK;
}

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }
// partial-sum slots per row block of the batch-1 kernel: the segments a row block's K range can be cut into by the flat
// tile partition over G warp groups (hq_gemv_e8.cuh); sized for the largest G the launcher may use
static int64_t gv_slots(const hq_ctx* ctx, int64_t n_rb_total, int64_t n_kt) {
    const int64_t T = n_rb_total * n_kt, G = (int64_t)ctx->sm_count * GV_NWG;
    const int64_t per = T / G > 0 ? T / G : 1;
    const int64_t s = (n_kt + per - 1) / per + 1;
    return s < n_kt + 1 ? s : n_kt + 1;
}

// weights that may share one launch: the E8 fast path, same n_in / k / seed (= same RHT signs) / operating point
bool linear_group_compatible(const hq_weight* const* ws, int n_w) {
    if (n_w < 1 || n_w > E8_MAXW) return false;
    for (int i = 0; i < n_w; ++i) {
        if (!linear_uses_e8_fast(ws[i])) return false;
        if (ws[i]->n_in != ws[0]->n_in || ws[i]->k0 != ws[0]->k0 || ws[i]->seed != ws[0]->seed ||
            ws[i]->snr_db != ws[0]->snr_db)
            return false;
    }
    return true;
}

size_t linear_group_workspace_bytes(const hq_ctx* ctx, const hq_weight* const* ws, int n_w, int64_t B) {
    int64_t n_rb = 0;
    for (int i = 0; i < n_w; ++i) n_rb += ws[i]->n_rb;
    E8Plan pl = e8_plan(ctx, n_rb, ws[0]->n_kt, ws[0]->n_in, B);
    size_t bytes = align256((size_t)pl.n_bt * ws[0]->n_kt * e8_bblob_bytes(pl.NB));
    const int64_t slots = B == 1 ? gv_slots(ctx, n_rb, ws[0]->n_kt) : 0;
    if (pl.n_split > 1 || B == 1)
        for (int i = 0; i < n_w; ++i) bytes += align256((size_t)(slots > pl.n_split ? slots : pl.n_split) * B * ws[i]->m * 4);
    if (B >= LG_MIN_B) {   // the large-M path: activation blob of 256-row tiles + the decoded copy of the largest weight
        int64_t rb_max = 0;
        for (int i = 0; i < n_w; ++i) rb_max = ws[i]->n_rb > rb_max ? ws[i]->n_rb : rb_max;
        bytes += align256((size_t)((B + LG_NB - 1) / LG_NB) * (ws[0]->n_in / 128) * LG_BBLOB) + align256((size_t)rb_max * (ws[0]->n_in / 128) * LG_ABLOB);
    }
    return bytes + 256;
}

// E8 / tile 256 takes the large-M path only (from LG_MIN_B activation rows); below that the generic kernel
static bool linear_uses_e8_large256(const hq_weight* w, int64_t B) {
    return w->lattice == LAT_E8 && w->n == 256 && w->k0 <= 3 && B >= LG_MIN_B;
}

size_t linear_workspace_bytes(const hq_ctx* ctx, const hq_weight* w, int64_t B) {
    if (linear_uses_e8_fast(w)) return linear_group_workspace_bytes(ctx, &w, 1, B);
    if (linear_uses_e8_large256(w, B))
        return align256((size_t)((B + LG_NB - 1) / LG_NB) * (w->n_in / 128) * LG_BBLOB) + align256((size_t)w->n_rb * (w->n_in / 128) * LG_ABLOB) + 256;
    int ns = generic_split(ctx, w, B);
    return align256((size_t)(B * w->n_in)) + align256((size_t)(B * w->n_kt) * 4) + (size_t)ns * B * w->m * 4 + 256;
}

// Large-M path (hq_linear_large.cuh): activation blob of 256-row tiles, then per weight one decode into the operand-layout
// scratch copy and one warp-specialised GEMM.  The scratch copy is reused by the weights of a group (stream order).
static hq_status launch_large(hq_ctx* ctx, const hq_weight* const* ws, int n_w, const void* x, int dtype, int64_t B,
                              int64_t ldx, void* const* ys_bf16, const int64_t* ldys, float* const* ys_f32, int32_t* acc_i32,
                              uint8_t* wsbuf, cudaStream_t st, int fp8 = 0) {
    const hq_weight* w0 = ws[0];
    const int64_t n_bt = (B + LG_NB - 1) / LG_NB;
    const int nch = w0->n / 128;                       // operand chunks of 128 K-bytes per RHT tile (tile 128 or 256)
    const int64_t n_kt128 = w0->n_in / 128;
    uint8_t* bblob = wsbuf;
    uint8_t* ablob = wsbuf + align256((size_t)n_bt * n_kt128 * LG_BBLOB);
    // fork: the first weight's decode does not depend on x, it runs on the side stream beside the activation cast
    HQ_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev_fork, st));
    HQ_CUDA_CHECK(ctx, cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0));
    if (nch == 1) launch_act_blob(x, dtype, B, w0->n_in, ldx, w0->dsign, LG_NB, bblob, st, fp8);
    else launch_act_blob256(x, dtype, B, w0->n_in, ldx, w0->dsign, LG_NB, bblob, st, fp8);
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (ctx->prof) {
        HQ_CUDA_CHECK(ctx, cudaEventCreate(&e0));
        HQ_CUDA_CHECK(ctx, cudaEventCreate(&e1));
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e0, st));
    }
    for (int i = 0; i < n_w; ++i) {
        const hq_weight* w = ws[i];
        E8AblobParams d;
        d.blob = w->blob; d.sub_off = w->group_off; d.lut = ctx->e8_lut; d.ablob = ablob; d.m = w->m;
        d.n_kt = (int)w->n_kt;
        d.inv_A = (float)(1.0 / (w->alpha * sqrt((double)w->n)));
        d.n_rb = (int)w->n_rb;
        const size_t dsmem = E8_LUT_BYTES + 256 * (size_t)(w->n / 8 + 1) * 4 + 16;
        const int64_t dpairs = ((int64_t)w->n_rb * d.n_kt + 1) / 2, dmax = (int64_t)ctx->sm_count * 3;   // 3 CTAs of 256 threads per SM
        dim3 dgrid((unsigned)(dpairs < dmax ? dpairs : dmax));
        cudaStream_t dst = i == 0 ? ctx->side : st;   // later weights reuse the scratch copy: stream order after the GEMM
#define HQ_LD1(KK, TT, F8)                                                                                                 \
    do {                                                                                                                   \
        HQ_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_e8_decode_ablob<KK, TT, F8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dsmem)); \
        k_e8_decode_ablob<KK, TT, F8><<<dgrid, 256, dsmem, dst>>>(d);                                                      \
    } while (0)
#define HQ_LD(KK)                                                                                                          \
    case KK:                                                                                                               \
        if (nch == 1) { if (fp8) HQ_LD1(KK, 128, true); else HQ_LD1(KK, 128, false); }                                     \
        else { if (fp8) HQ_LD1(KK, 256, true); else HQ_LD1(KK, 256, false); }                                              \
        break
        switch (w->k0) { HQ_LD(0); HQ_LD(1); HQ_LD(2); HQ_LD(3); }
#undef HQ_LD
#undef HQ_LD1
        HQ_CUDA_CHECK(ctx, cudaGetLastError());
        if (i == 0) {   // join
            HQ_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev_join, ctx->side));
            HQ_CUDA_CHECK(ctx, cudaStreamWaitEvent(st, ctx->ev_join, 0));
        }
        E8LargeParams g;
        g.ablob = ablob; g.bblob = bblob; g.y_bf16 = (__nv_bfloat16*)ys_bf16[i]; g.y_f32 = ys_f32 ? ys_f32[i] : nullptr;
        g.ldy = ldys[i]; g.m = w->m; g.B = B; g.n_rb = (int)w->n_rb; g.n_bt = (int)n_bt; g.n_kt = (int)n_kt128;
        g.acc_i32 = (n_w == 1) ? acc_i32 : nullptr;
        const int64_t tiles = (int64_t)g.n_rb * g.n_bt;
        const unsigned grid = (unsigned)(tiles < ctx->sm_count ? tiles : ctx->sm_count);
#define HQ_LGEMM(NCH_, F8)                                                                                                 \
    do {                                                                                                                   \
        HQ_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_e8_gemm_large<NCH_, F8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LG_SMEM)); \
        k_e8_gemm_large<NCH_, F8><<<grid, 384, LG_SMEM, st>>>(g);                                                          \
    } while (0)
        if (nch == 1) { if (fp8) HQ_LGEMM(1, true); else HQ_LGEMM(1, false); }
        else { if (fp8) HQ_LGEMM(2, true); else HQ_LGEMM(2, false); }
#undef HQ_LGEMM
        HQ_CUDA_CHECK(ctx, cudaGetLastError());
    }
    if (ctx->prof) {
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e1, st));
        ctx->prof_ev.push_back(e0);
        ctx->prof_ev.push_back(e1);
    }
    return HQ_OK;
}

// hq_linear_cast with HQ_CAST_FP8_E4M3 (§4.8): the large-M pipeline with E4M3 operands and an fp32 accumulator
hq_status launch_linear_fp8(hq_ctx* ctx, const hq_weight* w, const void* x, int dtype, int64_t B, int64_t ldx, void* y_bf16,
                            int64_t ldy, float* y_f32, float* acc_f32, uint8_t* wsbuf, cudaStream_t st) {
    // the debug copy of the accumulators travels through the INT8 path's pointer: the kernel stores the TMEM words as they are
    return launch_large(ctx, &w, 1, x, dtype, B, ldx, &y_bf16, &ldy, &y_f32, (int32_t*)acc_f32, wsbuf, st, 1);
}

// one activation cast, ONE fused decode + MMA launch over the stacked row blocks of all weights, one finalize each
hq_status launch_linear_group(hq_ctx* ctx, const hq_weight* const* ws, int n_w, const void* x, int dtype, int64_t B,
                              int64_t ldx, void* const* ys_bf16, const int64_t* ldys, float* const* ys_f32,
                              int32_t* acc_i32, uint8_t* wsbuf, cudaStream_t st, const hq_fold* fold) {
    const hq_weight* w0 = ws[0];
    int64_t n_rb = 0;
    for (int i = 0; i < n_w; ++i) n_rb += ws[i]->n_rb;
    if (fold && (B != 1 || w0->n_kt > GV_MAX_KT || dtype != HQ_BF16)) {   // the folds live in the batch-1 kernel's prologue / epilogue
        ctx->err = "the RMSNorm / SiLU.mul / residual folds need batch 1, bf16 and n_in <= 16384";
        return HQ_ERR_UNSUPPORTED;
    }
    if (B >= LG_MIN_B) return launch_large(ctx, ws, n_w, x, dtype, B, ldx, ys_bf16, ldys, ys_f32, acc_i32, wsbuf, st);
    E8Plan pl = e8_plan(ctx, n_rb, w0->n_kt, w0->n_in, B);
    // the tile descriptor of the fused kernel packs its fields (hq_linear_e8.cuh E8Desc): reject shapes that would alias
    for (int i = 0; i < n_w; ++i)
        if (ws[i]->n_rb >= 65536 || ws[i]->n_rb * w0->n_kt >= (1ll << 31)) { ctx->err = "m_out too large for the fused kernel (< 8388608 rows, row blocks x K-tiles < 2^31)"; return HQ_ERR_SHAPE; }
    if (w0->n_kt >= 4096 || pl.n_bt >= 4096 || pl.n_split >= 4096) { ctx->err = "n_in / n_tile and batch tiles must be below 4096 on the fused path"; return HQ_ERR_SHAPE; }
    uint8_t* bblob = wsbuf;
    uint8_t* at = wsbuf + align256((size_t)pl.n_bt * w0->n_kt * e8_bblob_bytes(pl.NB));
    const bool gemv = B == 1 && w0->n_kt <= GV_MAX_KT;   // the batch-1 kernel quantizes x itself
    if (!gemv) {
        launch_act_blob(x, dtype, B, w0->n_in, ldx, w0->dsign, pl.NB, bblob, st);
        HQ_CUDA_CHECK(ctx, cudaGetLastError());
    }
    E8Params p;
    memset(&p, 0, sizeof(p));
    uint32_t min_ulen = 0xffffffffu;
    p.rb_base[0] = 0;
    for (int i = 0; i < n_w; ++i) {
        p.blob[i] = ws[i]->blob; p.sub_off[i] = ws[i]->group_off; p.m[i] = ws[i]->m;
        p.partials[i] = (float*)at;
        const int64_t slots = B == 1 ? gv_slots(ctx, n_rb, w0->n_kt) : 0;
        if (pl.n_split > 1 || B == 1) at += align256((size_t)(slots > pl.n_split ? slots : pl.n_split) * B * ws[i]->m * 4);
        p.inv_A[i] = (float)(1.0 / (ws[i]->alpha * sqrt((double)ws[i]->n)));
        p.rb_base[i + 1] = p.rb_base[i] + (int)ws[i]->n_rb;
        if (ws[i]->min_ulen < min_ulen) min_ulen = ws[i]->min_ulen;
    }
    for (int i = n_w; i < E8_MAXW; ++i) p.rb_base[i + 1] = p.rb_base[n_w];
    for (int i = 0; i < n_w; ++i) {
        p.y_bf16[i] = (__nv_bfloat16*)ys_bf16[i]; p.ldy[i] = ldys[i]; p.y_f32[i] = ys_f32 ? ys_f32[i] : nullptr;
    }
    // split-arrival counters: zero whenever the kernel is not running (the last arrival resets its counter)
    const size_t cnt_need = (size_t)n_rb * pl.n_bt * 4 * sizeof(unsigned int);
    if (cnt_need > ctx->e8_cnt_bytes) {
        if (ctx->e8_cnt) { HQ_CUDA_CHECK(ctx, cudaDeviceSynchronize()); ctx->alloc.free(ctx->alloc.user, ctx->e8_cnt); ctx->e8_cnt = nullptr; ctx->e8_cnt_bytes = 0; }
        const size_t cap = cnt_need < (1u << 16) ? (1u << 16) : 2 * cnt_need;
        ctx->e8_cnt = (unsigned int*)ctx->alloc.alloc(ctx->alloc.user, cap);
        if (!ctx->e8_cnt) { ctx->err = "allocator returned NULL for the split counters"; return HQ_ERR_ALLOC; }
        ctx->e8_cnt_bytes = cap;
        HQ_CUDA_CHECK(ctx, cudaMemsetAsync(ctx->e8_cnt, 0, cap, st));
    }
    p.counters = ctx->e8_cnt;
    p.n_w = n_w; p.lut = ctx->e8_lut;
    p.n_kt = (int)w0->n_kt; p.n_split = pl.n_split; p.L = pl.L; p.n_items = pl.n_items; p.n_bt = pl.n_bt;
    p.u_dense = ((min_ulen + 31) >> 5) >= (uint32_t)E8_DENSE ? E8_DENSE : 0;
    p.bblob = bblob; p.B = B; p.acc_i32 = (n_w == 1) ? acc_i32 : nullptr;
    p.x = x; p.dtype = dtype; p.dsign = w0->dsign;
    if (fold) {
        p.fold_mode = fold->mode; p.fold_eps = fold->eps; p.fold_aux = (const __nv_bfloat16*)fold->aux_dev;
        for (int i = 0; i < n_w; ++i) p.res[i] = fold->residuals_dev ? (const __nv_bfloat16*)fold->residuals_dev[i] : nullptr;
    }
    if (gemv) p.n_items = (int)(n_rb * w0->n_kt);   // the batch-1 kernel partitions tiles, not items
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (ctx->prof) {
        HQ_CUDA_CHECK(ctx, cudaEventCreate(&e0));
        HQ_CUDA_CHECK(ctx, cudaEventCreate(&e1));
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e0, st));
    }
    hq_status s = gemv        ? (gv_pick_nwg(ctx, p.n_items) == 4 ? launch_gemv<4>(ctx, w0->k0, p, pl, st) : launch_gemv<5>(ctx, w0->k0, p, pl, st))
                  : (B == 1)  ? launch_e8_v<16, 1, 6, 1>(ctx, w0->k0, p, pl, st)
                  : (B <= 16) ? launch_e8_v<16, 16, 5, 1>(ctx, w0->k0, p, pl, st)
                              : launch_e8_v<64, 64, 3, 1>(ctx, w0->k0, p, pl, st);
    if (s != HQ_OK) return s;
    if (ctx->prof) {
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e1, st));
        ctx->prof_ev.push_back(e0);
        ctx->prof_ev.push_back(e1);
    }
    return HQ_OK;
}

// decode-only ceiling measurement (hq_e8_ceiling.cuh)
template <int NWG>
static hq_status decode_ceiling_nwg(hq_ctx* ctx, const hq_weight* w, int reps, cudaStream_t st, double* scalars_per_s) {
    E8CeilParams p;
    p.blob = w->blob; p.sub_off = w->group_off; p.lut = ctx->e8_lut; p.n_groups = 4 * w->G; p.reps = reps;
    const size_t threads = (size_t)ctx->sm_count * NWG * 128;
    p.sink = (unsigned int*)ctx->alloc.alloc(ctx->alloc.user, threads * 4);
    if (!p.sink) { ctx->err = "allocator returned NULL"; return HQ_ERR_ALLOC; }
    const size_t smem = 1024 + E8_LUT_BYTES + (size_t)NWG * (16384 + 128 * E8_SCR_STRIDE * 4);
    cudaEvent_t e0, e1;
    HQ_CUDA_CHECK(ctx, cudaEventCreate(&e0));
    HQ_CUDA_CHECK(ctx, cudaEventCreate(&e1));
    float ms = 0.0f;
#define HQ_CE(KK)                                                                                                       \
    case KK:                                                                                                            \
        HQ_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_e8_decode_ceiling<KK, NWG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        p.reps = 2; k_e8_decode_ceiling<KK, NWG><<<ctx->sm_count, NWG * 128, smem, st>>>(p);   /* warm-up */                \
        p.reps = reps;                                                                                                  \
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e0, st));                                                                    \
        k_e8_decode_ceiling<KK, NWG><<<ctx->sm_count, NWG * 128, smem, st>>>(p);                                        \
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e1, st));                                                                    \
        break
    switch (w->k0) { HQ_CE(0); HQ_CE(1); HQ_CE(2); HQ_CE(3); }
#undef HQ_CE
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    HQ_CUDA_CHECK(ctx, cudaEventSynchronize(e1));
    HQ_CUDA_CHECK(ctx, cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    ctx->alloc.free(ctx->alloc.user, p.sink);
    *scalars_per_s = (double)threads * 128.0 * reps / (ms * 1e-3);
    return HQ_OK;
}
// reps < 0: |reps| repetitions with 4 warp groups (16 warps per SM) instead of the fused kernel's 6
hq_status launch_decode_ceiling(hq_ctx* ctx, const hq_weight* w, int reps, cudaStream_t st, double* scalars_per_s) {
    return reps > 0 ? decode_ceiling_nwg<6>(ctx, w, reps, st, scalars_per_s) : decode_ceiling_nwg<4>(ctx, w, -reps, st, scalars_per_s);
}

hq_status launch_linear(hq_ctx* ctx, const hq_weight* w, const void* x, int dtype, int64_t B, int64_t ldx,
                        void* y_bf16, int64_t ldy, float* y_f32, int32_t* acc_i32, uint8_t* ws, cudaStream_t st) {
    if (linear_uses_e8_fast(w))
        return launch_linear_group(ctx, &w, 1, x, dtype, B, ldx, &y_bf16, &ldy, &y_f32, acc_i32, ws, st);
    if (linear_uses_e8_large256(w, B)) return launch_large(ctx, &w, 1, x, dtype, B, ldx, &y_bf16, &ldy, &y_f32, acc_i32, ws, st);
    const float inv_A = (float)(1.0 / (w->alpha * sqrt((double)w->n)));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int8_t* q = (int8_t*)ws;
    float* s_x = (float*)(ws + align256((size_t)(B * w->n_in)));
    float* partials = (float*)((uint8_t*)s_x + align256((size_t)(B * w->n_kt) * 4));
    const int n_split = generic_split(ctx, w, B);
    launch_act_quant(x, dtype, B, w->n_in, ldx, w->lattice, w->n, w->dsign, q, s_x, nullptr, st);
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    LinearParams p;
    p.blob = w->blob; p.group_off = w->group_off; p.m = w->m; p.n_kt = w->n_kt;
    p.n = w->n; p.k0 = w->k0; p.k1 = w->k1; p.rbits = w->rbits; p.inv_A = inv_A;
    p.q = q; p.s_x = s_x; p.B = B; p.n_split = n_split; p.partials = partials; p.acc_i32 = acc_i32;
    if (ctx->prof) {
        HQ_CUDA_CHECK(ctx, cudaEventCreate(&e0));
        HQ_CUDA_CHECK(ctx, cudaEventCreate(&e1));
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e0, st));
    }
    hq_status s = (B <= 16) ? launch_generic_nb<16>(ctx, w, p, st) : launch_generic_nb<64>(ctx, w, p, st);
    if (s != HQ_OK) return s;
    if (ctx->prof) {
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e1, st));
        ctx->prof_ev.push_back(e0);
        ctx->prof_ev.push_back(e1);
    }
    int64_t tot = B * w->m;
    HQ_CUDA_CHECK(ctx, launch_pdl(k_linear_finalize, dim3((unsigned)((tot + 255) / 256)), dim3(256), 0, st, (const float*)partials,
                                  n_split, B, w->m, (__nv_bfloat16*)y_bf16, ldy, y_f32));
    return HQ_OK;
}

}  // namespace hq

// ---------------------------------------------------------------------------------------------
// hq_linear_static (include/hq.h): the batch-1 fused kernel (k_gemv_e8) with its scratch - the split-K arrival
// counters and partial sums - in a file-scope device array instead of the context's allocator-backed workspace, for
// callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Every GPU
// that loads the library holds the array until the process exits.  All calls share it and it keeps the last call's
// contents: the counters are cleared on the caller's stream before every launch; the partial sums need no clearing
// (every slot that is read was written by the same launch).  Calls that overlap on the GPU race on it.
namespace hq {

constexpr size_t ST_CNT_BYTES = 32u * 1024u;                       // 2048 row blocks x 4 warps x u32
constexpr size_t ST_PART_BYTES = HQ_LINEAR_STATIC_SCRATCH_BYTES - ST_CNT_BYTES;
static __device__ __align__(256) unsigned char g_static_scratch[HQ_LINEAR_STATIC_SCRATCH_BYTES];

// The array's name is a host-side stand-in in host code, not a device address: the address a kernel may use comes from
// cudaGetSymbolAddress, asked once per device with that device current (hq_create calls this).
constexpr int ST_MAX_DEV = 64;
static std::mutex g_static_mu;
static void* g_static_ptr[ST_MAX_DEV];

hq_status linear_static_setup(hq_ctx* ctx) {
    if (ctx->device < 0 || ctx->device >= ST_MAX_DEV) { ctx->err = "device index beyond the static scratch table"; return HQ_ERR_UNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[ctx->device]) {
        void* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
        if (e != cudaSuccess || !ptr) {
            ctx->err = std::string("cudaGetSymbolAddress(static scratch): ") + cudaGetErrorString(e);
            return HQ_ERR_CUDA;
        }
        g_static_ptr[ctx->device] = ptr;
    }
    ctx->static_scratch = (uint8_t*)g_static_ptr[ctx->device];
    return HQ_OK;
}

hq_status launch_linear_static(hq_ctx* ctx, const hq_weight* w, const void* x, int dtype, void* y_bf16, float* y_f32,
                               cudaStream_t st) {
    if (!ctx->static_scratch) { ctx->err = "the static scratch address was not obtained at hq_create"; return HQ_ERR_CUDA; }
    if (!linear_uses_e8_fast(w) || w->n_kt > GV_MAX_KT) {
        ctx->err = "hq_linear_static takes E8 / tile 128 / k <= 3 weights with n_in <= 16384";
        return HQ_ERR_UNSUPPORTED;
    }
    const int64_t n_rb = w->n_rb, n_kt = w->n_kt;
    if (n_rb >= 65536 || n_rb * n_kt >= (1ll << 31)) { ctx->err = "m_out too large for the fused kernel"; return HQ_ERR_SHAPE; }
    const size_t cnt_need = (size_t)n_rb * 4 * sizeof(unsigned int);
    const size_t part_need = (size_t)gv_slots(ctx, n_rb, n_kt) * (size_t)w->m * 4;
    if (cnt_need > ST_CNT_BYTES || part_need > ST_PART_BYTES) {
        ctx->err = "hq_linear_static: this weight needs " + std::to_string(cnt_need) + " counter bytes and " + std::to_string(part_need) +
                   " partial-sum bytes; the static scratch holds " + std::to_string(ST_CNT_BYTES) + " + " + std::to_string(ST_PART_BYTES) +
                   " (m_out <= 262144): use hq_linear";
        return HQ_ERR_SHAPE;
    }
    E8Plan pl = e8_plan(ctx, n_rb, n_kt, w->n_in, 1);
    E8Params p;
    memset(&p, 0, sizeof(p));
    p.blob[0] = w->blob; p.sub_off[0] = w->group_off; p.m[0] = w->m;
    p.counters = (unsigned int*)ctx->static_scratch;
    p.partials[0] = (float*)(ctx->static_scratch + ST_CNT_BYTES);
    p.inv_A[0] = (float)(1.0 / (w->alpha * sqrt((double)w->n)));
    for (int i = 0; i < E8_MAXW; ++i) p.rb_base[i + 1] = (int)n_rb;
    p.y_bf16[0] = (__nv_bfloat16*)y_bf16; p.ldy[0] = w->m; p.y_f32[0] = y_f32;
    p.n_w = 1; p.lut = ctx->e8_lut;
    p.n_kt = (int)n_kt; p.n_split = pl.n_split; p.L = pl.L; p.n_bt = 1;
    p.n_items = (int)(n_rb * n_kt);   // the batch-1 kernel partitions tiles
    p.u_dense = ((w->min_ulen + 31) >> 5) >= (uint32_t)E8_DENSE ? E8_DENSE : 0;
    p.B = 1; p.x = x; p.dtype = dtype; p.dsign = w->dsign;
    // what must start at zero: the arrival counters (the partial sums are written before they are read)
    HQ_CUDA_CHECK(ctx, cudaMemsetAsync(p.counters, 0, cnt_need, st));
    return gv_pick_nwg(ctx, p.n_items) == 4 ? launch_gemv<4>(ctx, w->k0, p, pl, st) : launch_gemv<5>(ctx, w->k0, p, pl, st);
}

}  // namespace hq
