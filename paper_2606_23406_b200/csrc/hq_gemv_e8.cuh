// hq_gemv_e8.cuh — the batch-1 fused kernel: Rice decode -> INT8 lattice points -> TENSOR MEMORY -> tcgen05.mma kind::i8
// (north_star (a)-(d); the headline path of BASELINE config 2).
//
// What differs from k_linear_e8 (hq_linear_e8.cuh, still the kernel for 2..63 activation rows):
//  * the decoded tile never touches shared memory.  Phase 2 leaves a row's 128 codes in registers, eight per run of 32
//    symbols; `tcgen05.st` writes them to the row's TMEM lane (lane = weight row, 32 columns per tile) and the MMA takes
//    its A operand from tensor memory (`tcgen05.mma [d], [a_tmem], b_desc`).  No A tile in shared memory, no swizzled
//    128-bit stores, no fence.proxy.async per tile.
//  * warps are independent.  A warp owns 32 rows (one sub-group, FORMAT §5) of an M = 128 instruction: it issues its own
//    four MMAs per tile with the other 96 output lanes masked off (`disable_output_lane`), commits to its own mbarrier
//    and drains its own accumulator lanes one tile later.  No arrival counters, no waiting for the slowest warp of a
//    warp group (12 % of the issued instructions of k_linear_e8 were that spin, profiles/r02_decode_ceiling.md).
//  * the activation vector is quantized IN the kernel (A1-A2: RHT + amax INT8 cast per tile of 128, FORMAT R1/R7, the
//    same warp routine as k_act_blob) into a shared-memory operand that every MMA of the CTA reads: row kt of the
//    K-major SWIZZLE_128B operand is the INT8 tile of K-tile kt, so the B descriptor of K-tile kt is the 8-row group
//    kt / 8 and the wanted accumulator column is kt % 8 (the other columns are products with other K-tiles' activations
//    and are never read).  No activation kernel, no TMA per tile, one launch per hq_linear_group at batch 1.
// Everything else is k_linear_e8's: persistent CTA per SM, contiguous item ranges, register-prefetched coalesced loads two
// levels deep, L2 prefetch, phase 1 / phase 2 of hq_e8_decode.cuh, split-K reduced in-kernel in split order.
#pragma once
#include "hq_act.cuh"
#include "hq_common.cuh"
#include "hq_e8_decode.cuh"
#include "hq_internal.h"
#include "hq_linear_e8.cuh"
#include "hq_tc.cuh"

namespace hq {


constexpr int GV_TCOLS_WG = 48;   // TMEM columns per warp group: A tile (32: 128 INT8 per lane) + accumulator (16)
constexpr int GV_MAX_KT = 128;    // n_in <= 16384: the whole activation operand stays in shared memory
constexpr int GV_STAGE_WORDS = E8_NW + 12;   // per row: the next tile's U words and R words (K <= 3), staged by cp.async

__host__ __device__ constexpr uint32_t gv_xq_bytes(int n_kt) { return (uint32_t)(((n_kt + 7) / 8 + 1) * 1024); }
template <int NWG>
__host__ __device__ constexpr size_t gv_smem_bytes(int n_kt) {
    return 1024 + (size_t)E8_LUT_BYTES + gv_xq_bytes(n_kt) + (size_t)((n_kt * 4 + 127) & ~127) +
           (size_t)NWG * 128 * (E8_SCR_STRIDE * 4 + 16 + GV_STAGE_WORDS * 4) + 8 * (NWG * 4 + 1) + 16 + GV_MAX_KT * 4;
}

// The rare row the SWAR decoder declines (a unary quotient >= 16, or more than E8_NW U words): that lane alone walks its
// U-section with clz, un-strips block by block and contracts the codes with the activation operand in shared memory
// itself; the INT32 sum replaces the lane's accumulator (bit-identical to what the MMA would give: the same integers
// in another order).  The other 31 rows of the warp, and tensor memory, are not touched.  To keep the call out of the
// tile loop (its live registers would spill), a flagged tile is only marked there - the epilogue skips the lane's
// accumulator for it - and the marked tiles are redone after the segment's loop, their terms added last.
template <int K>
__device__ int gv_row_fallback(const uint8_t* sgp, int lane, uint32_t ul, uint32_t xrow_a, uint32_t ksw) {
    constexpr int KW = 4 * K;
    const uint16_t* hdr = (const uint16_t*)sgp;
    struct { uint32_t v[KW > 0 ? KW : 1]; } rw;
#pragma unroll
    for (int j = 0; j < KW; ++j) rw.v[j] = __ldg((const uint32_t*)(sgp + 128) + j * 32 + lane);
    const uint32_t* uarea = (const uint32_t*)(sgp + 128) + KW * 32;
    // word t of this row sits at uarea[sum_i min(nw_i, t) + #{i < lane : nw_i > t}] (FORMAT §5): advance the index
    // word by word from the 32 lengths of the sub-group
    uint32_t nws[8];   // nw_i, one byte each
#pragma unroll
    for (int i = 0; i < 8; ++i) nws[i] = 0u;
    for (int i = 0; i < 32; ++i) nws[i >> 2] |= (((uint32_t)__ldg(hdr + i) + 31u) >> 5) << (8 * (i & 3));
    const uint32_t nw = (ul + 31) >> 5;
    uint32_t row_base = 0;   // words of word-rows < t
    auto word = [&](uint32_t tt) -> uint32_t {   // called with increasing tt
        if (tt >= nw) return 0u;
        uint32_t below = 0, all = 0;
        for (int i = 0; i < 32; ++i) {
            const uint32_t n = (nws[i >> 2] >> (8 * (i & 3))) & 0xffu;
            if (n > tt) { ++all; if (i < lane) ++below; }
        }
        const uint32_t v = __ldg(uarea + row_base + below);
        row_base += all;
        return v;
    };
    uint32_t tword = 0, cur = word(0), avail = 32;
    auto next_q = [&]() -> uint32_t {   // zeros up to the terminating one
        uint32_t q = 0;
        for (;;) {
            if (cur == 0u) {
                q += avail;
                if (++tword > nw) return q;   // corrupt stream guard
                cur = word(tword); avail = 32;
                continue;
            }
            const uint32_t lz = (uint32_t)__clz((int)cur);
            q += lz;
            cur = lz >= 31u ? 0u : (cur << (lz + 1));
            avail -= lz + 1;
            if (avail == 0u) { ++tword; cur = word(tword); avail = 32; }
            return q;
        }
    };
    int acc = 0;
    for (int c = 0; c < 4; ++c) {
        int zs[32];
        for (int u = 0; u < 32; ++u) {
            const uint32_t q = next_q();
            const int g = 2 * (u >> 3) + (u & 1), bl = (u & 7) >> 1;
            uint32_t r = 0;
            int lo = 0;
#pragma unroll
            for (int pb = 0; pb < 3; ++pb) {   // field planes of the remainder (FORMAT §4)
                const int wd = 1 << pb;
                if (!(K & wd)) continue;
                const int per = 8 / wd;
                const uint32_t V = rw.v[c * K + lo + g / per];
                r |= ((V >> (8 * bl + wd * (g % per))) & ((1u << wd) - 1u)) << lo;
                lo += wd;
            }
            zs[u] = (int)((q << K) | r);
        }
        for (int b = 0; b < 4; ++b) {
            int z[8], cc[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) z[i] = zs[8 * (i >> 1) + 2 * b + (i & 1)];   // stream position 8w + 2b + e, i = 2w + e
            unstrip<LAT_E8>(z, cc);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int col = 32 * c + 4 * i + b;   // e8_kcol
                uint32_t xb;
                asm volatile("ld.shared.s8 %0, [%1];" : "=r"(xb) : "r"(xrow_a + ((((col >> 4) ^ ksw) << 4) | (col & 15))) : "memory");
                acc += cc[i] * (int)xb;
            }
        }
    }
    return acc;
}

// The flagged tiles of a segment (bit kt - ka of the lane's 128-bit mask in shared memory), after the segment's tile
// loop: returns the sum of their rescaled contributions sw * s_x * acc, in K-tile order.
template <int K>
__device__ __noinline__ float gv_segment_fallback(const uint8_t* blob, const uint32_t* soff, int lane, int ka, uint32_t mask_a,
                                                  uint32_t xq_a, uint32_t sx_a, float inv_A, int32_t* acc_out, int64_t mw) {
    float corr = 0.0f;
    for (int wq = 0; wq < 4; ++wq) {
        uint32_t bits = lds32(mask_a + wq * 4);
        while (bits) {
            const int b = __ffs((int)bits) - 1;
            bits &= bits - 1;
            const int kt = ka + 32 * wq + b;
            const uint8_t* sgp = blob + 16 * (size_t)__ldg(soff + (32 * wq + b) * 4);
            const uint32_t ul = __ldg((const uint16_t*)sgp + lane);
            const float sw = f16_bits_to_f32(__ldg((const uint16_t*)sgp + 32 + lane)) * inv_A;
            const int acc = gv_row_fallback<K>(sgp, lane, ul, xq_a + (uint32_t)((kt >> 3) * 1024 + (kt & 7) * 128), (uint32_t)(kt & 7));
            if (acc_out) acc_out[(int64_t)kt * mw] = acc;
            corr += (sw * lds_f32(sx_a + kt * 4)) * (float)acc;
        }
        sts32(mask_a + wq * 4, 0u);
    }
    return corr;
}

// The bitstream words of a tile travel global -> shared by cp.async (no register is held while they fly): U word i of
// this lane's row at stg_a + i * 128, R word j at stg_a + (E8_NW + j) * 128.  Absent words are stored as zero.
template <int KW>
__device__ __forceinline__ void gv_load_hdr_dense(const uint8_t* sgp, int lane, bool dense, uint32_t stg_a, uint32_t& ul, uint32_t& nrm) {
    ul = __ldg((const uint16_t*)sgp + lane);
    nrm = __ldg((const uint16_t*)sgp + 32 + lane);
    if (dense) {
        const uint32_t* ua = (const uint32_t*)(sgp + 128) + KW * 32 + lane;
#pragma unroll
        for (int i = 0; i < E8_DENSE; ++i) cp_async4(stg_a + i * 128, ua + i * 32);
    }
}
template <int KW>
__device__ __forceinline__ void gv_load_r(const uint8_t* sgp, int lane, uint32_t stg_a) {
    const uint32_t* rarea = (const uint32_t*)(sgp + 128);
#pragma unroll
    for (int j = 0; j < KW; ++j) cp_async4(stg_a + (E8_NW + j) * 128, rarea + j * 32 + lane);
}
// U words a row may or may not have (word i of the rows that have it are compacted, FORMAT §5): words [FIRST, E8_NW),
// `base` = words of the word-rows below FIRST.  No branch: an absent word is a zero-fill copy.
template <int FIRST>
__device__ __forceinline__ void gv_load_ragged_from(const uint32_t* uarea, uint32_t base, uint32_t stg_a, uint32_t nw) {
    const uint32_t lt = lanemask_lt();
#pragma unroll
    for (int i = FIRST; i < E8_NW; ++i) {
        const bool has = nw > (uint32_t)i;
        const uint32_t mk = __ballot_sync(0xffffffffu, has);
        cp_async4_zfill(stg_a + i * 128, uarea + base + __popc(mk & lt), has);
        base += __popc(mk);
    }
}
// a sub-group whose rows are not known to hold E8_DENSE words each (a row block's ragged edge, a low-rate stream): rare,
// kept out of the tile loop's instruction footprint
__device__ __noinline__ void gv_load_ragged_all(const uint32_t* uarea, uint32_t stg_a, uint32_t nw) {
    gv_load_ragged_from<0>(uarea, 0u, stg_a, nw);
}
template <int KW>
__device__ __forceinline__ void gv_load_ragged(const uint8_t* sgp, bool dense, uint32_t stg_a, uint32_t ul) {
    const uint32_t* uarea = (const uint32_t*)(sgp + 128) + KW * 32;
    const uint32_t nw = (ul + 31) >> 5;
    if (dense) gv_load_ragged_from<E8_DENSE>(uarea, E8_DENSE * 32, stg_a, nw);
    else gv_load_ragged_all(uarea, stg_a, nw);
}

// The folds of a decoder layer into the activation prologue (FORMAT R8 / R9; "the butterfly folds into the
// preceding LayerNorm"): the element the RHT sees is bf16((h r) g) or bf16(silu_c(a) b) instead of x itself.
struct GvFold {
    int mode;                      // 0 plain, 1 RMSNorm, 2 SiLU.mul
    float eps;
    const __nv_bfloat16* aux;      // gain (mode 1) or the second factor (mode 2)
    uint32_t ssq_a;                // shared memory: n_kt tile sums of squares (mode 1)
    int n_in;
};
__device__ __forceinline__ float gv_bf16r(float v) { return __bfloat162float(__float2bfloat16_rn(v)); }
__device__ __forceinline__ float gv_exp_c(float t) {   // FORMAT R9, every step one IEEE fp32 operation
    t = fminf(fmaxf(t, -87.0f), 88.0f);
    const float m = rintf(__fmul_rn(t, 0x1.715476p+0f));
    float f = __fmaf_rn(m, -0x1.62e000p-1f, t);
    f = __fmaf_rn(m, -0x1.0bfbe8p-15f, f);
    float p = 0x1.a01a02p-13f;
    p = __fmaf_rn(p, f, 0x1.6c16c2p-10f);
    p = __fmaf_rn(p, f, 0x1.111112p-7f);
    p = __fmaf_rn(p, f, 0x1.555556p-5f);
    p = __fmaf_rn(p, f, 0x1.555556p-3f);
    p = __fmaf_rn(p, f, 0.5f);
    p = __fmaf_rn(p, f, 1.0f);
    p = __fmaf_rn(p, f, 1.0f);
    return __fmul_rn(p, __int_as_float(((int)m + 127) << 23));
}
__device__ __forceinline__ float gv_silu_c(float a) { return __fdiv_rn(a, __fadd_rn(1.0f, gv_exp_c(-a))); }
__device__ __forceinline__ void gv_unpack_bf16x4(uint2 v, float* x) {
    x[0] = __uint_as_float(v.x << 16); x[1] = __uint_as_float(v.x & 0xffff0000u);
    x[2] = __uint_as_float(v.y << 16); x[3] = __uint_as_float(v.y & 0xffff0000u);
}
// R8: r = 1 / sqrt(treesum(h^2) / n + eps).  R2's tree over the whole vector = the tree inside each tile of 128 (two
// in-lane levels, five shuffle levels) followed by the tree over the tile sums (lane l holds tiles 4l .. 4l+3, absent
// ones zero).  Every warp of the CTA takes part (block barrier inside); the tile sums are shared through ssq_a.
template <int NW>
__device__ __forceinline__ float gv_rms_scale(const void* xp, const GvFold& fo, int n_kt, int wid, int lane) {
    for (int kt = wid; kt < n_kt; kt += NW) {
        float a[4];
        gv_unpack_bf16x4(__ldg((const uint2*)((const __nv_bfloat16*)xp + (int64_t)kt * 128 + 4 * lane)), a);
        float s = __fadd_rn(__fadd_rn(__fmul_rn(a[0], a[0]), __fmul_rn(a[1], a[1])), __fadd_rn(__fmul_rn(a[2], a[2]), __fmul_rn(a[3], a[3])));
#pragma unroll
        for (int m = 1; m < 32; m <<= 1) s = __fadd_rn(s, __shfl_xor_sync(0xffffffffu, s, m));
        if (lane == 0) asm volatile("st.shared.f32 [%0], %1;" ::"r"(fo.ssq_a + kt * 4), "f"(s) : "memory");
    }
    __syncthreads();
    float v[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) v[e] = 4 * lane + e < n_kt ? lds_f32(fo.ssq_a + (4 * lane + e) * 4) : 0.0f;
    float s = __fadd_rn(__fadd_rn(v[0], v[1]), __fadd_rn(v[2], v[3]));
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) s = __fadd_rn(s, __shfl_xor_sync(0xffffffffu, s, m));
    const float ms = __fdiv_rn(s, (float)fo.n_in);
    return __fdiv_rn(1.0f, __fsqrt_rn(__fadd_rn(ms, fo.eps)));
}

__device__ __forceinline__ void gv_load_x(const void* xp, int dtype, bool vec, const int8_t* dsign, int kt, int lane, float* x, uint32_t& sg) {
    const int64_t base = (int64_t)kt * 128 + 4 * lane;
    if (vec && dtype == HQ_BF16) {
        const uint2 v = __ldg((const uint2*)((const __nv_bfloat16*)xp + base));
        x[0] = __uint_as_float(v.x << 16); x[1] = __uint_as_float(v.x & 0xffff0000u);
        x[2] = __uint_as_float(v.y << 16); x[3] = __uint_as_float(v.y & 0xffff0000u);
    } else if (vec) {
        const float4 v = __ldg((const float4*)((const float*)xp + base));
        x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j)
            x[j] = dtype == HQ_BF16 ? __bfloat162float(((const __nv_bfloat16*)xp)[base + j]) : ((const float*)xp)[base + j];
    }
    sg = __ldg((const uint32_t*)(dsign + kt * 128) + lane);
}

// The start of a CTA, one call per warp (noinline: none of its registers count against the tile loop):
//  * the loads of the warp's first tile, a chain of three dependent global reads (sub-group offset -> header -> ragged U
//    words), interleaved with
//  * A1-A2: the activation tiles the CTA's tile range touches - K-tiles kt0 + j (mod n_kt), j < nt, one warp per tile -
//    through the RHT and the INT8 cast (FORMAT R1, R7) into the shared operand (row kt of a K-major SWIZZLE_128B tile =
//    the INT8 codes of K-tile kt, K order of e8_kcol) and s_x[kt]; the FWHT runs while the weight loads are in flight.
// x belongs to the stream order (griddepcontrol.wait comes before its first load); the weights do not.
// Ends with a block barrier.  Leaves ulen, norm bits and the next tile's offset of the warp's first tile at ret_a.
template <int K, int NW>
__device__ __noinline__ void gv_first_prologue(const void* xp, int dtype, const int8_t* dsign, int n_kt, uint32_t xq_a,
                                               uint32_t sx_a, int wid, int lane, int kt0, int nt, const uint8_t* blob,
                                               const uint32_t* soff, int has, int dense_i, uint32_t stg_a, uint32_t ret_a,
                                               GvFold fo) {
    constexpr int KW = 4 * K;
    const bool dense = dense_i != 0;
    uint32_t off0 = 0, off1 = 0;
    if (has) {
        off0 = __ldg(soff);
        if (has > 1) off1 = __ldg(soff + 4);
    }
    // The weights do not belong to the stream order (they are never written at inference time): the whole dependent chain
    // of the first tile - offset -> header -> ragged words - is issued BEFORE griddepcontrol.wait, i.e. while the CTAs of
    // the previous launch that are still running finish (a CTA of this kernel starts as soon as ITS SM is free).
    uint32_t ul = 0, nrm = 0;
    const uint8_t* sgp = blob + 16 * (size_t)off0;
    if (has) {
        gv_load_hdr_dense<KW>(sgp, lane, dense, stg_a, ul, nrm);
        gv_load_r<KW>(sgp, lane, stg_a);
        gv_load_ragged<KW>(sgp, dense, stg_a, ul);
    }
    bool ragged_due = false;
    griddep_wait();
    const bool vec = dtype == HQ_BF16 ? (((uintptr_t)xp) & 7) == 0 : (((uintptr_t)xp) & 15) == 0;
    const int col0 = act_col0(lane);
    float x[4], xn[4];
    uint32_t sg = 0, sgn = 0;
    auto tile_of = [&](int j) { const int kt = kt0 + j; return kt >= n_kt ? kt - n_kt : kt; };
    int j = wid;
    uint2 auxn = make_uint2(0u, 0u);
    auto load_aux = [&](int kt) { if (fo.mode) auxn = __ldg((const uint2*)(fo.aux + (int64_t)kt * 128 + 4 * lane)); };
    if (j < nt) { gv_load_x(xp, dtype, vec, dsign, tile_of(j), lane, xn, sgn); load_aux(tile_of(j)); }
    // R8: the scale of the whole vector, behind the first tile's loads (one more block barrier; mode is CTA-uniform)
    const float rms_r = fo.mode == 1 ? gv_rms_scale<NW>(xp, fo, n_kt, wid, lane) : 1.0f;
#pragma unroll 1
    for (; j < nt; j += NW) {
        const int kt = tile_of(j);
        if (fo.mode) {   // the bf16 vector a separate RMSNorm / SiLU.mul kernel would have written, element by element
            float ax[4];
            gv_unpack_bf16x4(auxn, ax);
#pragma unroll
            for (int e = 0; e < 4; ++e)
                xn[e] = gv_bf16r(fo.mode == 1 ? __fmul_rn(__fmul_rn(xn[e], rms_r), ax[e]) : __fmul_rn(gv_silu_c(xn[e]), ax[e]));
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) x[e] = (sgn >> (8 * e)) & 0x80u ? -xn[e] : xn[e];
        if (j + NW < nt) { gv_load_x(xp, dtype, vec, dsign, tile_of(j + NW), lane, xn, sgn); load_aux(tile_of(j + NW)); }
        int qv[4];
        const float sx = warp_act_tile128(x, lane, qv);
        if (ragged_due) {   // the header has arrived behind the FWHT
            gv_load_ragged<KW>(sgp, dense, stg_a, ul);
            ragged_due = false;
        }
        const uint32_t row_a = xq_a + (uint32_t)((kt >> 3) * 1024 + (kt & 7) * 128);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int col = col0 + 4 * e;
            sts8(row_a + ((((col >> 4) ^ (kt & 7)) << 4) | (col & 15)), (uint32_t)(uint8_t)(int8_t)qv[e]);
        }
        if (lane == 0) asm volatile("st.shared.f32 [%0], %1;" ::"r"(sx_a + kt * 4), "f"(sx) : "memory");
    }
    if (ragged_due) gv_load_ragged<KW>(sgp, dense, stg_a, ul);
    sts32(ret_a, ul); sts32(ret_a + 4, nrm); sts32(ret_a + 8, off1); sts32(ret_a + 12, off0);
    fence_proxy_async_smem();   // the operand is read by the tensor core (async proxy)
    __syncthreads();
}

// K = Rice parameter, NWG = warp groups of 4 warps per CTA (one CTA per SM).  Batch 1 only (p.B == 1, p.n_bt == 1).
//
// Work: the tiles (row block, K-tile) of all stacked weights in row-block-major order form one flat range of T tiles;
// warp group g of the G on the device owns the contiguous sub-range [g T / G, (g+1) T / G) - balanced to one tile - i.e. a
// few runs of K-tiles inside one, two or three row blocks ("segments").  Inside a segment only the K-tile index moves:
// every pointer is loop invariant.  A row block whose K range is cut by range boundaries gets one partial sum per
// segment (slot = g - g_first(row block), or the K-tile index when there are fewer tiles than warp groups); the last segment
// to arrive adds them in slot order (deterministic).
template <int K, int NWG>
__global__ void __launch_bounds__(NWG * 128, 1)
k_gemv_e8(E8Params p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    constexpr int KW = 4 * K;   // R words per row
    constexpr int NW = NWG * 4;
    // the warp index through a shuffle: the compiler then knows it is warp-uniform (descriptors stay in uniform registers)
    const int wid = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int tid = threadIdx.x, wg = wid >> 2, warp = wid & 3, lane = tid & 31, t = warp * 32 + lane;
    const uint32_t smem_a = smem_u32(smem);
    const uint32_t xq_a = smem_a + E8_LUT_BYTES;                                  // activation operand, 1024-aligned
    const uint32_t XQB = gv_xq_bytes(p.n_kt);
    const uint32_t sx_a = xq_a + XQB;                                             // s_x[n_kt]
    const uint32_t SXB = (uint32_t)((p.n_kt * 4 + 127) & ~127);
    const uint32_t scr_a = sx_a + SXB + (uint32_t)tid * E8_SCR_STRIDE * 4;        // this row's nibble words
    const uint32_t mask_a = sx_a + SXB + (uint32_t)(NWG * 128 * E8_SCR_STRIDE * 4) + (uint32_t)tid * 16;   // flagged tiles of the segment
    // staging of the next tile's bitstream words: word j of this warp's rows at stg_a + j * 128 (lane-interleaved: no conflicts)
    const uint32_t stg_a = sx_a + SXB + (uint32_t)(NWG * 128 * (E8_SCR_STRIDE * 4 + 16)) + (uint32_t)wid * (GV_STAGE_WORDS * 128) + (uint32_t)lane * 4;
    uint64_t* bars = (uint64_t*)(smem + E8_LUT_BYTES + XQB + SXB + (size_t)NWG * 128 * (E8_SCR_STRIDE * 4 + 16 + GV_STAGE_WORDS * 4));
    uint64_t* bar_w = bars + wid;            // this warp's MMAs done
    uint64_t* bar_lut = bars + NW;
    uint32_t* tmem_slot = (uint32_t*)(bars + NW + 1);
    const GvFold fold{p.fold_mode, p.fold_eps, p.fold_aux, smem_u32(bars + NW + 3), p.n_kt * 128};

    if (wid == 0) tmem_alloc(tmem_slot, 512);
    if (tid == 0) {
        for (int i = 0; i < NW; ++i) mbar_init(&bars[i], 1);
        mbar_init(bar_lut, 1);
        mbar_fence_init();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    griddep_launch();
    if (tid == 0) {  // the phase-1 table arrives by one TMA bulk copy while the first loads are in flight
        mbar_arrive_expect_tx(bar_lut, E8_LUT_BYTES);
        bulk_g2s(smem, p.lut, E8_LUT_BYTES, bar_lut);
    }
    const uint32_t tmem_wg = *tmem_slot + (uint32_t)wg * GV_TCOLS_WG;
    const uint32_t ta = tmem_wg;                                   // A tile: columns 0..31 (lane 0 for the MMA)
    const uint32_t td = tmem_wg + 32;                              // accumulator: 16 columns
    const uint32_t lane_sel = (uint32_t)(warp * 32) << 16;         // this warp's TMEM lane quarter (ld / st)
    const uint32_t idesc = make_idesc_i8(128, 16);
    const uint32_t dm0 = warp == 0 ? 0u : 0xffffffffu, dm1 = warp == 1 ? 0u : 0xffffffffu,
                   dm2 = warp == 2 ? 0u : 0xffffffffu, dm3 = warp == 3 ? 0u : 0xffffffffu;   // lanes this warp does NOT write
    const uint32_t lut_lane = smem_a + (uint32_t)(lane & (E8_LUT_COPIES - 1)) * 4;
    const int n_kt = p.n_kt;

    // ---- this warp group's flat tile range
    const int gwg = blockIdx.x * NWG + wg, GWG = gridDim.x * NWG;
    const int64_t T = p.n_items;   // row blocks of all weights x n_kt
    const int f_begin = (int)(((int64_t)gwg * T) / GWG), f_end = (int)(((int64_t)(gwg + 1) * T) / GWG);
    int f = f_begin;
    auto wg_of_tile = [&](int64_t ft) -> int { return (int)(((ft + 1) * GWG - 1) / T); };   // the warp group whose range holds tile ft

    // the K-tiles this CTA's tile range touches: kt0 + j (mod n_kt), j < nt_cta - the only activation tiles it quantizes
    const int64_t cta_b = ((int64_t)blockIdx.x * NWG * T) / GWG, cta_e = ((int64_t)(blockIdx.x + 1) * NWG * T) / GWG;
    const int nt_cta = (int)min((int64_t)n_kt, cta_e - cta_b), kt0_cta = (int)(cta_b % n_kt);

    if (f >= f_end) {   // nothing to do for this warp group: it still helps with the activations and joins the barriers
        gv_first_prologue<K, NW>(p.x, p.dtype, p.dsign, n_kt, xq_a, sx_a, wid, lane, kt0_cta, nt_cta, nullptr, nullptr, 0, 0, stg_a, scr_a, fold);
        tc_fence_before();
        __syncthreads();
        if (wid == 0) tmem_dealloc(*tmem_slot, 512);
        return;
    }
    asm volatile("st.shared.v4.u32 [%0], {%1,%1,%1,%1};" ::"r"(mask_a), "r"(0u) : "memory");
    bool first_seg = true;
    uint32_t n_mma = 0;    // commits of this warp so far: the barrier's phase
    float yacc = 0.0f;

    while (f < f_end) {
        // ---- segment: K-tiles [ka, kb) of global row block rbg
        const int rbg = f / n_kt, ka = f - rbg * n_kt;
        const int kb = min(n_kt, ka + (f_end - f));
        f += kb - ka;
        int w = 0;
#pragma unroll
        for (int i = 1; i < E8_MAXW; ++i)
            if (i < p.n_w && rbg >= p.rb_base[i]) w = i;
        const int rbl = rbg - p.rb_base[w];
        const int64_t mw = p.m[w];
        const int64_t r = (int64_t)rbl * 128 + t;
        const bool row_in = r < mw;
        const bool dense = ((int64_t)rbl * 128 + warp * 32 + 32 <= mw) && p.u_dense >= E8_DENSE;   // warp-uniform
        const uint8_t* blob = p.blob[w];
        const uint32_t* soff = p.sub_off[w] + (((size_t)rbl * n_kt + ka) * 4 + warp);   // this warp's sub-group of tile ka; +4 per tile
        const float inv_A = p.inv_A[w];

        auto load_hdr_dense = [&](const uint8_t* sgp, uint32_t& ul, uint32_t& nrm) { gv_load_hdr_dense<KW>(sgp, lane, dense, stg_a, ul, nrm); };
        auto load_r = [&](const uint8_t* sgp) { gv_load_r<KW>(sgp, lane, stg_a); };
        auto load_ragged = [&](const uint8_t* sgp, uint32_t ul) { gv_load_ragged<KW>(sgp, dense, stg_a, ul); };
        // epilogue of K-tile kt (this warp's MMAs on it have completed): drain the accumulator lane, rescale, accumulate (A7)
        auto epilogue = [&](int kt, float sw, bool ovr) {
            uint32_t v;
            tmem_ld1(td + lane_sel + ((uint32_t)kt & 7u), v);
            tmem_ld_wait();
            if (ovr) v = 0u;   // this tile of the row is redone by gv_segment_fallback
            if (p.acc_i32 && row_in) p.acc_i32[(int64_t)kt * mw + r] = (int)v;
            yacc += (sw * lds_f32(sx_a + kt * 4)) * (float)(int)v;
            tc_fence_before();
        };

        uint32_t ul_c, nrm_c, ul_n = 0, nrm_n = 0;
        // segment prologue: offsets of its first two tiles, then everything of the first tile
        uint32_t off_n1;
        const uint8_t* sgp_c;
        if (first_seg) {   // the kernel's first tile: its loads are interleaved with the activation prologue (all warps meet there)
            gv_first_prologue<K, NW>(p.x, p.dtype, p.dsign, n_kt, xq_a, sx_a, wid, lane, kt0_cta, nt_cta, blob, soff,
                                     (ka + 1 < kb) ? 2 : 1, dense ? 1 : 0, stg_a, scr_a, fold);
            first_seg = false;
            ul_c = lds32(scr_a); nrm_c = lds32(scr_a + 4); off_n1 = lds32(scr_a + 8);
            sgp_c = blob + 16 * (size_t)lds32(scr_a + 12);
            mbar_wait(bar_lut, 0u);
        } else {
            off_n1 = (ka + 1 < kb) ? __ldg(soff + 4) : 0u;
            sgp_c = blob + 16 * (size_t)__ldg(soff);
            load_hdr_dense(sgp_c, ul_c, nrm_c);
            load_r(sgp_c);
            load_ragged(sgp_c, ul_c);
        }
        float sw_prev = 0.0f;
        bool ovr_prev = false, seg_flagged = false;

        for (int kt = ka; kt < kb; ++kt) {
            const bool has1 = kt + 1 < kb, has2 = kt + 2 < kb;
            const uint32_t off_n2 = has2 ? __ldg(soff + (kt + 2 - ka) * 4) : 0u;
            // ---- phase 1: unary section -> nibble words (A4)
            const uint32_t nw = (ul_c + 31) >> 5;
            const uint32_t maxul = __reduce_max_sync(0xffffffffu, ul_c);   // longest U-section of the sub-group, bits
            const uint32_t maxnw = (maxul + 31) >> 5;
            cp_async_wait_all();   // this lane's words of the tile have landed (each lane reads only what it copied)
            {
                uint32_t Uw[E8_NW];
#pragma unroll
                for (int i = 0; i < E8_NW; ++i) Uw[i] = lds32(stg_a + i * 128);
                uint32_t T = 0, acc = 0, wo = scr_a;
#pragma unroll
                for (int i = 0; i < E8_NW; ++i) {   // an absent word is zero: no terminators, nothing appended
                    if (i < E8_DENSE) {
                        e8_unary_word(Uw[i], lut_lane, T, acc, wo);
                    } else if ((uint32_t)i < maxnw) {   // tail words: only the bytes some row of the warp still uses
                        const int nb = (int)min(4u, (maxul - 32u * (uint32_t)i + 7u) >> 3);
                        e8_unary_word(Uw[i], lut_lane, T, acc, wo, nb);
                    }
                }
            }
            // the U registers are free: header and dense U words of the next tile (its offset arrived an iteration ago)
            const uint8_t* sgp_n = blob + 16 * (size_t)off_n1;
            if (has1) load_hdr_dense(sgp_n, ul_n, nrm_n);

            // ---- this warp's MMAs of the previous tile: issued a whole phase 1 ago, so this wait rarely spins
            if (kt > ka) {
                mbar_wait(bar_w, (n_mma - 1) & 1u);
                tc_fence_after();
                epilogue(kt - 1, sw_prev, ovr_prev);
            }
            // ---- phase 2: nibble words + remainders -> INT8 points, registers -> this row's TMEM lane (A5)
            const bool present = row_in && ul_c > 0;
            uint32_t total = 0;
            {
                uint32_t Rw[KW > 0 ? KW : 1];
#pragma unroll
                for (int j = 0; j < KW; ++j) Rw[j] = lds32(stg_a + (E8_NW + j) * 128);
                uint32_t prevWo = 15u << 24;  // e_{-1} = -1 mod 16
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    uint32_t W[4], C[8];
#pragma unroll
                    for (int i = 0; i < 4; ++i) W[i] = lds32(scr_a + (c * 4 + i) * 4);
                    e8_run<K>(W, Rw + c * K, prevWo, total, C);
                    if (!present) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) C[i] = 0u;
                    }
                    tmem_st8(ta + lane_sel + 8 * c, C);   // K index 32c + 4i + b = column 8c + i, byte b
                }
            }
            const bool need_generic = present && (nw > (uint32_t)E8_NW || total + 128u != ul_c);
            if (need_generic) {   // a quotient >= 16 or a long row: marked, redone after the segment's loop (rare)
                const uint32_t ma = mask_a + (uint32_t)(((kt - ka) >> 5) * 4);
                sts32(ma, lds32(ma) | (1u << ((kt - ka) & 31)));
                seg_flagged = true;
            }
            // the R registers are free: remainder words of the next tile, and its ragged U words (the header has arrived)
            if (has1) { load_r(sgp_n); load_ragged(sgp_n, ul_n); }
            const float sw_cur = f16_bits_to_f32((uint16_t)nrm_c) * inv_A;
            // ---- A6: this warp's rows are in tensor memory; one lane issues the tile's four MMAs with the other warps'
            // output lanes masked off, and commits them to the warp's barrier
            tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                tc_fence_after();
                const uint32_t b0s = xq_a + (uint32_t)(kt >> 3) * 1024u;
#pragma unroll
                for (int ks = 0; ks < 4; ++ks)
                    mma_i8_ts_masked(td, ta + 8 * ks, make_desc_sw128(b0s + ks * 32), idesc, dm0, dm1, dm2, dm3, ks > 0);
                mma_commit(bar_w);
            }
            __syncwarp();
            ++n_mma;
            // ---- rotate
            sw_prev = sw_cur; ovr_prev = need_generic;
            sgp_c = sgp_n; ul_c = ul_n; nrm_c = nrm_n;
            // pull the sub-group of tile kt+2 into L2 (no registers held): its demand loads are issued an iteration from now
            if (has2 && lane < 18) asm volatile("prefetch.global.L2 [%0];" ::"l"(blob + 16 * (size_t)off_n2 + lane * 128));
            off_n1 = off_n2;
        }
        // drain: the last tile's epilogue; then the segment's sum is y (the segment covers the row block's whole K range)
        // or a partial sum in this segment's slot
        mbar_wait(bar_w, (n_mma - 1) & 1u);
        tc_fence_after();
        epilogue(kb - 1, sw_prev, ovr_prev);
        if (__any_sync(0xffffffffu, seg_flagged)) {
            if (seg_flagged)
                yacc += gv_segment_fallback<K>(blob, soff, lane, ka, mask_a, xq_a, sx_a, inv_A, p.acc_i32 ? p.acc_i32 + r : nullptr, mw);
            __syncwarp();
        }
        if (row_in) {
            if (ka == 0 && kb == n_kt) {
                if (p.res[w]) yacc = __fadd_rn(yacc, __bfloat162float(p.res[w][r]));   // R10
                if (p.y_bf16[w]) p.y_bf16[w][r] = __float2bfloat16_rn(yacc);
                if (p.y_f32[w]) p.y_f32[w][r] = yacc;
            } else {
                p.partials[w][(int64_t)(T < GWG ? ka : gwg - wg_of_tile((int64_t)rbg * n_kt)) * mw + r] = yacc;
            }
        }
        yacc = 0.0f;
    }
    // ---- split-K reduction inside the kernel: publish this thread's partial sums (one fence), then arrive once per cut
    // row block of the range on a per-(row block, warp) counter; the LAST of the row block's segments to arrive adds the
    // partials in slot order - deterministic - and writes y (A7).  No block barrier, no extra launch.
    // Ordering: the lanes' partial sums -> __syncwarp -> lane 0's acq_rel atomic (release: cumulative over what the barrier
    // ordered before it; acquire: the other segments' partials) -> __syncwarp -> the lanes' L2 loads.  One atomic round trip
    // instead of fence + atomic + fence.
    __syncwarp();
    for (int ff = f_begin; ff < f_end;) {
        const int rbg = ff / n_kt, ka = ff - rbg * n_kt;
        const int kb = min(n_kt, ka + (f_end - ff));
        ff += kb - ka;
        if (ka == 0 && kb == n_kt) continue;   // written directly
        // fewer tiles than warp groups: every tile is a segment of its own (slot = K-tile index)
        const int n_seg = T < GWG ? n_kt : wg_of_tile((int64_t)rbg * n_kt + n_kt - 1) - wg_of_tile((int64_t)rbg * n_kt) + 1;
        int w = 0;
#pragma unroll
        for (int i = 1; i < E8_MAXW; ++i)
            if (i < p.n_w && rbg >= p.rb_base[i]) w = i;
        unsigned int last = 0;
        if (lane == 0) {
            unsigned int* cnt = p.counters + ((size_t)rbg * 4 + warp);
            unsigned int prev;
            asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], %2;" : "=r"(prev) : "l"(cnt), "r"(1u) : "memory");
            last = prev == (unsigned int)(n_seg - 1);
            if (last) *cnt = 0u;
        }
        last = __shfl_sync(0xffffffffu, last, 0);
        if (!last) continue;
        __syncwarp();
        const int64_t mw = p.m[w];
        const int64_t r = (int64_t)(rbg - p.rb_base[w]) * 128 + t;
        if (r >= mw) continue;
        const float* part = p.partials[w];
        float sum = 0.0f;
        for (int sp0 = 0; sp0 < n_seg; sp0 += 8) {   // slot order
            float v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = (sp0 + u < n_seg) ? __ldcg(part + r + (int64_t)(sp0 + u) * mw) : 0.0f;
#pragma unroll
            for (int u = 0; u < 8; ++u) sum += v[u];
        }
        if (p.res[w]) sum = __fadd_rn(sum, __bfloat162float(p.res[w][r]));   // R10
        if (p.y_bf16[w]) p.y_bf16[w][r] = __float2bfloat16_rn(sum);
        if (p.y_f32[w]) p.y_f32[w][r] = sum;
    }
    tc_fence_before();
    __syncthreads();
    if (wid == 0) tmem_dealloc(*tmem_slot, 512);
}

}  // namespace hq
