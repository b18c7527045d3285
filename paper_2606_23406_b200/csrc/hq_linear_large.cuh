// hq_linear_large.cuh — the large-M path of hq_linear for E8 tiles of 128 (north_star (e); BASELINE config 5).
//
// At thousands of activation rows the Rice decode must not be repeated per batch tile: the weights are decoded ONCE per
// call into a scratch copy that already has the tensor-core operand layout, and a warp-specialised GEMM streams it.
//   k_e8_decode_ablob : sub-group (FORMAT §5) -> 128 x 128 INT8 tile, K-major SWIZZLE_128B, K permuted by e8_kcol, followed
//                       by the 128 row scales rho / (alpha sqrt n) (§4.8).  Same two-phase SWAR decoder as the fused
//                       kernel (hq_e8_decode.cuh), same fallback.
//   k_e8_gemm_large   : persistent CTA per SM, tile = 128 weight rows x 256 activation rows.  Warp 0 = TMA producer
//                       (1-D bulk copies of the A and B blobs into a 4-stage ring), warp 1 = MMA issuer
//                       (4 x tcgen05.mma kind::i8 M=128 N=256 K=32 per K-tile into one of two TMEM accumulators),
//                       warps 4..11 = epilogue: per K-tile the INT32 accumulator is drained (tcgen05.ld), scaled by
//                       rho_tile * s_x,tile (both scales are per tile of 128, so the INT32 sum cannot run across tiles:
//                       §4.8) and added to fp32 registers; y is written once per output tile.
// The epilogue (I2F + FMUL + FFMA per accumulator) is the co-bound of this path: DESIGN.md §6.3.
#pragma once
#include "hq_common.cuh"
#include "hq_e8_decode.cuh"
#include "hq_linear_e8.cuh"
#include "hq_tc.cuh"

namespace hq {

constexpr int LG_NB = 256;                                   // activation rows per tile = MMA N
constexpr uint32_t LG_ABLOB = 16384u + 512u;                 // INT8 tile + 128 fp32 row scales
constexpr uint32_t LG_BBLOB = LG_NB * 128u + LG_NB * 4u;     // = e8_bblob_bytes(256)
constexpr uint32_t LG_STAGE = LG_NB * 128u + 16384u;          // operand bytes of one K-chunk of 128: B tile 32 KB + A tile 16 KB
constexpr int LG_NST = 4;
// The scales of an RHT tile (256 s_x + 128 row scales) travel in a ring of their own: an operand stage is released by the
// MMA's commit alone, not held while the epilogue drains the tile (that throttled the TMA pipeline to a third).
constexpr uint32_t LG_SCSLOT = LG_NB * 4u + 512u;
constexpr int LG_NSC = 8;
constexpr size_t LG_SMEM = 1024 + (size_t)LG_NST * LG_STAGE + (size_t)LG_NSC * LG_SCSLOT + 8 * (2 * LG_NST + 2 * LG_NSC + 4) + 16;

struct E8AblobParams {
    const uint8_t* blob;
    const uint32_t* sub_off;
    const uint32_t* lut;
    uint8_t* ablob;       // [n_rb][n_kt][LG_ABLOB]
    int64_t m;
    int n_kt, n_rb;
    float inv_A;
};

// TILE = RHT tile of the weight (128 or 256).  A tile of 256 is written as two operand chunks of 128 K-bytes (K index
// inside the tile: 32c + 4i + b for block 4c + b, coordinate i; chunk = c / 4), each followed by the same 128 row scales.
// FP8: the decoded integer coordinates are written as E4M3 bytes (FORMAT R12; §4.8) for the f8f6f4 GEMM.
template <int K, int TILE, bool FP8 = false>
__global__ void __launch_bounds__(256) k_e8_decode_ablob(E8AblobParams p) {   // two tiles per CTA pass: warps 0-3 and 4-7
    extern __shared__ __align__(16) uint8_t smem_raw[];
    constexpr int KW = K * TILE / 32;              // R words per row
    constexpr int NWT = E8_NW * TILE / 128;        // U words per row handled by the fast path
    constexpr int NRUN = TILE / 32;                // runs of 32 symbols
    constexpr int SCR = TILE / 8 + 1;              // nibble words per row + 1
    constexpr int NCH = TILE / 128;                // operand chunks per tile
    const int t = threadIdx.x & 127, sub = threadIdx.x >> 7, warp = t >> 5, lane = t & 31;
    const uint32_t smem_a = smem_u32(smem_raw);
    // the phase-1 table arrives by one bulk copy; the CTA's first loads are in flight meanwhile
    uint64_t* bar_lut = (uint64_t*)(smem_raw + E8_LUT_BYTES + 256 * SCR * 4);
    if (threadIdx.x == 0) {
        mbar_init(bar_lut, 1);
        mbar_fence_init();
        mbar_arrive_expect_tx(bar_lut, E8_LUT_BYTES);
        bulk_g2s(smem_raw, p.lut, E8_LUT_BYTES, bar_lut);
    }
    __syncthreads();
    const uint32_t lut_lane = smem_a + (uint32_t)(lane & (E8_LUT_COPIES - 1)) * 4;
    const uint32_t scr_a = smem_a + E8_LUT_BYTES + (uint32_t)threadIdx.x * SCR * 4;
    const uint32_t lane_lt = (1u << lane) - 1u;
    // contiguous range of (row block, tile) pairs per CTA: a few CTAs per SM, each amortising its table over many tiles
    const int64_t G = (int64_t)p.n_rb * p.n_kt;
    const int64_t g_begin = (int64_t)blockIdx.x * G / gridDim.x, g_end = (int64_t)(blockIdx.x + 1) * G / gridDim.x;
    uint32_t off_c = g_begin + sub < g_end ? __ldg(p.sub_off + (g_begin + sub) * 4 + warp) : 0u;
    bool lut_ready = false;
    for (int64_t g = g_begin + sub; g < g_end; g += 2) {
        const int rb = (int)(g / p.n_kt);
        const int64_t r = (int64_t)rb * 128 + t;
        const uint8_t* sgp = p.blob + 16 * (size_t)off_c;
        const uint32_t off_n = g + 2 < g_end ? __ldg(p.sub_off + (g + 2) * 4 + warp) : 0u;
        const uint32_t ul = __ldg((const uint16_t*)sgp + lane), nrm = __ldg((const uint16_t*)sgp + 32 + lane);
        const uint32_t* rarea = (const uint32_t*)(sgp + 128);
        const uint32_t* uarea = rarea + KW * 32;
        uint32_t Rw[KW > 0 ? KW : 1], Uw[NWT];
#pragma unroll
        for (int j = 0; j < KW; ++j) Rw[j] = __ldg(rarea + j * 32 + lane);
        const uint32_t nw = (ul + 31) >> 5;
        {
            uint32_t base = 0;
#pragma unroll
            for (int w = 0; w < NWT; ++w) {
                const bool has = nw > (uint32_t)w;
                const uint32_t mk = __ballot_sync(0xffffffffu, has);
                Uw[w] = has ? __ldg(uarea + base + __popc(mk & lane_lt)) : 0u;
                base += __popc(mk);
            }
        }
        // the next tile's sub-group into L2 while this one is decoded (its demand loads then hit)
        if (g + 2 < g_end && lane < (TILE == 128 ? 18 : 34))
            asm volatile("prefetch.global.L2 [%0];" ::"l"(p.blob + 16 * (size_t)off_n + lane * 128));
        if (!lut_ready) { mbar_wait(bar_lut, 0u); lut_ready = true; }
        {
            uint32_t T = 0, acc = 0, wo = scr_a;
#pragma unroll
            for (int w = 0; w < NWT; ++w) e8_unary_word(Uw[w], lut_lane, T, acc, wo);
        }
        uint8_t* tile = p.ablob + g * (size_t)(NCH * LG_ABLOB);
        const bool present = r < p.m && ul > 0;
        uint32_t total = 0, prevWo = 15u << 24;
#pragma unroll
        for (int c = 0; c < NRUN; ++c) {
            uint32_t W[4], C[8];
#pragma unroll
            for (int w = 0; w < 4; ++w) W[w] = lds32(scr_a + (c * 4 + w) * 4);
            e8_run<K>(W, Rw + c * K, prevWo, total, C);
            if (!present) {
#pragma unroll
                for (int i = 0; i < 8; ++i) C[i] = 0u;
            }
            if (FP8) {
#pragma unroll
                for (int i = 0; i < 8; ++i) C[i] = s8x4_to_e4m3x4(C[i]);
            }
            uint8_t* rowp = tile + (c >> 2) * LG_ABLOB + (t >> 3) * 1024 + (t & 7) * 128;
            *(uint4*)(rowp + (((2 * (c & 3)) ^ (t & 7)) << 4)) = make_uint4(C[0], C[1], C[2], C[3]);
            *(uint4*)(rowp + (((2 * (c & 3) + 1) ^ (t & 7)) << 4)) = make_uint4(C[4], C[5], C[6], C[7]);
        }
        if (present && (nw > (uint32_t)NWT || total + (uint32_t)TILE != ul)) {   // a quotient >= 16 or a long row: generic decoder
            SubGroup sg = sub_group(sgp, KW);
            WordsRowU uw{nullptr, sg.uarea, sg.ulen, nw, 0u, lane};
            WordsRowR rw{sg.rarea, lane, KW};
            decode_row_generic<LAT_E8>(rw, 0u, uw, 0u, TILE, K, K, [&](int bk, const int* c) {
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int col = e8_kcol(8 * (bk & 15) + e);
                    uint8_t* rowp = tile + (bk >> 4) * LG_ABLOB + (t >> 3) * 1024 + (t & 7) * 128;
                    rowp[(((col >> 4) ^ (t & 7)) << 4) | (col & 15)] =
                        FP8 ? (uint8_t)(s8x4_to_e4m3x4((uint32_t)(uint8_t)(int8_t)c[e]) & 0xffu) : (uint8_t)(int8_t)c[e];
                }
            });
        }
        const float sw = present ? f16_bits_to_f32((uint16_t)nrm) * p.inv_A : 0.0f;
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) ((float*)(tile + ch * LG_ABLOB + 16384))[t] = sw;
        off_c = off_n;
    }
}

// packed fp32 pairs (sm_100 f32x2 arithmetic): one instruction for two accumulators
__device__ __forceinline__ uint64_t pack_u32x2(uint32_t lo, uint32_t hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
    return r;
}
__device__ __forceinline__ uint64_t pack_f32x2(float lo, float hi) { return pack_u32x2(__float_as_uint(lo), __float_as_uint(hi)); }
__device__ __forceinline__ float f32x2_lo(uint64_t v) { return __uint_as_float((uint32_t)v); }
__device__ __forceinline__ float f32x2_hi(uint64_t v) { return __uint_as_float((uint32_t)(v >> 32)); }
__device__ __forceinline__ uint64_t mul_f32x2(uint64_t a, uint64_t b) {
    uint64_t r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ uint64_t fma_f32x2(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// Tile order of the persistent GEMM: panels of LG_PANEL row blocks, inside a panel batch-tile major.  The 148 tiles in
// flight then touch LG_PANEL weight row blocks and ~148 / LG_PANEL batch tiles (a few MB of operands each way) instead of
// every row block of the weight (the whole 69 MB scratch copy per wave in plain batch-tile-major order): the operand
// tiles are re-read from L2, not from DRAM.
constexpr int LG_PANEL = 16;
__device__ __forceinline__ void lg_tile_coords(int tile, int n_rb, int n_bt, int& bt, int& rb) {
    const int per_panel = LG_PANEL * n_bt;
    const int panel = tile / per_panel, rem = tile - panel * per_panel;
    const int rows = min(LG_PANEL, n_rb - panel * LG_PANEL);
    bt = rem / rows;
    rb = panel * LG_PANEL + (rem - bt * rows);
}

struct E8LargeParams {
    const uint8_t* ablob;   // [n_rb][n_kt][LG_ABLOB]
    const uint8_t* bblob;   // [n_bt][n_kt][LG_BBLOB]
    __nv_bfloat16* y_bf16;  // [B][ldy] or null
    float* y_f32;           // [B][m] or null
    int64_t ldy, m, B;
    int n_rb, n_bt, n_kt;
    int32_t* acc_i32;       // [n_kt][B][m] or null: parity / debug copy of every K-tile's INT32 accumulator
};

// NCH = operand chunks (TMA stages of 128 K-bytes) per RHT tile: 1 (tile 128) or 2 (tile 256).  The INT32 accumulator runs
// over the NCH chunks of a tile and is drained once per TILE: at tile 256 the rescale costs half as many issue slots per
// MAC (the tile is chosen on kernel grounds).  p.n_kt counts chunks.
// FP8: both operands hold E4M3 bytes, the MMA is kind::f8f6f4 with an fp32 accumulator (no int -> float in the drain).
template <int NCH, bool FP8 = false>
__global__ void __launch_bounds__(384, 1) k_e8_gemm_large(E8LargeParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    const uint32_t smem_a = smem_u32(smem);
    const uint32_t sc_a = smem_a + LG_NST * LG_STAGE;   // scale ring
    uint64_t* full = (uint64_t*)(smem + (size_t)LG_NST * LG_STAGE + (size_t)LG_NSC * LG_SCSLOT);
    uint64_t* empty = full + LG_NST;
    uint64_t* scf = empty + LG_NST;      // scales of a tile landed
    uint64_t* sce = scf + LG_NSC;        // scales of a tile read by the eight epilogue warps
    uint64_t* acc_full = sce + LG_NSC;
    uint64_t* acc_empty = acc_full + 2;
    uint32_t* tmem_slot = (uint32_t*)(acc_empty + 2);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    if (warp == 0) tmem_alloc(tmem_slot, 512);
    if (tid == 32) {
        for (int s = 0; s < LG_NST; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        for (int s = 0; s < LG_NSC; ++s) { mbar_init(&scf[s], 1); mbar_init(&sce[s], 8); }
        for (int a = 0; a < 2; ++a) { mbar_init(&acc_full[a], 1); mbar_init(&acc_empty[a], 8); }
        mbar_fence_init();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int n_tiles = p.n_rb * p.n_bt;

    if (warp < 4) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (tid == 0) {   // ---- TMA producer
            uint32_t it = 0;
            for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
                int bt, rb;
                lg_tile_coords(tile, p.n_rb, p.n_bt, bt, rb);
                const uint8_t* ag = p.ablob + (size_t)rb * p.n_kt * LG_ABLOB;
                const uint8_t* bg = p.bblob + (size_t)bt * p.n_kt * LG_BBLOB;
                for (int kt = 0; kt < p.n_kt; ++kt, ++it) {
                    const uint32_t s = it % LG_NST, ph = (it / LG_NST) & 1u;
                    mbar_wait(&empty[s], ph ^ 1u);
                    mbar_arrive_expect_tx(&full[s], LG_STAGE);
                    uint8_t* st = smem + (size_t)s * LG_STAGE;
                    bulk_g2s(st, bg + (size_t)kt * LG_BBLOB, LG_NB * 128u, &full[s]);
                    bulk_g2s(st + LG_NB * 128u, ag + (size_t)kt * LG_ABLOB, 16384u, &full[s]);
                    if (it % NCH == NCH - 1) {   // last chunk of an RHT tile: its scales into the scale ring
                        const uint32_t tl = it / NCH, q = tl % LG_NSC;
                        mbar_wait(&sce[q], ((tl / LG_NSC) & 1u) ^ 1u);
                        mbar_arrive_expect_tx(&scf[q], LG_SCSLOT);
                        uint8_t* sc = smem + (size_t)LG_NST * LG_STAGE + (size_t)q * LG_SCSLOT;
                        bulk_g2s(sc, bg + (size_t)kt * LG_BBLOB + LG_NB * 128u, LG_NB * 4u, &scf[q]);
                        bulk_g2s(sc + LG_NB * 4u, ag + (size_t)kt * LG_ABLOB + 16384u, 512u, &scf[q]);
                    }
                }
            }
        } else if (tid == 32) {   // ---- MMA issuer
            const uint32_t idesc = FP8 ? make_idesc_e4m3(128, LG_NB) : make_idesc_i8(128, LG_NB);
            uint32_t it = 0;
            for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
                for (int kt = 0; kt < p.n_kt; ++kt, ++it) {
                    const uint32_t s = it % LG_NST, ph = (it / LG_NST) & 1u;
                    const uint32_t tl = it / NCH, ch = it % NCH, a = tl & 1u;   // RHT tile, chunk inside it, accumulator
                    if (ch == 0) mbar_wait(&acc_empty[a], ((tl >> 1) & 1u) ^ 1u);
                    mbar_wait(&full[s], ph);
                    tc_fence_after();
                    const uint32_t sb = smem_a + s * LG_STAGE, sa = sb + LG_NB * 128u;
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks) {
                        if (FP8) mma_e4m3(tmem + a * LG_NB, make_desc_sw128(sa + ks * 32), make_desc_sw128(sb + ks * 32), idesc, (ks > 0 || ch > 0));
                        else mma_i8(tmem + a * LG_NB, make_desc_sw128(sa + ks * 32), make_desc_sw128(sb + ks * 32), idesc, (ks > 0 || ch > 0));
                    }
                    mma_commit(&empty[s]);
                    if (ch == NCH - 1) mma_commit(&acc_full[a]);
                }
            }
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
        // ---- epilogue: TMEM lane quarter q = warp % 4, column half = (warp - 4) / 4
        const int q = warp & 3, half = (warp - 4) >> 2;
        const int row = q * 32 + lane;
        // fp32 accumulators as packed pairs: the rescale is two packed instructions (mul.f32x2, fma.f32x2) per pair
        uint64_t yacc[64];
#pragma unroll
        for (int i = 0; i < 64; ++i) yacc[i] = 0ull;
        uint32_t it = 0;
        uint32_t v[2][32];
        const uint32_t tlane = tmem + half * 128 + ((uint32_t)(q * 32) << 16);
        // first chunk of K-step `i`: wait for its operands (scales) and its accumulator, start the TMEM load
        // step i = RHT tile i of this CTA's stream; its scales sit in the stage of its LAST chunk
        auto begin_step = [&](uint32_t i) {
            mbar_wait(&scf[i % LG_NSC], (i / LG_NSC) & 1u);   // the TMA-written scales are visible to this thread
            mbar_wait(&acc_full[i & 1u], (i >> 1) & 1u);
            tc_fence_after();
            const uint32_t ta = tlane + (i & 1u) * LG_NB;
            tmem_ld16(ta, v[0]);
            tmem_ld16(ta + 16, v[0] + 16);
        };
        const int my_tiles = blockIdx.x < n_tiles ? (n_tiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
        const int n_tl = p.n_kt / NCH;   // RHT tiles along K
        const uint32_t n_steps = (uint32_t)my_tiles * (uint32_t)n_tl;
        if (n_steps) begin_step(0);
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            int bt, rb;
            lg_tile_coords(tile, p.n_rb, p.n_bt, bt, rb);
            for (int kt = 0; kt < n_tl; ++kt, ++it) {
                const uint32_t q = it % LG_NSC, a = it & 1u;
                const uint32_t sb = sc_a + q * LG_SCSLOT;
                const float sw = lds_f32(sb + LG_NB * 4 + row * 4);
                const uint64_t sw2 = pack_f32x2(sw, sw);
                const uint32_t sx_a = sb + half * 512;
                const uint32_t taddr = tlane + a * LG_NB;
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    const int c0 = ch * 32;
                    tmem_ld_wait();
                    if (ch < 3) {   // the next chunk's accumulators fly while this one is rescaled
                        tmem_ld16(taddr + c0 + 32, v[(ch + 1) & 1]);
                        tmem_ld16(taddr + c0 + 48, v[(ch + 1) & 1] + 16);
                    } else {        // the accumulator is in registers: hand the TMEM buffer back to the MMA warp,
                        tc_fence_before();   // and start on the next K-step's accumulator while this chunk is rescaled
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&acc_empty[a]);
                        if (it + 1 < n_steps) begin_step(it + 1);
                    }
                    const uint32_t* vc = v[ch & 1];
                    if (p.acc_i32) {   // parity / debug output, off the hot path
                        const int64_t rr = (int64_t)rb * 128 + row;
                        const int64_t bb = (int64_t)bt * LG_NB + half * 128 + c0;
                        if (rr < p.m)
                            for (int e = 0; e < 32; ++e)
                                if (bb + e < p.B) p.acc_i32[((int64_t)kt * p.B + bb + e) * p.m + rr] = (int)vc[e];
                    }
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const uint4 s4 = lds128(sx_a + (c0 + 4 * e) * 4);
                        const uint64_t f01 = FP8 ? pack_u32x2(vc[4 * e + 0], vc[4 * e + 1]) : pack_f32x2((float)(int)vc[4 * e + 0], (float)(int)vc[4 * e + 1]);
                        const uint64_t f23 = FP8 ? pack_u32x2(vc[4 * e + 2], vc[4 * e + 3]) : pack_f32x2((float)(int)vc[4 * e + 2], (float)(int)vc[4 * e + 3]);
                        yacc[(c0 >> 1) + 2 * e + 0] = fma_f32x2(mul_f32x2(f01, sw2), pack_u32x2(s4.x, s4.y), yacc[(c0 >> 1) + 2 * e + 0]);
                        yacc[(c0 >> 1) + 2 * e + 1] = fma_f32x2(mul_f32x2(f23, sw2), pack_u32x2(s4.z, s4.w), yacc[(c0 >> 1) + 2 * e + 1]);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&sce[q]);   // the scales of this tile have been read
            }
            const int64_t r = (int64_t)rb * 128 + row;
            const int64_t b0 = (int64_t)bt * LG_NB + half * 128;
            if (r < p.m) {
                const int64_t nc = p.B - b0 < 128 ? p.B - b0 : 128;   // columns of this half inside the batch
                if (p.y_bf16) {
                    __nv_bfloat16* yp = p.y_bf16 + b0 * p.ldy + r;
                    if (nc == 128) {
#pragma unroll
                        for (int c = 0; c < 64; ++c) {
                            yp[0] = __float2bfloat16_rn(f32x2_lo(yacc[c]));
                            yp[p.ldy] = __float2bfloat16_rn(f32x2_hi(yacc[c]));
                            yp += 2 * p.ldy;
                        }
                    } else {
#pragma unroll
                        for (int c = 0; c < 128; ++c)
                            if (c < nc) yp[c * p.ldy] = __float2bfloat16_rn((c & 1) ? f32x2_hi(yacc[c >> 1]) : f32x2_lo(yacc[c >> 1]));
                    }
                }
                if (p.y_f32) {
                    float* yp = p.y_f32 + b0 * p.m + r;
#pragma unroll
                    for (int c = 0; c < 128; ++c)
                        if (c < nc) yp[c * p.m] = (c & 1) ? f32x2_hi(yacc[c >> 1]) : f32x2_lo(yacc[c >> 1]);
                }
            }
#pragma unroll
            for (int c = 0; c < 64; ++c) yacc[c] = 0ull;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 512);
}

}  // namespace hq
