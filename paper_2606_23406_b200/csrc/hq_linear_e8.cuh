// hq_linear_e8.cuh — the fused decode + INT8 MMA kernel for E8 tiles of 128 (north_star (a)-(d)).
//
// Persistent CTA of NWG independent warp groups (128 threads each, one CTA per SM).  A warp group owns a
// stream of tiles (row block rb, K-tile kt); lane = weight row, warp = sub-group (FORMAT §5):
//   A3  coalesced 128-byte loads of the sub-group's U / R words straight into registers, software pipeline
//       offset(t+2) -> header + dense words(t+1) -> ragged words(t+1), L2 prefetch of t+2, no shared-memory staging
//       of the bitstream;
//   A4  phase 1 of hq_e8_decode.cuh: unary section -> nibble stream (shared-memory scratch, conflict-free);
//   A5  phase 2: gaps + remainders -> INT8 lattice points, SWAR over four blocks, written with 128-bit stores into
//       the K-major SWIZZLE_128B A operand tile (decoded weights never leave shared memory);
//   A6  one thread issues 4 x tcgen05.mma kind::i8 (M=128, N=NB, K=32) per tile; the activation operand tile
//       arrives by a TMA bulk copy (already in UMMA layout, written by k_act_blob); accumulators sit in TMEM;
//   A7  the next iteration drains the accumulator row (tcgen05.ld) and rescales by rho/(alpha sqrt n) * s_x; split-K
//       partial sums are reduced in-kernel by the last split to arrive (deterministic order).
// The MMA of tile t overlaps phase 1 of tile t+1; the A tile is single-buffered per warp group.  The four warps of a
// warp group never meet at a barrier: the last one to finish its rows issues the MMA.
// CTA blockIdx.x owns a contiguous range of items (row block, batch tile of NB activation rows, split);
// up to E8_MAXW weights that share x are stacked into one item space (hq_linear_group).
#pragma once
#include "hq_common.cuh"
#include "hq_e8_decode.cuh"
#include "hq_internal.h"
#include "hq_tc.cuh"

namespace hq {

constexpr int E8_DENSE = 8;        // U word-rows assumed present in every row of a full sub-group when u_dense says so
constexpr int E8_NW = 10;          // U words per row handled by the fast path (tile 128: 8.1 on average at 4 bps)
constexpr int E8_SCR_STRIDE = 17;  // nibble words per row + 1 (bank-conflict-free)

__host__ __device__ constexpr uint32_t e8_bblob_bytes(int NB) { return (uint32_t)(NB * 128 + NB * 4); }
__host__ __device__ constexpr uint32_t e8_bslot_bytes(int NB) { return (e8_bblob_bytes(NB) + 1023u) & ~1023u; }
__host__ __device__ constexpr uint32_t e8_wg_bytes(int NB) {
    return (16384u + 2u * e8_bslot_bytes(NB) + 128u * E8_SCR_STRIDE * 4u + 1023u) & ~1023u;
}
template <int NB, int NWG>
constexpr size_t e8_smem_bytes() {
    return 1024 + (size_t)E8_LUT_BYTES + (size_t)NWG * e8_wg_bytes(NB) + 8 * (NWG * 3 + 1) + 16 + 4 * NWG + 16;
}
// K index inside a tile of the code of (block blk, coordinate i) in the A / B operand tiles
__host__ __device__ inline int e8_kcol(int j) {  // j = 8*blk + i (natural order)
    int blk = j >> 3, i = j & 7;
    return 32 * (blk >> 2) + 4 * i + (blk & 3);
}

constexpr int E8_MAXW = 4;   // weights per launch (hq_linear_group: matrices that share x, e.g. q/k/v or gate/up)
struct E8Params {
    const uint8_t* blob[E8_MAXW];
    const uint32_t* sub_off[E8_MAXW];
    int64_t m[E8_MAXW];
    float* partials[E8_MAXW];   // [n_split][B][m_w]
    __nv_bfloat16* y_bf16[E8_MAXW];   // outputs [B][ldy_w] (may be null)
    float* y_f32[E8_MAXW];      // optional fp32 outputs [B][m_w]
    int64_t ldy[E8_MAXW];
    unsigned int* counters;     // [global row block][batch tile][4 warps], zero between launches: split arrivals
    float inv_A[E8_MAXW];
    int rb_base[E8_MAXW + 1];   // the weights' row blocks stacked: weight w owns global row blocks [rb_base[w], rb_base[w+1])
    int n_w;
    const uint32_t* lut;        // global copy of the phase-1 table, E8_LUT_WORDS words
    int n_kt, n_split, L, n_items;   // item = (global row block, batch tile, split): L = n_kt / n_split consecutive tiles
    int n_bt;                   // batch tiles of NB activation rows; adjacent items share the row block (weights stay hot)
    int u_dense;                // every present row of the tensors has at least this many U words
    const uint8_t* bblob;       // [n_bt][n_kt][e8_bblob_bytes(NB)]
    int64_t B;
    int32_t* acc_i32;           // [n_kt][B][m] or null (single weight only)
    // batch 1 (k_gemv_e8, hq_gemv_e8.cuh): the kernel quantizes the activation vector itself
    const void* x;              // [n_in] bf16 or f32
    int dtype;
    const int8_t* dsign;        // [n_in] RHT signs
    // the folds of a decoder layer (FORMAT R8-R10), batch-1 kernel only
    int fold_mode;              // 0 plain; 1 RMSNorm: x = residual stream h, fold_aux = gain; 2 SiLU.mul: x = gate, fold_aux = up
    float fold_eps;
    const __nv_bfloat16* fold_aux;          // [n_in] bf16
    const __nv_bfloat16* res[E8_MAXW];      // [m_w] bf16 added to the output (R10), may be null
};

// Tile descriptor, three registers; the stream of tiles of one warp group is advanced without divisions.
struct E8Desc {
    uint32_t gk;      // rb * n_kt + kt, bit 31 = valid
    uint32_t ks;      // kt | split << 12 | last-of-item << 31
    uint32_t rb;      // row block inside its weight (16 bits) | batch tile << 16 (12 bits) | weight index << 28
    __device__ __forceinline__ uint32_t rbl() const { return rb & 0xffffu; }
    __device__ __forceinline__ uint32_t bt() const { return (rb >> 16) & 0xfffu; }
    __device__ __forceinline__ uint32_t w() const { return rb >> 28; }
    __device__ __forceinline__ bool valid() const { return (gk >> 31) != 0; }
    __device__ __forceinline__ uint32_t kt() const { return ks & 0xfffu; }
    __device__ __forceinline__ uint32_t split() const { return (ks >> 12) & 0xfffu; }
    __device__ __forceinline__ bool last() const { return (ks >> 31) != 0; }
    __device__ __forceinline__ uint32_t g() const { return gk & 0x7fffffffu; }
};
// CTA c owns the contiguous item range [c*I/G, (c+1)*I/G) (per-SM balance to within one item); its warp
// group w takes items first+w, first+w+NWG, ...
struct E8Iter {
    int item, end, j, rb, split;   // current position
    int dS, dR, step;              // step % n_split, step / n_split
    __device__ __forceinline__ void init(const E8Params& p, int first, int end_, int step_) {
        item = first; end = end_; j = 0; step = step_;
        rb = first / p.n_split; split = first % p.n_split;
        dS = step_ % p.n_split; dR = step_ / p.n_split;
    }
    __device__ __forceinline__ E8Desc get(const E8Params& p) const {
        E8Desc d;
        const bool v = item < end;
        const int kt = split * p.L + j;
        int rbg = rb, bt = 0;                                  // `rb` counts (global row block, batch tile) pairs
        if (p.n_bt > 1) { rbg = rb / p.n_bt; bt = rb - rbg * p.n_bt; }
        int w = 0;
#pragma unroll
        for (int i = 1; i < E8_MAXW; ++i)
            if (i < p.n_w && rbg >= p.rb_base[i]) w = i;
        const int rbl = rbg - p.rb_base[w];
        d.gk = (uint32_t)(rbl * p.n_kt + kt) | 0x80000000u;
        d.ks = (uint32_t)kt | ((uint32_t)split << 12) | ((j == p.L - 1) ? 0x80000000u : 0u);
        d.rb = (uint32_t)rbl | ((uint32_t)bt << 16) | ((uint32_t)w << 28);
        if (!v) { d.gk = 0; d.ks = 0; d.rb = 0; }
        return d;
    }
    __device__ __forceinline__ void next(const E8Params& p) {
        if (++j == p.L) {
            j = 0; item += step;
            split += dS; rb += dR;
            if (split >= p.n_split) { split -= p.n_split; ++rb; }
        }
    }
};

// K = Rice parameter, NB = MMA N (activation rows per batch tile), BC = accumulator columns drained per row
// (1 when batch == 1, else NB), NWG = warp groups per CTA, CPS = CTAs per SM (two half-size CTAs per SM let the
// tail of one launch overlap the prologue of the next under PDL).
template <int K, int NB, int BC, int NWG, int CPS>
__global__ void __launch_bounds__(NWG * 128, CPS)
k_linear_e8(E8Params p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    constexpr uint32_t BSLOT = e8_bslot_bytes(NB);
    constexpr uint32_t WG_BYTES = e8_wg_bytes(NB);
    constexpr int KW = 4 * K;   // R words per row
    const int tid = threadIdx.x, wg = tid >> 7, t = tid & 127, warp = t >> 5, lane = t & 31;
    const uint32_t smem_a = smem_u32(smem);
    const uint32_t wg_a = smem_a + E8_LUT_BYTES + (uint32_t)wg * WG_BYTES;
    const uint32_t sA_base = wg_a;                                  // 128 x 128 int8, SWIZZLE_128B
    const uint32_t sB_a = wg_a + 16384;                             // 2 slots
    const uint32_t scr_a = sB_a + 2 * BSLOT + (uint32_t)t * E8_SCR_STRIDE * 4;  // this row's nibble words
    uint64_t* bars = (uint64_t*)(smem + E8_LUT_BYTES + (size_t)NWG * WG_BYTES);
    uint64_t* bar_b = bars + wg * 3;        // [2] activation tile landed
    uint64_t* bar_mma = bars + wg * 3 + 2;  // MMA of the current tile done
    uint64_t* bar_lut = bars + NWG * 3;
    uint32_t* tmem_slot = (uint32_t*)(bars + NWG * 3 + 1);
    uint32_t* arrive_cnt = tmem_slot + 2 + wg;   // warps of this warp group that finished their part of the A tile

    constexpr uint32_t TCOLS_WG = NB < 32 ? 32 : NB;
    constexpr uint32_t TCOLS = TCOLS_WG * NWG <= 128 ? 128 : (TCOLS_WG * NWG <= 256 ? 256 : 512);
    if (tid < 32) tmem_alloc(tmem_slot, TCOLS);
    if (t == 0) {
        mbar_init(&bar_b[0], 1); mbar_init(&bar_b[1], 1); mbar_init(bar_mma, 1);
        *arrive_cnt = 0;
        if (wg == 0) mbar_init(bar_lut, 1);
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
    const uint32_t tmem_acc = *tmem_slot + (uint32_t)wg * TCOLS_WG;
    const uint32_t idesc = make_idesc_i8(128, NB);
    const uint32_t lut_lane = smem_a + (uint32_t)(lane & (E8_LUT_COPIES - 1)) * 4;
    const uint32_t sA_a = sA_base + (uint32_t)((t >> 3) * 1024 + (t & 7) * 128);   // this row of the A tile
    const int it_first = (int)(((int64_t)blockIdx.x * p.n_items) / gridDim.x) + wg;
    const int it_end = (int)(((int64_t)(blockIdx.x + 1) * p.n_items) / gridDim.x);
    const uint32_t lane_lt = (1u << lane) - 1u;
    const uint32_t cnt_a = smem_u32(arrive_cnt);

    // ---- tile queue (tau .. tau+2) and software pipeline registers
    E8Iter it;
    it.init(p, it_first, it_end, NWG);
    E8Desc q0 = it.get(p); it.next(p);
    E8Desc q1 = it.get(p); it.next(p);
    E8Desc q2 = it.get(p); it.next(p);
    if (!q0.valid()) {   // nothing to do for this warp group (the CTA still joins the final barrier)
        __syncthreads();
        if (tid < 32) tmem_dealloc(*tmem_slot, TCOLS);
        return;
    }
    auto load_off = [&](const E8Desc& d) -> uint32_t {
        return d.valid() ? __ldg(p.sub_off[d.w()] + ((size_t)d.g() * 4 + warp)) : 0u;
    };
    auto issue_b = [&](const E8Desc& d, int slot) {  // wg thread 0: TMA bulk copy of a tile's activation operand
        if (!d.valid()) return;
        mbar_arrive_expect_tx(&bar_b[slot], e8_bblob_bytes(NB));
        bulk_g2s(smem + E8_LUT_BYTES + (size_t)wg * WG_BYTES + 16384 + slot * BSLOT,
                 p.bblob + ((size_t)d.bt() * p.n_kt + d.kt()) * e8_bblob_bytes(NB), e8_bblob_bytes(NB), &bar_b[slot]);
    };
    // a sub-group whose 32 rows are all present has at least p.u_dense words in every row: those word-rows are
    // dense (no rank needed); the rest are compacted (FORMAT §5)
    // U word-rows.  In a sub-group whose 32 rows are all present every row has at least p.u_dense words; the launcher
    // passes u_dense = E8_DENSE (8: the common case at tile 128, 2 unary bits per symbol) or 0.  Dense word-rows need
    // only the sub-group offset; the rest are compacted (FORMAT §5) and need the header.
    auto is_dense = [&](bool full_rows) -> bool { return full_rows && p.u_dense >= E8_DENSE; };   // warp-uniform
    auto load_u_dense = [&](const uint8_t* sgp, bool full_rows, uint32_t* U) {
        if (!is_dense(full_rows)) return;
        const uint32_t* ua = (const uint32_t*)(sgp + 128) + KW * 32 + lane;
#pragma unroll
        for (int w = 0; w < E8_DENSE; ++w) U[w] = __ldg(ua + w * 32);
    };
    auto load_u_ragged = [&](const uint8_t* sgp, uint32_t ul, bool full_rows, uint32_t* U) {
        const uint32_t* uarea = (const uint32_t*)(sgp + 128) + KW * 32;
        const uint32_t nw = (ul + 31) >> 5;
        if (is_dense(full_rows)) {
            uint32_t base = E8_DENSE * 32;
#pragma unroll
            for (int w = E8_DENSE; w < E8_NW; ++w) {
                const bool has = nw > (uint32_t)w;
                const uint32_t mk = __ballot_sync(0xffffffffu, has);
                U[w] = has ? __ldg(uarea + base + __popc(mk & lane_lt)) : 0u;
                base += __popc(mk);
            }
        } else {
            uint32_t base = 0;
#pragma unroll
            for (int w = 0; w < E8_NW; ++w) {
                const bool has = nw > (uint32_t)w;
                const uint32_t mk = __ballot_sync(0xffffffffu, has);
                U[w] = has ? __ldg(uarea + base + __popc(mk & lane_lt)) : 0u;
                base += __popc(mk);
            }
        }
    };
    auto load_r = [&](const uint8_t* sgp, uint32_t* R) {
        const uint32_t* rarea = (const uint32_t*)(sgp + 128);
#pragma unroll
        for (int j = 0; j < KW; ++j) R[j] = __ldg(rarea + j * 32 + lane);
    };
    auto rows_full = [&](const E8Desc& d) -> bool { return (int64_t)d.rbl() * 128 + warp * 32 + 32 <= p.m[d.w()]; };

    uint32_t Uw[E8_NW], Rw[KW > 0 ? KW : 1];
    // prologue: offsets of tiles 0 and 1 together, then everything of tile 0 that needs only its offset
    uint32_t off_n1 = load_off(q1);
    const uint8_t* sgp_c = p.blob[q0.w()] + 16 * (size_t)load_off(q0);
    uint32_t ul_c = __ldg((const uint16_t*)sgp_c + lane), nrm_c = __ldg((const uint16_t*)sgp_c + 32 + lane);
    load_u_dense(sgp_c, rows_full(q0), Uw);
    load_r(sgp_c, Rw);
    load_u_ragged(sgp_c, ul_c, rows_full(q0), Uw);
    const uint8_t* sgp_n1 = nullptr;
    uint32_t ul_n1 = 0, nrm_n1 = 0;

    float yacc[BC];
#pragma unroll
    for (int b = 0; b < BC; ++b) yacc[b] = 0.0f;
    float sw_prev = 0.0f;      // rho / (alpha sqrt n) of the tile whose MMA is in flight
    E8Desc prev; prev.gk = 0; prev.ks = 0; prev.rb = 0;

    // epilogue of tile `x` = tile number tau (its MMA has completed): drain the accumulator row, rescale, accumulate (A7)
    auto epilogue = [&](const E8Desc& x, int tau) {
        const int64_t r = (int64_t)x.rbl() * 128 + t;
        const int64_t mw = p.m[x.w()];
        const int64_t b0 = (int64_t)x.bt() * NB;
        mbar_wait(&bar_b[tau & 1], (uint32_t)((tau >> 1) & 1));   // the TMA-written scales are visible to this thread
        const uint32_t sx_a = sB_a + (tau & 1) * BSLOT + NB * 128;
        const uint32_t taddr = tmem_acc + ((uint32_t)(warp * 32) << 16);
        if (BC == 1) {
            uint32_t v;
            tmem_ld1(taddr, v);
            tmem_ld_wait();
            if (p.acc_i32 && r < mw) p.acc_i32[((int64_t)x.kt() * p.B + b0) * mw + r] = (int)v;
            yacc[0] += (sw_prev * lds_f32(sx_a)) * (float)(int)v;
        } else {
#pragma unroll
            for (int c0 = 0; c0 < BC; c0 += 16) {
                uint32_t v[16];
                tmem_ld16(taddr + c0, v);
                tmem_ld_wait();
                if (p.acc_i32 && r < mw) {   // parity / debug output, off the hot path
                    for (int e = 0; e < 16; ++e)
                        if (b0 + c0 + e < p.B) p.acc_i32[((int64_t)x.kt() * p.B + b0 + c0 + e) * mw + r] = (int)v[e];
                }
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const uint4 s4 = lds128(sx_a + (c0 + 4 * e) * 4);
                    yacc[c0 + 4 * e + 0] += (sw_prev * __uint_as_float(s4.x)) * (float)(int)v[4 * e + 0];
                    yacc[c0 + 4 * e + 1] += (sw_prev * __uint_as_float(s4.y)) * (float)(int)v[4 * e + 1];
                    yacc[c0 + 4 * e + 2] += (sw_prev * __uint_as_float(s4.z)) * (float)(int)v[4 * e + 2];
                    yacc[c0 + 4 * e + 3] += (sw_prev * __uint_as_float(s4.w)) * (float)(int)v[4 * e + 3];
                }
            }
        }
        tc_fence_before();
        if (x.last()) {   // split-K: this item's partial sums go to the workspace (reduced after the tile loop)
            float* part = p.partials[x.w()];
            if (r < mw) {
                if (p.n_split == 1) {   // the item covered all of K: yacc is y
                    __nv_bfloat16* yb = p.y_bf16[x.w()];
                    float* yf = p.y_f32[x.w()];
                    const int64_t ldy = p.ldy[x.w()];
#pragma unroll
                    for (int b = 0; b < BC; ++b) {
                        if (b0 + b < p.B) {
                            if (yb) yb[(b0 + b) * ldy + r] = __float2bfloat16_rn(yacc[b]);
                            if (yf) yf[(b0 + b) * mw + r] = yacc[b];
                        }
                    }
                } else {
#pragma unroll
                    for (int b = 0; b < BC; ++b)
                        if (b0 + b < p.B) part[((int64_t)x.split() * p.B + b0 + b) * mw + r] = yacc[b];
                }
            }
#pragma unroll
            for (int b = 0; b < BC; ++b) yacc[b] = 0.0f;
        }
    };
    // split-K reduction inside the kernel: after its last tile a warp publishes its partial sums (one fence) and
    // arrives once per item on a per-(row block, batch tile, warp) counter; the LAST of the n_split arrivals adds the
    // partials in split order - deterministic - and writes y (A7).  No block barrier, no extra launch.
    auto arrive = [&](const E8Desc& x) {
        const int64_t r = (int64_t)x.rbl() * 128 + t;
        const int64_t mw = p.m[x.w()];
        const int64_t b0 = (int64_t)x.bt() * NB;
        float* part = p.partials[x.w()];
        unsigned int last = 0;
        if (lane == 0) {
            unsigned int* cnt = p.counters + (((size_t)(p.rb_base[x.w()] + x.rbl()) * p.n_bt + x.bt()) * 4 + warp);
            last = atomicAdd(cnt, 1u) == (unsigned int)(p.n_split - 1);
            if (last) *cnt = 0u;
        }
        last = __shfl_sync(0xffffffffu, last, 0);
        if (!last) return;
        __threadfence();
        if (r >= mw) return;
        __nv_bfloat16* yb = p.y_bf16[x.w()];
        float* yf = p.y_f32[x.w()];
        const int64_t ldy = p.ldy[x.w()];
        constexpr int CB = BC < 4 ? BC : 4;   // columns summed together: CB x 8 loads in flight
        const int64_t sstride = p.B * mw;
        for (int bb = 0; bb < BC; bb += CB) {
            if (b0 + bb >= p.B) break;
            float sum[CB];
#pragma unroll
            for (int c = 0; c < CB; ++c) sum[c] = 0.0f;
            for (int sp0 = 0; sp0 < p.n_split; sp0 += 8) {   // split order per column
                float v[CB][8];
#pragma unroll
                for (int c = 0; c < CB; ++c)
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        v[c][u] = (sp0 + u < p.n_split && b0 + bb + c < p.B)
                                      ? __ldcg(part + (b0 + bb + c) * mw + r + (sp0 + u) * sstride) : 0.0f;
#pragma unroll
                for (int c = 0; c < CB; ++c)
#pragma unroll
                    for (int u = 0; u < 8; ++u) sum[c] += v[c][u];
            }
#pragma unroll
            for (int c = 0; c < CB; ++c) {
                if (b0 + bb + c < p.B) {
                    if (yb) yb[(b0 + bb + c) * ldy + r] = __float2bfloat16_rn(sum[c]);
                    if (yf) yf[(b0 + bb + c) * mw + r] = sum[c];
                }
            }
        }
    };

    mbar_wait(bar_lut, 0u);

    for (int tau = 0;; ++tau) {
        // ---- move the pipeline: offset of tile tau+2
        const uint32_t off_n2 = load_off(q2);

        // ---- phase 1: unary section -> nibble words (A4)
        const uint32_t nw = (ul_c + 31) >> 5;
        const uint32_t maxul = __reduce_max_sync(0xffffffffu, ul_c);   // longest U-section of the sub-group, bits
        const uint32_t maxnw = (maxul + 31) >> 5;
        {
            uint32_t T = 0, acc = 0, wo = scr_a;
#pragma unroll
            for (int w = 0; w < E8_NW; ++w) {   // an absent word is zero: no terminators, nothing appended
                if (w < E8_DENSE) {
                    e8_unary_word(Uw[w], lut_lane, T, acc, wo);
                } else if ((uint32_t)w < maxnw) {   // tail words: only the bytes some row of the warp still uses
                    const int nb = (int)min(4u, (maxul - 32u * (uint32_t)w + 7u) >> 3);
                    e8_unary_word(Uw[w], lut_lane, T, acc, wo, nb);
                }
            }
        }
        // the U registers are free: header and dense U words of tile tau+1 (its offset arrived an iteration ago)
        sgp_n1 = p.blob[q1.w()] + 16 * (size_t)off_n1;
        if (q1.valid()) {
            ul_n1 = __ldg((const uint16_t*)sgp_n1 + lane);
            nrm_n1 = __ldg((const uint16_t*)sgp_n1 + 32 + lane);
            load_u_dense(sgp_n1, rows_full(q1), Uw);
        }

        // ---- the previous tile's MMA must be done before its accumulators are read and the A tile is rewritten
        if (tau > 0) {
            mbar_wait(bar_mma, (uint32_t)((tau - 1) & 1));
            tc_fence_after();
            epilogue(prev, tau - 1);
        }
        // ---- phase 2: nibble words + remainders -> INT8 points in the A tile (A5)
        const int64_t r = (int64_t)q0.rbl() * 128 + t;
        const bool present = r < p.m[q0.w()] && ul_c > 0;
        uint32_t total = 0;
        {
            uint32_t prevWo = 15u << 24;  // e_{-1} = -1 mod 16
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                uint32_t W[4], C[8];
#pragma unroll
                for (int w = 0; w < 4; ++w) W[w] = lds32(scr_a + (c * 4 + w) * 4);
                e8_run<K>(W, Rw + c * K, prevWo, total, C);
                if (!present) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) C[i] = 0u;
                }
                const uint32_t u0 = (uint32_t)(((2 * c) ^ (t & 7)) << 4), u1 = (uint32_t)(((2 * c + 1) ^ (t & 7)) << 4);
                sts128(sA_a + u0, C[0], C[1], C[2], C[3]);
                sts128(sA_a + u1, C[4], C[5], C[6], C[7]);
            }
        }
        if (present && (nw > (uint32_t)E8_NW || total + 128u != ul_c)) {
            // a quotient >= 16 or a long row: generic decoder, straight from global memory
            SubGroup sg = sub_group(sgp_c, KW);
            WordsRowU uw{nullptr, sg.uarea, sg.ulen, nw, 0u, lane};
            WordsRowR rw{sg.rarea, lane, KW};
            decode_row_generic<LAT_E8>(rw, 0u, uw, 0u, 128, K, K, [&](int bk, const int* c) {
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int col = e8_kcol(8 * bk + e);
                    sts8(sA_a + ((((col >> 4) ^ (t & 7)) << 4) | (col & 15)), (uint32_t)(uint8_t)(int8_t)c[e]);
                }
            });
        }
        // the R registers are free: remainder words of tile tau+1, and its ragged U words (the header has arrived)
        if (q1.valid()) {
            load_r(sgp_n1, Rw);
            load_u_ragged(sgp_n1, ul_n1, rows_full(q1), Uw);
        }
        const float sw_cur = f16_bits_to_f32((uint16_t)nrm_c) * p.inv_A[q0.w()];
        fence_proxy_async_smem();
        tc_fence_before();
        if (tau == 0) {
            // everything up to here touched only the weights; the activation operand, the partial sums and the debug
            // outputs belong to the stream order: join it (no-op unless launched with PDL)
            griddep_wait();
            if (t == 0) issue_b(q0, 0);
        }
        // No block barrier: the last of the four warps to finish the tile issues the MMA.  (A warp cannot arrive for tile
        // tau+1 before the MMA of tile tau was issued - it waits for its commit before phase 2 - so the arrivals of a
        // tile are the counter values 4 tau .. 4 tau + 3.)
        __syncwarp();
        bool issuer = false;
        if (lane == 0) {
            uint32_t old;
            asm volatile("atom.acq_rel.cta.shared::cta.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(cnt_a) : "memory");
            issuer = (old & 3u) == 3u;
        }
        if (issuer) {
            issue_b(q1, (tau + 1) & 1);   // that slot's last reader, the epilogue of tile tau-1, precedes every arrival
            mbar_wait(&bar_b[tau & 1], (uint32_t)((tau >> 1) & 1));
            tc_fence_after();
            const uint32_t b0s = sB_a + (tau & 1) * BSLOT;
#pragma unroll
            for (int ks = 0; ks < 4; ++ks)
                mma_i8(tmem_acc, make_desc_sw128(sA_base + ks * 32), make_desc_sw128(b0s + ks * 32), idesc, ks > 0);
            mma_commit(bar_mma);
        }
        // ---- rotate
        prev = q0;
        sw_prev = sw_cur;
        if (!q1.valid()) {  // drain: the last tile's epilogue
            mbar_wait(bar_mma, (uint32_t)(tau & 1));
            tc_fence_after();
            epilogue(prev, tau);
            break;
        }
        sgp_c = sgp_n1; ul_c = ul_n1; nrm_c = nrm_n1;
        // pull the sub-group of tile tau+2 into L2 (no registers held): its demand loads are issued an iteration from now
        if (q2.valid() && lane < 18)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(p.blob[q2.w()] + 16 * (size_t)off_n2 + lane * 128));
        off_n1 = off_n2;
        q0 = q1; q1 = q2;
        q2 = it.get(p); it.next(p);
    }
    // publish this thread's partial sums, then arrive for every item this warp group went through
    __threadfence();
    __syncwarp();
    if (p.n_split > 1) {
        E8Iter it2;
        it2.init(p, it_first, it_end, NWG);
        for (;;) {
            const E8Desc d = it2.get(p);
            if (!d.valid()) break;
            if (d.last()) arrive(d);
            it2.next(p);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (tid < 32) tmem_dealloc(*tmem_slot, TCOLS);
}

}  // namespace hq
