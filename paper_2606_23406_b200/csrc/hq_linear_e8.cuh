// hq_linear_e8.cuh — the fused decode + INT8 MMA kernel for E8 tiles of 128 (north_star (a)-(d)).
//
// Persistent CTA of E8_NWG independent warp groups (128 threads each, one CTA per SM).  A warp group owns a
// stream of tiles (row block rb, K-tile kt); lane = weight row, warp = sub-group (FORMAT §5):
//   A3  coalesced 128-byte loads of the sub-group's U / R words straight into registers, three-deep software
//       pipeline (offset -> header -> words), no shared-memory staging of the bitstream;
//   A4  phase 1 of hq_e8_decode.cuh: unary section -> nibble stream (shared-memory scratch, conflict-free);
//   A5  phase 2: gaps + remainders -> INT8 lattice points, SWAR over four blocks, written with 128-bit stores into
//       the K-major SWIZZLE_128B A operand tile (decoded weights never leave shared memory);
//   A6  one thread issues 4 x tcgen05.mma kind::i8 (M=128, N=NB, K=32) per tile; the activation operand tile
//       arrives by a TMA bulk copy (already in UMMA layout, written by k_act_blob); accumulators sit in TMEM;
//   A7  the next iteration drains the accumulator row (tcgen05.ld) and rescales by rho/(alpha sqrt n) * s_x.
// The MMA of tile t overlaps phase 1 of tile t+1; the A tile is single-buffered per warp group.
#pragma once
#include "hq_common.cuh"
#include "hq_e8_decode.cuh"
#include "hq_internal.h"
#include "hq_tc.cuh"

namespace hq {

constexpr int E8_NWG = 4;          // warp groups per CTA
constexpr int E8_NW = 10;          // U words per row handled by the fast path (tile 128: 8.1 on average at 4 bps)
constexpr int E8_SCR_STRIDE = 17;  // nibble words per row + 1 (bank-conflict-free)

__host__ __device__ constexpr uint32_t e8_bblob_bytes(int NB) { return (uint32_t)(NB * 128 + NB * 4); }
__host__ __device__ constexpr uint32_t e8_bslot_bytes(int NB) { return (e8_bblob_bytes(NB) + 1023u) & ~1023u; }
// K index inside a tile of the code of (block blk, coordinate i) in the A / B operand tiles
__host__ __device__ inline int e8_kcol(int j) {  // j = 8*blk + i (natural order)
    int blk = j >> 3, i = j & 7;
    return 32 * (blk >> 2) + 4 * i + (blk & 3);
}

struct E8Params {
    const uint8_t* blob;
    const uint32_t* sub_off;
    const uint32_t* lut;     // global copy of the phase-1 table, E8_LUT_WORDS words
    int64_t m;
    int n_kt, n_rb, n_bt, n_split, L, n_items;   // item = (rb, bt, split): L = n_kt / n_split consecutive tiles
    float inv_A;
    const uint8_t* bblob;    // [n_bt][n_kt][e8_bblob_bytes(NB)]
    int64_t B;
    float* partials;         // [n_split][B][m]
    int32_t* acc_i32;        // [n_kt][B][m] or null
};

struct E8Tile {
    bool valid;
    int item, rb, bt, split, kt;
    bool first, last;
};
__device__ __forceinline__ E8Tile e8_tile(const E8Params& p, int gw, int GW, int tau) {
    E8Tile t;
    t.item = gw + (tau / p.L) * GW;
    t.valid = t.item < p.n_items;
    const int j = tau % p.L;
    t.split = t.item % p.n_split;
    const int rest = t.item / p.n_split;
    t.bt = rest % p.n_bt;
    t.rb = rest / p.n_bt;
    t.kt = t.split * p.L + j;
    t.first = j == 0;
    t.last = j == p.L - 1;
    return t;
}

template <int K, int NB>
__global__ void __launch_bounds__(E8_NWG * 128, 1)
k_linear_e8(E8Params p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    constexpr uint32_t BSLOT = e8_bslot_bytes(NB);
    constexpr uint32_t WG_BYTES = (16384 + 2 * BSLOT + 128 * E8_SCR_STRIDE * 4 + 1023u) & ~1023u;
    const int tid = threadIdx.x, wg = tid >> 7, t = tid & 127, warp = t >> 5, lane = t & 31;
    uint32_t* lut_s = (uint32_t*)smem;                                    // [E8_LUT_WORDS]
    uint8_t* wg_base = smem + E8_LUT_BYTES + (size_t)wg * WG_BYTES;
    uint8_t* sA = wg_base;                                                // 128 x 128 int8, SWIZZLE_128B
    uint8_t* sB = sA + 16384;                                             // 2 slots
    uint32_t* scr = (uint32_t*)(sB + 2 * BSLOT) + t * E8_SCR_STRIDE;      // this row's nibble words
    uint64_t* bars = (uint64_t*)(smem + E8_LUT_BYTES + (size_t)E8_NWG * WG_BYTES);
    uint64_t* bar_b = bars + wg * 3;       // [2] activation tile landed
    uint64_t* bar_mma = bars + wg * 3 + 2; // MMA of the current tile done
    uint32_t* tmem_slot = (uint32_t*)(bars + E8_NWG * 3);

    constexpr uint32_t TCOLS_WG = NB < 32 ? 32 : NB;
    constexpr uint32_t TCOLS = TCOLS_WG * E8_NWG;   // 128 or 256: a power of two
    if (tid < 32) tmem_alloc(tmem_slot, TCOLS);
    if (t == 0) {
        mbar_init(&bar_b[0], 1); mbar_init(&bar_b[1], 1); mbar_init(bar_mma, 1);
        mbar_fence_init();
    }
    for (int i = tid; i < E8_LUT_WORDS; i += E8_NWG * 128) lut_s[i] = __ldg(p.lut + i);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_acc = *tmem_slot + (uint32_t)wg * TCOLS_WG;
    const uint32_t idesc = make_idesc_i8(128, NB);
    const uint32_t* lut_lane = lut_s + (lane & (E8_LUT_COPIES - 1));
    const uint32_t a_row = (uint32_t)((t >> 3) * 1024 + (t & 7) * 128);
    const int gw = blockIdx.x * E8_NWG + wg, GW = gridDim.x * E8_NWG;

    // ---- software pipeline registers
    uint32_t off_n2 = 0;                  // sub-group offset of tile tau+2
    const uint8_t* sgp_n1 = nullptr;      // sub-group base of tile tau+1
    uint32_t ul_n1 = 0, nrm_n1 = 0;       // header of tile tau+1 (this lane's row)
    uint32_t Uw[E8_NW], Rw[4 * (K > 0 ? K : 1)], ul_c = 0, nrm_c = 0;   // tile tau (current)
    const uint8_t* sgp_c = nullptr;

    auto load_off = [&](int tau) -> uint32_t {
        E8Tile x = e8_tile(p, gw, GW, tau);
        if (!x.valid) return 0u;
        return __ldg(p.sub_off + ((int64_t)(x.rb * p.n_kt + x.kt) * 4 + warp));
    };
    auto issue_b = [&](int tau) {  // wg thread 0: TMA bulk copy of the activation tile of tile tau
        E8Tile x = e8_tile(p, gw, GW, tau);
        if (!x.valid) return;
        const int s = tau & 1;
        mbar_arrive_expect_tx(&bar_b[s], e8_bblob_bytes(NB));
        bulk_g2s(sB + s * BSLOT, p.bblob + ((size_t)x.bt * p.n_kt + x.kt) * e8_bblob_bytes(NB), e8_bblob_bytes(NB), &bar_b[s]);
    };
    // words of a tile whose header (ul) is known: U word-rows by ballot rank, R words interleaved
    auto load_words = [&](const uint8_t* sgp, uint32_t ul, uint32_t* U, uint32_t* R) {
        const uint32_t* rarea = (const uint32_t*)(sgp + 128);
        const uint32_t* uarea = rarea + K * 4 * 32;
#pragma unroll
        for (int j = 0; j < 4 * K; ++j) R[j] = __ldg(rarea + j * 32 + lane);
        const uint32_t nw = (ul + 31) >> 5;
        uint32_t base = 0;
#pragma unroll
        for (int w = 0; w < E8_NW; ++w) {
            const bool has = nw > (uint32_t)w;
            const uint32_t mk = __ballot_sync(0xffffffffu, has);
            U[w] = has ? __ldg(uarea + base + __popc(mk & ((1u << lane) - 1u))) : 0u;
            base += __popc(mk);
        }
    };

    // prologue: tile 0 words, tile 1 header, tile 2 offset
    {
        E8Tile x0 = e8_tile(p, gw, GW, 0);
        if (x0.valid) {
            sgp_c = p.blob + 16 * (size_t)load_off(0);
            ul_c = __ldg((const uint16_t*)sgp_c + lane);
            nrm_c = __ldg((const uint16_t*)sgp_c + 32 + lane);
            load_words(sgp_c, ul_c, Uw, Rw);
        }
        E8Tile x1 = e8_tile(p, gw, GW, 1);
        if (x1.valid) {
            sgp_n1 = p.blob + 16 * (size_t)load_off(1);
            ul_n1 = __ldg((const uint16_t*)sgp_n1 + lane);
            nrm_n1 = __ldg((const uint16_t*)sgp_n1 + 32 + lane);
        }
        off_n2 = load_off(2);
        if (t == 0) issue_b(0);
    }

    float yacc[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) yacc[b] = 0.0f;
    float sw_prev = 0.0f;      // rho / (alpha sqrt n) of the tile whose MMA is in flight
    E8Tile prev; prev.valid = false;

    // epilogue of tile `x` (its MMA has completed): drain the accumulator row, rescale, accumulate (A7)
    auto epilogue = [&](const E8Tile& x, int tau) {
        const int64_t r = (int64_t)x.rb * 128 + t;
        const int64_t b0 = (int64_t)x.bt * NB;
        mbar_wait(&bar_b[tau & 1], (uint32_t)((tau >> 1) & 1));   // the TMA-written scales are visible to this thread
        const float* sx = (const float*)(sB + (tau & 1) * BSLOT + NB * 128);
#pragma unroll
        for (int c0 = 0; c0 < NB; c0 += 16) {
            uint32_t v[16];
            tmem_ld16(tmem_acc + ((uint32_t)(warp * 32) << 16) + c0, v);
            tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const int a = (int)v[e];
                if (p.acc_i32 && r < p.m && b0 + c0 + e < p.B) p.acc_i32[((int64_t)x.kt * p.B + b0 + c0 + e) * p.m + r] = a;
                yacc[c0 + e] += (sw_prev * sx[c0 + e]) * (float)a;
            }
        }
        tc_fence_before();
        if (x.last) {
            if (r < p.m) {
#pragma unroll
                for (int b = 0; b < NB; ++b)
                    if (b0 + b < p.B) p.partials[((int64_t)x.split * p.B + b0 + b) * p.m + r] = yacc[b];
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) yacc[b] = 0.0f;
        }
    };

    for (int tau = 0;; ++tau) {
        const E8Tile cur = e8_tile(p, gw, GW, tau);
        if (!cur.valid) break;
        // ---- move the pipeline: words of tau+1 (header known), header of tau+2 (offset known), offset of tau+3
        uint32_t Un[E8_NW], Rn[4 * (K > 0 ? K : 1)];
        const E8Tile nx1 = e8_tile(p, gw, GW, tau + 1);
        if (nx1.valid) load_words(sgp_n1, ul_n1, Un, Rn);
        const E8Tile nx2 = e8_tile(p, gw, GW, tau + 2);
        const uint8_t* sgp_n2 = p.blob + 16 * (size_t)off_n2;
        uint32_t ul_n2 = 0, nrm_n2 = 0;
        if (nx2.valid) {
            ul_n2 = __ldg((const uint16_t*)sgp_n2 + lane);
            nrm_n2 = __ldg((const uint16_t*)sgp_n2 + 32 + lane);
        }
        off_n2 = load_off(tau + 3);

        // ---- phase 1: unary section -> nibble words (A4)
        const uint32_t nw = (ul_c + 31) >> 5;
        uint32_t maxnw = nw;
#pragma unroll
        for (int o = 16; o; o >>= 1) maxnw = max(maxnw, __shfl_xor_sync(0xffffffffu, maxnw, o));
        {
            uint32_t acc = 0, fs = 0;
            uint32_t* wo = scr;
#pragma unroll
            for (int w = 0; w < E8_NW; ++w)
                if ((uint32_t)w < maxnw) e8_unary_word(Uw[w], lut_lane, acc, fs, wo);
        }
        // ---- the previous tile's MMA must be done before its accumulators are read and the A tile is rewritten
        if (prev.valid) {
            mbar_wait(bar_mma, (uint32_t)((tau - 1) & 1));
            tc_fence_after();
            epilogue(prev, tau - 1);
        }
        // ---- phase 2: nibble words + remainders -> INT8 points in the A tile (A5)
        const int64_t r = (int64_t)cur.rb * 128 + t;
        bool ok = nw <= (uint32_t)E8_NW && r < p.m && ul_c > 0;
        uint32_t total = 0;
        {
            uint32_t prevWo = 15u << 24;  // e_{-1} = -1 mod 16
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                uint32_t W[4], C[8], qsum = 0;
#pragma unroll
                for (int w = 0; w < 4; ++w) W[w] = scr[c * 4 + w];
                e8_run<K>(W, Rw + c * K, prevWo, qsum, C);
                total += __dp4a(qsum, 0x01010101u, 0u);
                if (!(r < p.m && ul_c > 0)) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) C[i] = 0u;
                }
                const uint32_t u0 = (uint32_t)(((2 * c) ^ (t & 7)) << 4), u1 = (uint32_t)(((2 * c + 1) ^ (t & 7)) << 4);
                *(uint4*)(sA + a_row + u0) = make_uint4(C[0], C[1], C[2], C[3]);
                *(uint4*)(sA + a_row + u1) = make_uint4(C[4], C[5], C[6], C[7]);
            }
        }
        ok = ok && (total + 128u == ul_c);
        if (!ok && r < p.m && ul_c > 0) {  // a quotient >= 16 or a long row: generic decoder, straight from global memory
            SubGroup sg = sub_group(sgp_c, 4 * K);
            WordsRowU uw{nullptr, sg.uarea, sg.ulen, nw, 0u, lane};
            WordsRowR rw{sg.rarea, lane, 4 * K};
            decode_row_generic<LAT_E8>(rw, 0u, uw, 0u, 128, K, K, [&](int bk, const int* c) {
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int col = e8_kcol(8 * bk + e);
                    sA[a_row + ((((col >> 4) ^ (t & 7)) << 4) | (col & 15))] = (uint8_t)(int8_t)c[e];
                }
            });
        }
        const float sw_cur = f16_bits_to_f32((uint16_t)nrm_c) * p.inv_A;
        fence_proxy_async_smem();
        tc_fence_before();
        asm volatile("bar.sync %0, 128;" ::"r"(wg + 1) : "memory");
        if (t == 0) {
            issue_b(tau + 1);   // slot (tau+1)&1: its last reader, the epilogue of tile tau-1, is behind the barrier
            mbar_wait(&bar_b[tau & 1], (uint32_t)((tau >> 1) & 1));
            tc_fence_after();
            const uint32_t a0 = smem_u32(sA), b0s = smem_u32(sB + (tau & 1) * BSLOT);
#pragma unroll
            for (int ks = 0; ks < 4; ++ks)
                mma_i8(tmem_acc, make_desc_sw128(a0 + ks * 32), make_desc_sw128(b0s + ks * 32), idesc, ks > 0);
            mma_commit(bar_mma);
        }
        // ---- rotate the pipeline registers
        prev = cur;
        sw_prev = sw_cur;
        sgp_c = sgp_n1; ul_c = ul_n1; nrm_c = nrm_n1;
#pragma unroll
        for (int w = 0; w < E8_NW; ++w) Uw[w] = Un[w];
#pragma unroll
        for (int j = 0; j < 4 * K; ++j) Rw[j] = Rn[j];
        sgp_n1 = sgp_n2; ul_n1 = ul_n2; nrm_n1 = nrm_n2;
        if (!nx1.valid) {  // drain: the last tile's epilogue
            mbar_wait(bar_mma, (uint32_t)(tau & 1));
            tc_fence_after();
            epilogue(prev, tau);
            break;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (tid < 32) tmem_dealloc(*tmem_slot, TCOLS);
}

template <int NB>
constexpr size_t e8_smem_bytes() {
    return 1024 + (size_t)E8_LUT_BYTES +
           (size_t)E8_NWG * ((16384 + 2 * e8_bslot_bytes(NB) + 128 * E8_SCR_STRIDE * 4 + 1023u) & ~1023u) + 8 * (E8_NWG * 3) + 16;
}

}  // namespace hq
