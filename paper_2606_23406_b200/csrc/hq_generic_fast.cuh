// hq_generic_fast.cuh — row decoders for the lattices / tiles the E8-tile-128 kernels do not take (SURVEY §8(a) A4-A5 for
// Z, A2, D4 and for E8 at tiles 64 / 256 below 64 activation rows; BASELINE config 3).
//
// Phase 1 is hq_e8_decode.cuh's (the unary section is lattice independent: a byte table of terminator positions, nibble
// stream in shared memory).  Phase 2 per lattice:
//   Z, E8 : one Rice class, so the R-section's field planes line up with the stream positions exactly as in the E8
//           kernel: e8_run's SWAR gap + remainder merge gives zz for four symbols per register; Z un-zig-zags byte-
//           parallel, E8 un-strips byte-parallel (e8_run), and byte permutes bring the codes to natural coordinate order
//           (the operand order of k_linear_generic's activation tile);
//   A2, D4: two classes with different k: the SWAR gaps give q per stream position, the remainder of every symbol is
//           picked from its class's field planes (all positions are compile-time constants inside a super-chunk of
//           64 / 128 symbols), un-strip per lattice block (hq_common.cuh).
// A row is declined (false; the caller falls back to decode_row_generic) if it has a quotient >= 16, more U words than
// the caller gathered, k > 3 (Z, E8), or - D4 at tile 64 - a partial class chunk.
#pragma once
#include "hq_common.cuh"
#include "hq_e8_decode.cuh"
#include "hq_tc.cuh"

namespace hq {

// phase 1 over a row's gathered U words (shared memory, zero padded past the row's end); returns the nibble count * 4
__device__ __forceinline__ uint32_t gf_phase1(const uint32_t* urow, uint32_t nw, uint32_t lut_a, uint32_t scr_a) {
    uint32_t T = 0, acc = 0, wo = scr_a;
    for (uint32_t w = 0; w < nw; ++w) e8_unary_word<1>(urow[w], lut_a, T, acc, wo);
    return T;
}

// SWAR gaps of one run of 32 stream positions: Q[2w + e] byte b = quotient of stream position 8w + 2b + e
__device__ __forceinline__ void gf_gaps(const uint32_t* W, uint32_t& prevWo, uint32_t& qsum, uint32_t* Q) {
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t We = W[w] & 0x0f0f0f0fu, Wo = (W[w] >> 4) & 0x0f0f0f0fu;
        const uint32_t prev = __funnelshift_l(prevWo, Wo, 8);
        Q[2 * w] = (We + 0x1f1f1f1fu - prev) & 0x0f0f0f0fu;
        Q[2 * w + 1] = (Wo + 0x1f1f1f1fu - We) & 0x0f0f0f0fu;
        prevWo = Wo;
        qsum = __dp4a(Q[2 * w], 0x01010101u, qsum);
        qsum = __dp4a(Q[2 * w + 1], 0x01010101u, qsum);
    }
}

// Z and E8: `store(word_index, value)` receives the row's codes four per word in natural coordinate order
template <int LAT, int K, class Store>
__device__ __forceinline__ bool gf_row_one_class(int n, uint32_t ulen, const uint32_t* rarea, int lane, uint32_t scr_a, Store store) {
    static_assert(LAT == LAT_Z || LAT == LAT_E8, "single Rice class");
    uint32_t prevWo = 15u << 24, total = 0;
    for (int c = 0; c < n / 32; ++c) {
        uint32_t W[4], V[K > 0 ? K : 1];
#pragma unroll
        for (int w = 0; w < 4; ++w) W[w] = lds32(scr_a + (c * 4 + w) * 4);
#pragma unroll
        for (int j = 0; j < K; ++j) V[j] = __ldg(rarea + (c * K + j) * 32 + lane);
        if (LAT == LAT_E8) {
            uint32_t C[8];
            e8_run<K>(W, V, prevWo, total, C);
            // C[i] byte b = coordinate i of block 4c + b  ->  block-major words: 4 x 4 byte transposes
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
                const uint32_t t0 = __byte_perm(C[4 * hh], C[4 * hh + 1], 0x5140), t1 = __byte_perm(C[4 * hh + 2], C[4 * hh + 3], 0x5140);
                const uint32_t t2 = __byte_perm(C[4 * hh], C[4 * hh + 1], 0x7362), t3 = __byte_perm(C[4 * hh + 2], C[4 * hh + 3], 0x7362);
                store(8 * c + 0 + hh, __byte_perm(t0, t1, 0x5410));   // block 4c,   coordinates 4hh .. 4hh + 3
                store(8 * c + 2 + hh, __byte_perm(t0, t1, 0x7632));   // block 4c+1
                store(8 * c + 4 + hh, __byte_perm(t2, t3, 0x5410));   // block 4c+2
                store(8 * c + 6 + hh, __byte_perm(t2, t3, 0x7632));   // block 4c+3
            }
        } else {
            uint32_t Q[8];
            gf_gaps(W, prevWo, total, Q);
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                uint32_t cz[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const uint32_t z = Q[2 * w + e] * (1u << K) + e8_rem4<K>(V, 2 * w + e);   // zig-zagged code, four stream positions
                    const uint32_t fill = (z & 0x01010101u) * 0xffu;
                    cz[e] = ((z >> 1) & 0x7f7f7f7fu) ^ fill;                                   // c = (z >> 1) ^ -(z & 1)
                }
                // stream position 8w + 2b + e = coordinate: interleave the even and odd registers
                store(8 * c + 2 * w, __byte_perm(cz[0], cz[1], 0x5140));
                store(8 * c + 2 * w + 1, __byte_perm(cz[0], cz[1], 0x7362));
            }
        }
    }
    return total + (uint32_t)n == ulen;   // else a quotient >= 16 aliased
}

// A2 and D4: two Rice classes (FORMAT §3), any k0, k1 <= 7.
template <int LAT, class Store>
__device__ __forceinline__ bool gf_row_two_class(int n, uint32_t ulen, int k0, int k1, const uint32_t* rarea, int lane,
                                                 uint32_t scr_a, Store store) {
    static_assert(LAT == LAT_A2 || LAT == LAT_D4, "two Rice classes");
    constexpr int SC = LAT == LAT_A2 ? 64 : 128;        // stream positions per super-chunk: whole class chunks of 32
    constexpr int NR = SC / 32;                         // runs of 32 positions
    constexpr int NC0 = LAT == LAT_A2 ? 1 : 3;          // class-0 chunks per super-chunk (class 1: one)
    const int base1 = class_count(LAT, n, 0) * k0 / 32; // first R word of class 1
    uint32_t prevWo = 15u << 24, total = 0;
    for (int sc = 0; sc < n / SC; ++sc) {
        uint32_t Q[NR][8];
#pragma unroll
        for (int r = 0; r < NR; ++r) {
            uint32_t W[4];
#pragma unroll
            for (int w = 0; w < 4; ++w) W[w] = lds32(scr_a + ((sc * NR + r) * 4 + w) * 4);
            gf_gaps(W, prevWo, total, Q[r]);
        }
        // field planes of the super-chunk's class chunks: width 1 (if k & 1: one word), width 2 (if k & 2: two words),
        // width 4 (if k & 4: four words), in that order (FORMAT §4)
        uint32_t P0[NC0 + 1], P1[NC0 + 1][2], P2[NC0 + 1][4];
#pragma unroll
        for (int cc = 0; cc <= NC0; ++cc) {
            const bool c1 = cc == NC0;
            const int ka = c1 ? k1 : k0;
            const int wb = c1 ? base1 + sc * k1 : (sc * NC0 + cc) * k0;
            P0[cc] = (ka & 1) ? __ldg(rarea + wb * 32 + lane) : 0u;
            P1[cc][0] = (ka & 2) ? __ldg(rarea + (wb + (ka & 1)) * 32 + lane) : 0u;
            P1[cc][1] = (ka & 2) ? __ldg(rarea + (wb + (ka & 1) + 1) * 32 + lane) : 0u;
#pragma unroll
            for (int j = 0; j < 4; ++j) P2[cc][j] = (ka & 4) ? __ldg(rarea + (wb + (ka & 1) + (ka & 2) + j) * 32 + lane) : 0u;
        }
#pragma unroll
        for (int s0 = 0; s0 < SC; s0 += 4) {             // four stream positions = four codes = one output word
            int z[4], c[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int s = s0 + i;
                const int a = sym_class(LAT, s);
                const int ms = LAT == LAT_A2 ? (s >> 1) : (a ? (s >> 2) : 3 * (s >> 2) + (s & 3));   // index inside the class
                const int cc = a ? NC0 : (ms >> 5), u = ms & 31;
                const int g = 2 * (u >> 3) + (u & 1), ln = (u & 7) >> 1;
                const uint32_t f0 = (P0[cc] >> (8 * ln + g)) & 1u;
                const uint32_t f1 = (P1[cc][g >> 2] >> (8 * ln + 2 * (g & 3))) & 3u;
                const uint32_t f2 = (P2[cc][g >> 1] >> (8 * ln + 4 * (g & 1))) & 15u;
                const int ka = a ? k1 : k0;
                const uint32_t r = f0 | (f1 << (ka & 1)) | (f2 << (ka & 3));
                const uint32_t q = (Q[s >> 5][2 * ((s >> 3) & 3) + (s & 1)] >> (8 * ((s >> 1) & 3))) & 0xffu;
                z[i] = (int)((q << (a ? k1 : k0)) | r);
            }
            if (LAT == LAT_D4) {
                unstrip<LAT_D4>(z, c);
            } else {
                unstrip<LAT_A2>(z, c);
                unstrip<LAT_A2>(z + 2, c + 2);
            }
            store((sc * SC + s0) >> 2, (uint32_t)(uint8_t)(int8_t)c[0] | ((uint32_t)(uint8_t)(int8_t)c[1] << 8) |
                                           ((uint32_t)(uint8_t)(int8_t)c[2] << 16) | ((uint32_t)(uint8_t)(int8_t)c[3] << 24));
        }
    }
    return total + (uint32_t)n == ulen;
}

// one row, any supported combination; `urow` = the row's first `cap` U words in shared memory
template <int LAT, class Store>
__device__ __forceinline__ bool decode_row_fast(const uint32_t* urow, uint32_t cap, uint32_t ulen, const uint32_t* rarea, int lane,
                                                int n, int k0, int k1, uint32_t lut_a, uint32_t scr_a, Store store) {
    const uint32_t nw = (ulen + 31) >> 5;
    if (nw > cap || k0 > 7 || k1 > 7 || ((LAT == LAT_Z || LAT == LAT_E8) && k0 > 3)) return false;
    if (LAT == LAT_D4 && n < 128) return false;                          // partial class chunks (FORMAT §4)
    if (gf_phase1(urow, nw, lut_a, scr_a) != 4u * (uint32_t)n) return false;   // a valid row has exactly n terminators
    if constexpr (LAT == LAT_Z || LAT == LAT_E8) {
        switch (k0) {
            case 0: return gf_row_one_class<LAT, 0>(n, ulen, rarea, lane, scr_a, store);
            case 1: return gf_row_one_class<LAT, 1>(n, ulen, rarea, lane, scr_a, store);
            case 2: return gf_row_one_class<LAT, 2>(n, ulen, rarea, lane, scr_a, store);
            default: return gf_row_one_class<LAT, 3>(n, ulen, rarea, lane, scr_a, store);
        }
    } else {
        return gf_row_two_class<LAT>(n, ulen, k0, k1, rarea, lane, scr_a, store);
    }
}

}  // namespace hq
