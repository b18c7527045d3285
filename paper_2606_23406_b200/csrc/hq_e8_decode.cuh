// hq_e8_decode.cuh — the fast E8 tile decoder (hard part H1).
//
// One lane owns one row of a sub-group (FORMAT §5): its U words and R words arrive in registers by
// coalesced loads.  Two phases, both branch-free in the common case:
//
//  phase 1 (unary, §3.3): the row's U-section is walked 8 stream bits at a time.  A 256-entry table
//    maps a byte to the positions (mod 16, one nibble each, in order) of its one bits — every one bit
//    terminates a symbol.  The nibbles are appended to a per-row nibble stream in shared memory
//    (8 symbols per 32-bit word); no per-symbol loop, no clz.
//  phase 2 (remainders + un-strip, §4.6): per run of 32 symbols = four E8 blocks in FORMAT §3's
//    coordinate-pair order.  The unary quotient of a symbol is the gap between consecutive terminators,
//    q_j = (e_j - e_{j-1} - 1) mod 16 (exact for q <= 15); all further steps are SWAR on one register of
//    four bytes = ONE coordinate of FOUR blocks: z = (q << k) | r with r from the R-section field planes
//    (one shift + one mask per 4 symbols), c_i = (z ^ signfill) | coset, the block parity as a 7-input
//    XOR, the comb symbol (coordinate 7) as one more register.
//  A row with a quotient >= 16 or more than NW words is flagged and re-decoded by the generic decoder.
//
// Output: per run c, registers C[0..7], byte b of C[i] = code c_i of block 4c + b: the A operand's K
// index inside the tile is 32c + 4i + b, and the activation operand is stored in the same order.
#pragma once
#include "hq_common.cuh"
#include "hq_tc.cuh"

namespace hq {

constexpr int E8_LUT_COPIES = 16;                                  // replicas per entry: lane l uses copy l & 15
constexpr int E8_LUT_WORDS = 2 * 256 * E8_LUT_COPIES;              // [parity][byte][copy]
constexpr int E8_LUT_BYTES = E8_LUT_WORDS * 4;                     // 32 KB

// table entry for stream byte `b` (bit 7 first) and byte parity: nibble j = position of the j-th one + 8*par
__host__ __device__ inline uint32_t unary_lut_entry(uint32_t b, uint32_t par) {
    uint32_t v = 0, j = 0;
    for (int pos = 0; pos < 8; ++pos)
        if (b & (0x80u >> pos)) { v |= (uint32_t)(pos + 8 * par) << (4 * j); ++j; }
    return v;
}

// phase 1 for one stream word x (4 bytes, byte 0 = bits 31..24).  `lut_lane` = shared-space address of this
// lane's copy of entry 0 / parity 0.  State: T = 4 * (terminators seen so far in the row) = bit position in the
// nibble stream, acc = the partial nibble word, wo = shared-space address of the next nibble word of this row.
// Every shift amount and every "word completed" predicate comes from prefix popcounts of x, so the only
// loop-carried values are acc (one select per byte) and wo (one predicated add per byte).
// nbytes (warp-uniform, 1..4): only the first nbytes stream bytes of x can hold terminators (the tail words of a row)
template <int COPIES = E8_LUT_COPIES>
__device__ __forceinline__ void e8_unary_word(uint32_t x, uint32_t lut_lane, uint32_t& T, uint32_t& acc, uint32_t& wo,
                                              int nbytes = 4) {
    // The ALU pipe (LOP3 / SHF / SEL, half rate) is the busiest unit of this kernel: the byte-prefix shift, shared by
    // the table index and the prefix popcount, is taken as the high half of a multiply (FMA pipe).  (Doing the
    // variable shifts of the append as multiplies too was measured slower: IMAD.HI is quarter rate.)
    uint32_t N[4], Te[4];
    if (nbytes < 4) {   // tail word: byte by byte (a skipped byte is zero: it would append nothing)
        uint32_t Tb = T;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            if (i < nbytes) {
                const uint32_t pre = __umulhi(x, 1u << (8 + 8 * i));
                const uint32_t sel = (pre * (uint32_t)(COPIES * 4)) & (uint32_t)(0xff * COPIES * 4);
                const uint32_t Ni = lds32_ro(lut_lane + sel + ((i & 1) ? 256 * COPIES * 4 : 0));
                const uint32_t Tei = T + 4u * (uint32_t)__popc(pre);
                const uint32_t out0 = acc | __funnelshift_l(0u, Ni, Tb);
                const uint32_t out1 = __funnelshift_l(Ni, 0u, Tb);
                const bool full = ((Tei ^ Tb) & 32u) != 0u;
                if (full) { sts32(wo, out0); wo += 4; }
                acc = full ? out1 : out0;
                Tb = Tei;
            }
        }
        T = Tb;
        return;
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t pre = (i < 3) ? __umulhi(x, 1u << (8 + 8 * i)) : x;   // x >> (24 - 8i): bytes 0..i
        const uint32_t sel = (pre * (uint32_t)(COPIES * 4)) & (uint32_t)(0xff * COPIES * 4);   // byte i * entry stride
        N[i] = lds32_ro(lut_lane + sel + ((i & 1) ? 256 * COPIES * 4 : 0));
        Te[i] = T + 4u * (uint32_t)__popc(pre);   // nibble-stream position after byte i
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t Tb = i ? Te[i - 1] : T;                  // position before byte i
        const uint32_t out0 = acc | __funnelshift_l(0u, N[i], Tb);   // N << (Tb & 31)
        const uint32_t out1 = __funnelshift_l(N[i], 0u, Tb);         // the bits of N shifted out past bit 31
        const bool full = ((Te[i] ^ Tb) & 32u) != 0u;           // this byte completed a 32-bit nibble word
        if (full) { sts32(wo, out0); wo += 4; }
        acc = full ? out1 : out0;
    }
    T = Te[3];
}

// the K-bit remainders of symbol group g (0..7 = coordinate) of a 32-symbol run whose K field-plane words are
// V[0..K)  (FORMAT §4): byte b = block b of the run
template <int K>
__device__ __forceinline__ uint32_t e8_rem4(const uint32_t* V, int g) {
    uint32_t r = 0;
    int lo = 0;
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const int wd = 1 << b;
        if (!(K & wd)) continue;
        const int per = 8 / wd;
        const uint32_t mask = ((1u << wd) - 1u) * 0x01010101u;
        r |= ((V[lo + g / per] >> (wd * (g % per))) & mask) << lo;
        lo += wd;
    }
    return r;
}

// phase 2 for one run of 32 symbols: nibble words W[0..3], remainder words V[0..K) -> C[0..7].
// prevWo carries the last odd-position word (for the gap of the next even positions); qsum accumulates
// the quotients of the row.
template <int K>
__device__ __forceinline__ void e8_run(const uint32_t* W, const uint32_t* V, uint32_t& prevWo, uint32_t& qsum, uint32_t* C) {
    uint32_t Z[8];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t We = W[w] & 0x0f0f0f0fu, Wo = (W[w] >> 4) & 0x0f0f0f0fu;
        const uint32_t prev = __funnelshift_l(prevWo, Wo, 8);  // (Wo << 8) | (prevWo >> 24)
        const uint32_t qe = (We + 0x1f1f1f1fu - prev) & 0x0f0f0f0fu;
        const uint32_t qo = (Wo + 0x1f1f1f1fu - We) & 0x0f0f0f0fu;
        prevWo = Wo;
        qsum = __dp4a(qe, 0x01010101u, qsum);
        qsum = __dp4a(qo, 0x01010101u, qsum);
        Z[2 * w] = qe * (1u << K) + e8_rem4<K>(V, 2 * w);
        Z[2 * w + 1] = qo * (1u << K) + e8_rem4<K>(V, 2 * w + 1);
    }
    // un-strip (§4.6): Z[7] is comb = 2*zigzag(t) + coset (L274); every other Z[i] is zigzag(s_i)
    const uint32_t coset4 = Z[7] & 0x01010101u;
    uint32_t P = 0;
#pragma unroll
    for (int i = 0; i < 7; ++i) {
        const uint32_t fill = (Z[i] & 0x01010101u) * 0xffu;
        const uint32_t c2 = Z[i] ^ fill;  // 2 s_i (bit 0 clear)
        P ^= c2;
        C[i] = c2 | coset4;               // c_i = 2 s_i + coset
    }
    const uint32_t zt = (Z[7] >> 1) & 0x7f7f7f7fu;            // zigzag(t)
    const uint32_t t2 = zt ^ ((zt & 0x01010101u) * 0xffu);     // 2 t
    C[7] = ((t2 << 1) & 0xfefefefeu) | (P & 0x02020202u) | coset4;  // c_7 = 4 t + 2 parity + coset
}

// ---------------------------------------------------------------------------------------------
// The same decoder for one KV vector (FORMAT §6): 128 symbols, U-section = `ulen` bits starting at bit `upos` of the
// contiguous MSB-first word array `una` (the next vector's bits follow: the tail is masked), R-section = 4K words at
// rrow.  lut = shared-space address of an un-replicated table [2][256]; scr_a = 17 words of per-thread scratch.
// out(blk, c[8]) receives the blocks in order.  Returns false (nothing emitted) if the row needs the generic decoder.
// ---------------------------------------------------------------------------------------------
template <int K, class Out>
__device__ __forceinline__ bool e8_decode_row_kv(const uint32_t* __restrict__ una, uint32_t upos, uint32_t ulen,
                                                 const uint32_t* __restrict__ rrow, uint32_t lut, uint32_t scr_a, Out out) {
    const uint32_t nw = (ulen + 31) >> 5;
    if (nw > 16u) return false;
    uint32_t T = 0, acc = 0, wo = scr_a;
    {
        const uint32_t wi = upos >> 5, sh = upos & 31;
        uint32_t hi = __ldg(una + wi);
        for (uint32_t w = 0; w < nw; ++w) {
            const uint32_t lo = __ldg(una + wi + w + 1);
            uint32_t x = __funnelshift_l(lo, hi, sh);
            hi = lo;
            const uint32_t rem = ulen - 32u * w;
            if (rem < 32u) x &= ~(0xffffffffu >> rem);
            e8_unary_word<1>(x, lut, T, acc, wo);
        }
    }
    if (T != 4u * 128u) return false;   // a valid row has exactly 128 terminators
    uint32_t V[4 * (K > 0 ? K : 1)];
#pragma unroll
    for (int j = 0; j < 4 * K; ++j) V[j] = __ldg(rrow + j);
    uint32_t prevWo = 15u << 24, total = 0;
    uint32_t Cs[4][8];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        uint32_t W[4];
#pragma unroll
        for (int w = 0; w < 4; ++w) W[w] = lds32(scr_a + (c * 4 + w) * 4);
        e8_run<K>(W, V + c * K, prevWo, total, Cs[c]);
    }
    if (total + 128u != ulen) return false;   // a quotient >= 16 aliased
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            int cc[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) cc[i] = (int)(int8_t)(Cs[c][i] >> (8 * b));
            out(4 * c + b, cc);
        }
    return true;
}

}  // namespace hq
