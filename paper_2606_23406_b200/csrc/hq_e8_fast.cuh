// hq_e8_fast.cuh — the fast per-row decoder for E8 tiles (hard part H1).
//
// One lane owns one row of a group (its tile of n symbols).  Two phases, both branch-light:
//
//  phase 1 (unary, §3.3): the row's U-section is walked 8 stream bits at a time.  A 256-entry
//    table maps a byte to the positions (mod 16, one nibble each, in order) of its one bits — each
//    one bit terminates a symbol.  The nibbles are appended to a per-row nibble stream in shared
//    memory (8 symbols = one E8 block per 32-bit word) with a shift/funnel pair; no per-symbol loop,
//    no clz.  The unary quotient of symbol j is the gap between consecutive terminators:
//    q_j = (e_j - e_{j-1} - 1) mod 16, exact for q <= 15.
//  phase 2 (remainders + un-strip, §4.6): per block, SWAR on 4 symbols per 32-bit register:
//    nibble -> byte unpack (even / odd symbols), gap, z = (q << k) | r with r taken from the R-section
//    field planes (FORMAT §4: one shift + one mask per 4 symbols), then the E8 un-strip
//    c_i = 2 s_i + coset, s_7 = 2t + parity, all byte-parallel.
//  A row whose quotients do not sum to its ulen (some q >= 16: ~1e-6 per symbol) is re-decoded by
//  the generic decoder.
//
// Output order inside a block is (c0,c2,c4,c6,c1,c3,c5,c7): the activation operand is permuted the
// same way, so INT32 accumulators are unchanged.
#pragma once
#include "hq_common.cuh"

namespace hq {

// table entry for stream byte `b` (bit 7 first) and piece parity: nibble j = position of the j-th one + 8*par
__device__ inline uint32_t unary_lut_entry(uint32_t b, uint32_t par) {
    uint32_t v = 0, j = 0;
#pragma unroll
    for (int pos = 0; pos < 8; ++pos)
        if (b & (0x80u >> pos)) { v |= (uint32_t)(pos + 8 * par) << (4 * j); ++j; }
    return v;
}
// lut: 512 words in shared memory; call with all threads of the block, then __syncthreads()
__device__ inline void build_unary_lut(uint32_t* lut, int tid, int nthreads) {
    for (int i = tid; i < 512; i += nthreads) lut[i] = unary_lut_entry(i & 255, i >> 8);
}

// phase 1: U-section [ustart, ustart+ulen) of `uarea` -> nibble words scr[0 .. n/8)
__device__ __forceinline__ void e8_unary_to_nibbles(const uint32_t* __restrict__ uarea, uint32_t ustart, uint32_t ulen,
                                                    const uint32_t* __restrict__ lut, uint32_t* __restrict__ scr) {
    const uint32_t wi = ustart >> 5, bo = ustart & 31;
    uint32_t hi = uarea[wi];
    uint32_t acc = 0, fs = 0;
    uint32_t* wo = scr;
    const int nch = (int)((ulen + 31) >> 5);
    for (int t = 0; t < nch; ++t) {
        const uint32_t lo = uarea[wi + t + 1];
        uint32_t x = __funnelshift_l(lo, hi, bo);
        hi = lo;
        const uint32_t rem = ulen - 32u * (uint32_t)t;
        if (rem < 32u) x &= ~(0xffffffffu >> rem);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint32_t byte = (x >> (24 - 8 * i)) & 0xffu;
            const uint32_t N = lut[(i & 1) * 256 + byte];
            const uint32_t c4 = 4u * (uint32_t)__popc(byte);
            const uint32_t out0 = acc | (N << fs);
            const uint32_t out1 = __funnelshift_l(N, 0u, fs);  // bits of N shifted out past bit 31
            const uint32_t fs2 = fs + c4;
            const bool full = fs2 >= 32u;
            if (full) *wo++ = out0;
            acc = full ? out1 : out0;
            fs = fs2 & 31u;
        }
    }
    if (fs) *wo = acc;
}

// the K-bit remainders of the even (par=0) / odd (par=1) symbols of block `blk_in_chunk` (0..3) of a
// 32-symbol chunk whose K field-plane words are V[0..K)  (FORMAT §4)
template <int K>
__device__ __forceinline__ uint32_t e8_rem4(const uint32_t* V, int blk_in_chunk, int par) {
    uint32_t r = 0;
    int lo = 0;
    const int g = 2 * blk_in_chunk + par;
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

// phase 2 for one block: nibble word W (+ previous block's odd-position word) -> (c_even4, c_odd4)
// qsum accumulates qe+qo byte-wise (caller widens every <= 8 blocks).
template <int K>
__device__ __forceinline__ void e8_block(uint32_t W, uint32_t& prevWo, uint32_t re, uint32_t ro, uint32_t& qsum,
                                         uint32_t& ce, uint32_t& co) {
    const uint32_t We = W & 0x0f0f0f0fu, Wo = (W >> 4) & 0x0f0f0f0fu;
    const uint32_t prev = __funnelshift_l(prevWo, Wo, 8);  // (Wo << 8) | (prevWo >> 24)
    const uint32_t qe = (We + 0x1f1f1f1fu - prev) & 0x0f0f0f0fu;
    const uint32_t qo = (Wo + 0x1f1f1f1fu - We) & 0x0f0f0f0fu;
    prevWo = Wo;
    qsum += qe + qo;
    const uint32_t ze = qe * (1u << K) + re, zo = qo * (1u << K) + ro;
    // un-strip (§4.6): zo byte 3 is comb = 2*zigzag(t) + coset (L274); every other byte is zigzag(s_i)
    const uint32_t coset4 = __byte_perm(zo, 0u, 0x3333) & 0x01010101u;
    const uint32_t sgn_e = ze & 0x01010101u;
    const uint32_t sgn_o = (zo & 0x00010101u) | ((zo >> 1) & 0x01000000u);
    const uint32_t neg_e = sgn_e * 0xfeu + coset4;
    const uint32_t neg_o = sgn_o * 0xfeu + coset4;
    ce = (ze & 0xfefefefeu) ^ neg_e;                 // 2 s_i + coset
    uint32_t t = (zo & 0xfcfefefeu) ^ neg_o;          // byte 3: 4t + coset (bit 1 to be replaced by the parity)
    const uint32_t par = (((ce ^ (t & 0x00ffffffu)) & 0x02020202u) * 0x01010101u) & 0x02000000u;  // (sum_{i<7} s_i)&1 at bit 25
    co = (t & ~0x02000000u) | par;
}

// Fast decode of one row.  R-section words of the row: rrow[0 .. n*K/32) (word aligned: n*K % 32 == 0).
// emit(b, ce, co) receives block b's eight INT8 codes as two words, order (c0,c2,c4,c6),(c1,c3,c5,c7).
// Returns false if the row needs the generic decoder (a quotient >= 16).
template <int K, class Emit>
__device__ __forceinline__ bool e8_decode_row_fast(const uint32_t* __restrict__ uarea, uint32_t ustart, uint32_t ulen,
                                                   const uint32_t* __restrict__ rrow, const uint32_t* __restrict__ lut,
                                                   uint32_t* __restrict__ scr, int n, Emit emit) {
    e8_unary_to_nibbles(uarea, ustart, ulen, lut, scr);
    uint32_t prevWo = 15u << 24;  // e_{-1} = -1 mod 16
    uint32_t total = 0;
    const int nchunk = n / 32;
    for (int ch = 0; ch < nchunk; ++ch) {
        uint32_t V[K > 0 ? K : 1];
#pragma unroll
        for (int i = 0; i < K; ++i) V[i] = rrow[ch * K + i];
        uint32_t qsum = 0;
#pragma unroll
        for (int bl = 0; bl < 4; ++bl) {
            const uint32_t W = scr[ch * 4 + bl];
            uint32_t ce, co;
            e8_block<K>(W, prevWo, e8_rem4<K>(V, bl, 0), e8_rem4<K>(V, bl, 1), qsum, ce, co);
            emit(ch * 4 + bl, ce, co);
        }
        total += __dp4a(qsum, 0x01010101u, 0u);  // byte sums (<= 4*30 per byte lane) widened
    }
    return total + (uint32_t)n == ulen;
}

}  // namespace hq
