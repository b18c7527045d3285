// hq_common.cuh — device helpers shared by the CUDA translation units of libhq.so.
//
// Written from docs/FORMAT.md and the paper (PAPER.md line numbers cited); shares nothing with
// oracle/.  Everything that decides an integer (RHT, norm, nearest point) is IEEE binary32 with
// explicit __f*_rn intrinsics so that no FMA contraction can change a rounding (FORMAT §2).
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace hq {

constexpr int LAT_Z = 1, LAT_A2 = 2, LAT_D4 = 4, LAT_E8 = 8;
constexpr int ROWS_PER_GROUP = 128;  // FORMAT §5: a group is 128 rows x one K-tile

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 counter RNG (FORMAT §1; Salmon et al. SC'11).
// ---------------------------------------------------------------------------------------------
__host__ __device__ inline void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// sign bit of coordinate i in stream 1 (RHT D, eq.(1)) or 2 (KV rotation S, L216): 1 -> -1
__host__ __device__ inline int sign_bit(uint64_t seed, uint32_t stream, uint32_t i) {
    uint32_t o[4];
    philox4x32_10(i >> 7, 0u, 0u, stream, (uint32_t)seed, (uint32_t)(seed >> 32), o);
    return (o[(i >> 5) & 3] >> (i & 31)) & 1u;
}

// ---------------------------------------------------------------------------------------------
// fp16 storage of the norm (L500; FORMAT R3): RNE, saturating at 65504.
// ---------------------------------------------------------------------------------------------
__device__ inline uint16_t f32_to_f16_bits_sat(float f) {
    if (!(f == f)) return 0x7e00;
    float a = fabsf(f);
    uint16_t sign = (__float_as_uint(f) >> 31) ? 0x8000 : 0;
    if (a >= 65520.0f) return sign | 0x7bff;
    return __half_as_ushort(__float2half_rn(f));
}
__device__ inline float f16_bits_to_f32(uint16_t h) { return __half2float(__ushort_as_half(h)); }

// ---------------------------------------------------------------------------------------------
// Lattice constants.  M = G(Lambda) * V^(2/N) of the integer realizations (Table 2,
// covolumes from §4.5); alpha by eq.(9) L871.
// ---------------------------------------------------------------------------------------------
__host__ inline double second_moment(int lattice) {
    switch (lattice) {
        case LAT_Z: return 1.0 / 12.0;
        case LAT_A2: return 0.0802 * 2.0 * 1.7320508075688772935;
        case LAT_D4: return 0.0766 * 1.4142135623730950488;
        case LAT_E8: return 0.0717 * 4.0;
    }
    return 0.0;
}

__host__ __device__ inline int sym_class(int lattice, int j) {  // FORMAT §3
    if (lattice == LAT_D4) return (j & 3) == 3;
    if (lattice == LAT_A2) return j & 1;
    return 0;
}
__host__ __device__ inline int class_count(int lattice, int n, int a) {
    if (lattice == LAT_D4) return a ? n / 4 : 3 * n / 4;
    if (lattice == LAT_A2) return n / 2;
    return a ? 0 : n;
}
__host__ __device__ inline int rbits_of(int lattice, int n, int k0, int k1) {
    return class_count(lattice, n, 0) * k0 + class_count(lattice, n, 1) * k1;
}

#define HQ_S3 1.7320508075688772f  // (float)sqrt(3.0)

// ---------------------------------------------------------------------------------------------
// Nearest lattice point (§3.2, §4.5; FORMAT R5, R6), canonical fp32.
// ---------------------------------------------------------------------------------------------
template <int M>
__device__ inline void nearest_Dm(const float* z, int* f) {  // Conway-Sloane D_m
    float delta[M];
    int sum = 0;
#pragma unroll
    for (int i = 0; i < M; ++i) {
        float r = rintf(z[i]);
        f[i] = (int)r;
        delta[i] = __fsub_rn(z[i], r);
        sum += f[i];
    }
    if (sum & 1) {
        int j = 0;
        float best = fabsf(delta[0]);
#pragma unroll
        for (int i = 1; i < M; ++i) {
            float a = fabsf(delta[i]);
            if (a > best) { best = a; j = i; }
        }
#pragma unroll
        for (int i = 0; i < M; ++i)
            if (i == j) f[i] += (delta[i] < 0.0f) ? -1 : 1;
    }
}

template <int LAT>
__device__ inline void nearest_noclamp(const float* y, int* c) {
    if (LAT == LAT_Z) {
        c[0] = (int)rintf(y[0]);
    } else if (LAT == LAT_D4) {
        nearest_Dm<4>(y, c);
    } else if (LAT == LAT_E8) {
        float za[8], zb[8], da[8], db[8];
        int a[8], b[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            za[i] = __fmul_rn(y[i], 0.5f);
            zb[i] = __fmul_rn(__fsub_rn(y[i], 1.0f), 0.5f);
        }
        nearest_Dm<8>(za, a);
        nearest_Dm<8>(zb, b);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            a[i] = 2 * a[i];
            b[i] = 2 * b[i] + 1;
            float ea = __fsub_rn(y[i], (float)a[i]), eb = __fsub_rn(y[i], (float)b[i]);
            da[i] = __fmul_rn(ea, ea);
            db[i] = __fmul_rn(eb, eb);
        }
        // FORMAT R2 tree: adjacent pairs first
        float dist_a = __fadd_rn(__fadd_rn(__fadd_rn(da[0], da[1]), __fadd_rn(da[2], da[3])),
                                 __fadd_rn(__fadd_rn(da[4], da[5]), __fadd_rn(da[6], da[7])));
        float dist_b = __fadd_rn(__fadd_rn(__fadd_rn(db[0], db[1]), __fadd_rn(db[2], db[3])),
                                 __fadd_rn(__fadd_rn(db[4], db[5]), __fadd_rn(db[6], db[7])));
        bool pa = dist_a <= dist_b;
#pragma unroll
        for (int i = 0; i < 8; ++i) c[i] = pa ? a[i] : b[i];
    } else {  // A2: block (y, x) -> (n_y, n_x)
        const float s3 = HQ_S3, two_s3 = __fmul_rn(2.0f, HQ_S3);
        int ay = 2 * (int)rintf(__fdiv_rn(y[0], two_s3)), ax = 2 * (int)rintf(__fmul_rn(y[1], 0.5f));
        int by = 2 * (int)rintf(__fdiv_rn(__fsub_rn(y[0], s3), two_s3)) + 1;
        int bx = 2 * (int)rintf(__fmul_rn(__fsub_rn(y[1], 1.0f), 0.5f)) + 1;
        float eay = __fsub_rn(y[0], __fmul_rn(s3, (float)ay)), eax = __fsub_rn(y[1], (float)ax);
        float eby = __fsub_rn(y[0], __fmul_rn(s3, (float)by)), ebx = __fsub_rn(y[1], (float)bx);
        float dist_a = __fadd_rn(__fmul_rn(eay, eay), __fmul_rn(eax, eax));
        float dist_b = __fadd_rn(__fmul_rn(eby, eby), __fmul_rn(ebx, ebx));
        if (dist_a <= dist_b) { c[0] = ay; c[1] = ax; } else { c[0] = by; c[1] = bx; }
    }
}

// INT8 pre-clamp of the quantizer input (G8 / FORMAT R5); returns #coordinates changed.
template <int LAT>
__device__ inline int clamp_block(float* y) {
    int cnt = 0;
#pragma unroll
    for (int i = 0; i < LAT; ++i) {
        float lim = (LAT == LAT_E8) ? 125.0f : (LAT == LAT_Z) ? 127.0f : 126.0f;
        if (LAT == LAT_A2 && i == 0) lim = __fmul_rn(126.0f, HQ_S3);
        float v = y[i];
        if (v > lim) { v = lim; cnt++; }
        if (v < -lim) { v = -lim; cnt++; }
        y[i] = v;
    }
    return cnt;
}

// dither U = y - Q(y), y box-uniform over a fundamental domain of a rectangular sub-lattice
// (A.6 L843-847, Lemma 1; FORMAT R4).  w[] are the odd 24-bit integers of FORMAT §1.
template <int LAT>
__device__ inline void dither_from_uniforms(const uint32_t* w, float* U) {
    float y[LAT];
    int c[LAT];
#pragma unroll
    for (int j = 0; j < LAT; ++j) {
        float wf = (float)w[j];  // exact: < 2^24
        if (LAT == LAT_E8) y[j] = __fsub_rn(__fmul_rn(wf, 0x1p-22f), 2.0f);
        else if (LAT == LAT_D4) y[j] = __fsub_rn(__fmul_rn(wf, 0x1p-23f), 1.0f);
        else if (LAT == LAT_Z) y[j] = __fsub_rn(__fmul_rn(wf, 0x1p-24f), 0.5f);
        else {
            float t = __fsub_rn(__fmul_rn(wf, 0x1p-23f), 1.0f);
            y[j] = (j == 0) ? __fmul_rn(t, HQ_S3) : t;
        }
    }
    nearest_noclamp<LAT>(y, c);
#pragma unroll
    for (int j = 0; j < LAT; ++j) {
        float p = (float)c[j];
        if (LAT == LAT_A2 && j == 0) p = __fmul_rn(HQ_S3, p);
        U[j] = __fsub_rn(y[j], p);
    }
}

// the dim uniforms of lattice block `blk` of vector (token, head, role)  (FORMAT §1)
template <int LAT>
__device__ inline void dither_block(uint64_t seed, uint32_t blk, uint32_t token, uint32_t head,
                                    uint32_t role, float* U) {
    uint32_t w[LAT];
    uint32_t o[4];
    if (LAT == LAT_E8) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            philox4x32_10(2 * blk + h, token, head | (role << 16), 3u, (uint32_t)seed, (uint32_t)(seed >> 32), o);
#pragma unroll
            for (int j = 0; j < 4; ++j) w[4 * h + j] = 2u * (o[j] >> 9) + 1u;
        }
    } else {
        uint32_t e0 = (uint32_t)LAT * blk;  // LAT in {1,2,4}: all uniforms of the block share one counter
        philox4x32_10(e0 >> 2, token, head | (role << 16), 3u, (uint32_t)seed, (uint32_t)(seed >> 32), o);
#pragma unroll
        for (int j = 0; j < LAT; ++j) w[j] = 2u * (o[(e0 + j) & 3] >> 9) + 1u;
    }
    dither_from_uniforms<LAT>(w, U);
}

// ---------------------------------------------------------------------------------------------
// Strip / un-strip with zig-zag (§4.6; FORMAT §3).
// ---------------------------------------------------------------------------------------------
__device__ inline int zigzag(int v) { return v >= 0 ? 2 * v : -2 * v - 1; }
__device__ inline int unzigzag(int z) { return (z & 1) ? -((z + 1) >> 1) : (z >> 1); }

template <int LAT>
__device__ inline void strip(const int* c, int* z) {
    if (LAT == LAT_E8) {
        int coset = c[0] & 1, s[8], sum = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) s[i] = (c[i] - coset) >> 1;
#pragma unroll
        for (int i = 0; i < 7; ++i) sum += s[i];
        int p = sum & 1, t = (s[7] - p) >> 1;
#pragma unroll
        for (int i = 0; i < 7; ++i) z[i] = zigzag(s[i]);
        z[7] = 2 * zigzag(t) + coset;  // comb, L274
    } else if (LAT == LAT_D4) {
        int p = (c[0] + c[1] + c[2]) & 1, t = (c[3] - p) >> 1;
        z[0] = zigzag(c[0]); z[1] = zigzag(c[1]); z[2] = zigzag(c[2]); z[3] = zigzag(t);
    } else if (LAT == LAT_A2) {
        int p = c[1] & 1, ty = (c[0] - p) >> 1;
        z[0] = zigzag(ty); z[1] = zigzag(c[1]);
    } else {
        z[0] = zigzag(c[0]);
    }
}
template <int LAT>
__device__ inline void unstrip(const int* z, int* c) {
    if (LAT == LAT_E8) {
        int s[8], sum = 0, coset = z[7] & 1, t = unzigzag(z[7] >> 1);
#pragma unroll
        for (int i = 0; i < 7; ++i) { s[i] = unzigzag(z[i]); sum += s[i]; }
        s[7] = 2 * t + (sum & 1);
#pragma unroll
        for (int i = 0; i < 8; ++i) c[i] = 2 * s[i] + coset;
    } else if (LAT == LAT_D4) {
        c[0] = unzigzag(z[0]); c[1] = unzigzag(z[1]); c[2] = unzigzag(z[2]);
        c[3] = 2 * unzigzag(z[3]) + ((c[0] + c[1] + c[2]) & 1);
    } else if (LAT == LAT_A2) {
        c[1] = unzigzag(z[1]);
        c[0] = 2 * unzigzag(z[0]) + (c[1] & 1);
    } else {
        c[0] = unzigzag(z[0]);
    }
}

// ---------------------------------------------------------------------------------------------
// Stream order of a tile's symbols (FORMAT §3): position p -> block-major index blk*dim + i.
// E8: p = 32c + 8w + 2b + e  <->  block 4c + b, coordinate 2w + e; other lattices: identity.
// ---------------------------------------------------------------------------------------------
__host__ __device__ inline int stream_to_blockmajor(int lattice, int p) {
    if (lattice != LAT_E8) return p;
    int c = p >> 5, w = (p >> 3) & 3, b = (p >> 1) & 3, e = p & 1;
    return 8 * (4 * c + b) + 2 * w + e;
}

// ---------------------------------------------------------------------------------------------
// MSB-first bit streams over little-endian u32 words (FORMAT §4), read through a word accessor
// `word(i) -> uint32_t` (must return 0 past the end of the stream).
// ---------------------------------------------------------------------------------------------
struct WordsContig {  // a contiguous, padded word array
    const uint32_t* w;
    __device__ inline uint32_t operator()(uint32_t i) const { return w[i]; }
};
template <class W>
__device__ inline uint32_t get32(const W& word, uint32_t p) {  // 32 stream bits starting at bit p
    uint32_t i = p >> 5, s = p & 31;
    uint32_t hi = word(i), lo = word(i + 1);
    return __funnelshift_l(lo, hi, s);
}
template <class W>
__device__ inline uint32_t get_bits(const W& word, uint32_t p, int nb) {  // nb in [1,32], value MSB-first
    return get32(word, p) >> (32 - nb);
}

// the k-bit remainder of class-a symbol number m_idx (index within its class, stream order) of a tile
// whose R-section starts at stream bit rpos of `rword` (FORMAT §4 field planes). Generic (slow) path.
template <class W>
__device__ inline uint32_t get_remainder(const W& rword, uint32_t rpos, int lattice, int n, int k0, int k1, int a,
                                         int m_idx) {
    int ka = a ? k1 : k0;
    if (ka == 0) return 0;
    int na = class_count(lattice, n, a);
    uint32_t base = rpos + (a ? (uint32_t)(class_count(lattice, n, 0) * k0) : 0u);
    int ch = m_idx >> 5, u = m_idx & 31;
    int cnt = min(32, na - ch * 32);
    base += (uint32_t)(ch * 32 * ka);
    uint32_t r = 0;
    int lo = 0;
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        int wd = 1 << b;
        if (!(ka & wd)) continue;
        if (cnt == 32) {
            int per = 8 / wd, g = 2 * (u >> 3) + (u & 1), bl = (u & 7) >> 1;
            uint32_t V = get32(rword, base + (uint32_t)(32 * lo + 32 * (g / per)));
            r |= ((V >> (8 * bl + wd * (g % per))) & ((1u << wd) - 1u)) << lo;
        } else {
            r |= get_bits(rword, base + (uint32_t)(cnt * lo + u * wd), wd) << lo;
        }
        lo += wd;
    }
    return r;
}

// ---------------------------------------------------------------------------------------------
// Generic row decoder (any lattice / tile / k): U-section walked with clz, remainders by
// get_remainder, un-strip per lattice block; emits INT8 codes per block through `out(blk, c[LAT])`
// (blk = block-major block index).  Symbols arrive in stream order (FORMAT §3).
// ---------------------------------------------------------------------------------------------
template <class W>
struct UnaryReader {
    const W& word;
    uint32_t p, x;
    int avail;
    __device__ UnaryReader(const W& w, uint32_t p0) : word(w), p(p0), x(get32(w, p0)), avail(32) {}
    __device__ inline int next() {  // zeros up to the terminating one
        int q = 0;
        while (true) {
            if (x == 0) {
                q += avail; p += avail;
                x = get32(word, p); avail = 32;
                if (q > 70000) break;  // corrupt stream guard: stay bounded
                continue;
            }
            int lz = __clz(x);
            q += lz;
            int used = lz + 1;
            x = (used >= 32) ? 0u : (x << used);
            avail -= used; p += used;
            if (avail == 0) { x = get32(word, p); avail = 32; }
            break;
        }
        return q;
    }
};

template <int LAT, class RW, class UW, class Out>
__device__ inline void decode_row_generic(const RW& rword, uint32_t rpos, const UW& uword, uint32_t upos, int n,
                                          int k0, int k1, Out out) {
    UnaryReader<UW> ur(uword, upos);
    int cls_idx[2] = {0, 0};
    if (LAT == LAT_E8) {
        for (int ch = 0; ch < n / 32; ++ch) {
            int zc[32];
            for (int u = 0; u < 32; ++u) {
                int q = ur.next();
                uint32_t r = get_remainder(rword, rpos, LAT_E8, n, k0, k1, 0, ch * 32 + u);
                zc[u] = (q << k0) | (int)r;
            }
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                int z[8], c[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) z[i] = zc[8 * (i >> 1) + 2 * b + (i & 1)];
                unstrip<LAT_E8>(z, c);
                out(4 * ch + b, c);
            }
        }
    } else {
        for (int b = 0; b < n / LAT; ++b) {
            int z[LAT], c[LAT];
#pragma unroll
            for (int i = 0; i < LAT; ++i) {
                int j = b * LAT + i;
                int q = ur.next();
                int a = sym_class(LAT, j);
                int ka = a ? k1 : k0;
                uint32_t r = get_remainder(rword, rpos, LAT, n, k0, k1, a, cls_idx[a]);
                cls_idx[a]++;
                z[i] = (q << ka) | (int)r;
            }
            unstrip<LAT>(z, c);
            out(b, c);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Weight sub-group access (FORMAT §5): 32 rows, lane i = row i.
// ---------------------------------------------------------------------------------------------
struct SubGroup {
    const uint16_t* ulen;   // [32]
    const uint16_t* norm;   // [32]
    const uint32_t* rarea;  // [RW*32], word j of row i at j*32 + i
    const uint32_t* uarea;  // compacted word-rows
};
__device__ inline SubGroup sub_group(const uint8_t* base, int rw_words) {
    SubGroup s;
    s.ulen = (const uint16_t*)base;
    s.norm = s.ulen + 32;
    s.rarea = (const uint32_t*)(base + 128);
    s.uarea = s.rarea + rw_words * 32;
    return s;
}
// index (in uarea) of word t of row i, by scanning the header: sum_i' min(nw_i', t) + #{i' < i : nw_i' > t}
__device__ inline uint32_t u_word_index_slow(const uint16_t* ulen_hdr, int i, uint32_t t) {
    uint32_t at = 0;
    for (int r = 0; r < 32; ++r) {
        uint32_t nw = ((uint32_t)ulen_hdr[r] + 31u) >> 5;
        at += min(nw, t);
        if (r < i && nw > t) ++at;
    }
    return at;
}
// Warp-synchronous gather of every lane's first min(nw, cap) U words into row[0..cap) (row = this lane's
// scratch, any memory space).  All 32 lanes must call it.
__device__ inline void gather_u_words(const uint32_t* uarea, uint32_t nw, int lane, uint32_t* row, uint32_t cap) {
    uint32_t maxnw = nw;
#pragma unroll
    for (int o = 16; o; o >>= 1) maxnw = max(maxnw, __shfl_xor_sync(0xffffffffu, maxnw, o));
    uint32_t base = 0;
    for (uint32_t t = 0; t < min(maxnw, cap); ++t) {
        const bool has = nw > t;
        const uint32_t m = __ballot_sync(0xffffffffu, has);
        if (has) row[t] = uarea[base + __popc(m & ((1u << lane) - 1u))];
        base += __popc(m);
    }
}
// word accessor of a weight row: the first `cap` words from the gathered scratch, later ones by the slow index
struct WordsRowU {
    const uint32_t* row;     // gathered words
    const uint32_t* uarea;
    const uint16_t* ulen_hdr;
    uint32_t nw, cap;
    int lane;
    __device__ inline uint32_t operator()(uint32_t t) const {
        if (t >= nw) return 0u;
        if (t < cap) return row[t];
        return uarea[u_word_index_slow(ulen_hdr, lane, t)];
    }
};
struct WordsRowR {  // R words of row `lane`, interleaved over the 32 rows
    const uint32_t* rarea;
    int lane, rw_words;
    __device__ inline uint32_t operator()(uint32_t j) const { return j < (uint32_t)rw_words ? rarea[j * 32 + lane] : 0u; }
};

// exclusive prefix sum of the 128 ulen of a group; thread i gets its row's U-section start.
// scan_smem: 4 words. All 128 threads of the (sub)block call it; 
__device__ inline uint32_t row_ustart_128(uint32_t ul, uint32_t* scan_smem, int tid) {
    int lane = tid & 31, warp = tid >> 5;
    uint32_t x = ul;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) scan_smem[warp] = x;
    __syncthreads();
    uint32_t add = 0;
#pragma unroll
    for (int w = 0; w < 4; ++w)
        if (w < warp) add += scan_smem[w];
    __syncthreads();
    return x - ul + add;
}


}  // namespace hq
