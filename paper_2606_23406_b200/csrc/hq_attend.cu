// hq_attend.cu — attention over the compressed KV cache (§5.2,
// L178).  Scores and the P·V sum are taken in the CODE domain: RHT and S are orthogonal, so
//   <q, k̂> = (rho/(alpha sqrt n)) <S RHT q, c - U>                         (Prop. 1)
// and the V accumulation is un-rotated once at the end.  Tokens of the residual window are read
// exactly from the bf16 ring (§6.7.2).
#include "hq_common.cuh"
#include "hq_e8_decode.cuh"
#include "hq_internal.h"

namespace hq {

// U-section start of token t of (role, head): blk_off + sum of the block's earlier ulen (FORMAT §6)
__device__ inline uint32_t kv_ustart_serial(const uint16_t* ulen_h, const uint32_t* blk_h, int64_t t) {
    int64_t t0 = t & ~(int64_t)127;
    uint32_t s = blk_h[t >> 7];
    for (int64_t i = t0; i < t; ++i) s += ulen_h[i];
    return s;
}

template <int LAT>
__global__ void k_kv_decode_int8(const uint32_t* rem, const uint32_t* una, const uint16_t* ulen,
                                 const uint32_t* blk_off, int H, int d, int k0, int k1, int rbits,
                                 int64_t max_tokens, int64_t rem_words, int64_t una_words, int64_t n_blk,
                                 int64_t t0, int64_t n, int8_t* codes) {
    int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (idx >= n * H) return;
    int64_t t = t0 + idx / H;
    int h = (int)(idx % H);
    uint32_t us = kv_ustart_serial(ulen + h * max_tokens, blk_off + h * (n_blk + 1), t);
    int8_t* out = codes + idx * d;
    decode_row_generic<LAT>(WordsContig{rem + h * rem_words}, (uint32_t)(t * rbits), WordsContig{una + h * una_words}, us, d, k0, k1,
                            [&](int b, const int* c) {
#pragma unroll
                                for (int e = 0; e < LAT; ++e) out[b * LAT + e] = (int8_t)c[e];
                            });
}

void launch_kv_decode_int8(const hq_kv* kv, int role, int64_t t0, int64_t n, int8_t* codes, cudaStream_t st) {
    int H = kv->cfg.kv_heads, d = kv->cfg.head_dim;
    int64_t mt = kv->cfg.max_tokens;
    const uint32_t* rem = kv->rem + (int64_t)role * H * kv->rem_words;
    const uint32_t* una = kv->una + (int64_t)role * H * kv->una_words;
    const uint16_t* ulen = kv->ulen + (int64_t)role * H * mt;
    const uint32_t* blk = kv->blk_off + (int64_t)role * H * (kv->n_blk + 1);
    unsigned blocks = (unsigned)((n * H + 63) / 64);
#define HQ_KD(L)                                                                                                  \
    k_kv_decode_int8<L><<<blocks, 64, 0, st>>>(rem, una, ulen, blk, H, d, kv->k0, kv->k1, kv->rbits, mt,          \
                                               kv->rem_words, kv->una_words, kv->n_blk, t0, n, codes)
    switch (kv->cfg.codec.lattice) {
        case LAT_Z: HQ_KD(LAT_Z); break;
        case LAT_A2: HQ_KD(LAT_A2); break;
        case LAT_D4: HQ_KD(LAT_D4); break;
        default: HQ_KD(LAT_E8); break;
    }
#undef HQ_KD
}

// one cached vector -> out(blk, c[LAT]) per lattice block: the SWAR E8 decoder of hq_e8_decode.cuh when it applies
// (E8, head_dim 128, k <= 3), the generic decoder otherwise and for the rare rows the fast one declines
template <int LAT, class Out>
__device__ __forceinline__ void decode_token(const uint32_t* rem, uint32_t rpos, const uint32_t* una, uint32_t us,
                                             uint32_t ul, int d, int k0, int k1, uint32_t lut, uint32_t scr_a, Out out) {
    bool ok = false;
    if (LAT == LAT_E8 && d == 128 && k0 <= 3) {
        const uint32_t* rrow = rem + (rpos >> 5);   // rbits = 128 k: word aligned
        switch (k0) {
            case 0: ok = e8_decode_row_kv<0>(una, us, ul, rrow, lut, scr_a, out); break;
            case 1: ok = e8_decode_row_kv<1>(una, us, ul, rrow, lut, scr_a, out); break;
            case 2: ok = e8_decode_row_kv<2>(una, us, ul, rrow, lut, scr_a, out); break;
            default: ok = e8_decode_row_kv<3>(una, us, ul, rrow, lut, scr_a, out); break;
        }
    }
    if (!ok) decode_row_generic<LAT>(WordsContig{rem}, rpos, WordsContig{una}, us, d, k0, k1, out);
}

// ---------------------------------------------------------------------------------------------
// Split attention over the bitstream part.  CTA = (kv head h, split s), 128 threads.
// Per block of 128 tokens (thread = token):
//   K: decode the token's code vector block by block, regenerate the dither, dot with q'_g (G query
//      heads of this kv head) -> score; block max / exp -> p_g[t] in smem.
//   V: decode, write v' = (rho/A)(c - U) to smem [token][d]; then thread j (= coordinate) sums
//      p_g[t] v'[t][j] over the block into its running accumulators (online softmax rescale).
// Output per (h, split): m_g, l_g, acc_g[d] in the code domain.
// ---------------------------------------------------------------------------------------------
constexpr int ATT_MAXG = 8;

struct AttendParams {
    const uint32_t *rem, *una, *blk_off;
    const uint16_t *ulen, *norm;
    int H, d, k0, k1, rbits, G, dither, rotation;
    int64_t max_tokens, rem_words, una_words, n_blk;
    int64_t Tc;      // tokens served from the bitstream: [0, Tc)
    int n_split;
    float inv_A, inv_sqrt_d;
    uint64_t seed;
    const __nv_bfloat16* q;  // [q_heads, d]
    const int8_t *dsign, *ssign;
    const float *qjl, *qjl_t;   // HQ_ROT_QJL: S row-major and S transposed (null otherwise)
    float* ws;               // [H][n_split][G][d + 2]
    const uint32_t* pos_dev; // device_position caches: the held-token count is read here, not taken from Tc (graph replay)
    int window;
};
// tokens served from the bitstream
__device__ __forceinline__ int64_t attend_tc(const AttendParams& p) {
    if (!p.pos_dev) return p.Tc;
    const int64_t T = (int64_t)__ldcg(p.pos_dev);
    return T > p.window ? T - p.window : 0;
}

// q' = S * RHT(q) for one head, in smem (fp32), by one warp (FORMAT R1 order; any order would do here)
__device__ inline void warp_query_transform(float* s, int d, const int8_t* dsign, const int8_t* ssign, int rotation,
                                            const float* __restrict__ qjl_t, int lane) {
    for (int i = lane; i < d; i += 32)
        if (dsign[i] < 0) s[i] = -s[i];
    for (int h = 1; h < d; h <<= 1) {
        __syncwarp();
        for (int p = lane; p < d / 2; p += 32) {
            int i = ((p / h) * 2 * h) + (p % h);
            float a = s[i], b = s[i + h];
            s[i] = a + b;
            s[i + h] = a - b;
        }
    }
    __syncwarp();
    float cn = rsqrtf((float)d);
    for (int i = lane; i < d; i += 32) {
        float v = s[i] * cn;
        s[i] = (rotation == HQ_ROT_SIGNS && ssign[i] < 0) ? -v : v;
    }
    __syncwarp();
    if (rotation == HQ_ROT_QJL) {   // q' = S RHT(q) (§3.4 eq.(2)): one d x d matvec per query head, not per cached token (L502)
        float acc[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k] = 0.0f;
        for (int j = 0; j < d; ++j) {
            const float sj = s[j];
#pragma unroll
            for (int k = 0; k < 8; ++k)
                if (k * 32 < d) acc[k] = fmaf(__ldg(qjl_t + (int64_t)j * d + k * 32 + lane), sj, acc[k]);
        }
        __syncwarp();
#pragma unroll
        for (int k = 0; k < 8; ++k)
            if (k * 32 < d) s[k * 32 + lane] = acc[k];
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------
// The E8 dither of one lattice block, regenerated for attend (FORMAT §1, R4, R6; A.6 L843-847).  Same decisions and the
// same roundings as dither_block<LAT_E8> (hq_common.cuh) - every value below is the same fp32 number - but written for
// issue slots: the Philox round keys are precomputed once per thread (rk), rint is the magic-constant add (exact RNE for
// |z| < 2^22), the D8 parity fix is branch-free, and the coset points stay in fp32 (small integers are exact).
// ---------------------------------------------------------------------------------------------
struct PhiloxKeys { uint32_t k0[10], k1[10]; };
__device__ __forceinline__ PhiloxKeys philox_round_keys(uint64_t seed) {
    PhiloxKeys rk;
    uint32_t a = (uint32_t)seed, b = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) { rk.k0[r] = a; rk.k1[r] = b; a += 0x9E3779B9u; b += 0xBB67AE85u; }
    return rk;
}
__device__ __forceinline__ void philox4x32_10_keys(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxKeys& rk,
                                                   uint32_t* o) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0, l0, h1, l1;   // one 32 x 32 -> 64 multiply each (IMAD.WIDE), not a high and a low half
        asm("{\n\t.reg .u64 t;\n\tmul.wide.u32 t, %2, %3;\n\tmov.b64 {%0, %1}, t;\n\t}" : "=r"(l0), "=r"(h0) : "r"(c0), "r"(0xD2511F53u));
        asm("{\n\t.reg .u64 t;\n\tmul.wide.u32 t, %2, %3;\n\tmov.b64 {%0, %1}, t;\n\t}" : "=r"(l1), "=r"(h1) : "r"(c2), "r"(0xCD9E8D57u));
        c0 = h1 ^ c1 ^ rk.k0[r]; c1 = l1; c2 = h0 ^ c3 ^ rk.k1[r]; c3 = l0;
    }
    o[0] = c0; o[1] = c1; o[2] = c2; o[3] = c3;
}
// Q_{D8}(z) in fp32: f = rint(z); if sum f is odd, the first coordinate with the largest |z - f| moves one step away
__device__ __forceinline__ void nearest_d8_f32(const float* z, float* f) {
    const float M = 12582912.0f;   // 1.5 * 2^23
    float dl[8], sum = 0.0f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        f[i] = __fsub_rn(__fadd_rn(z[i], M), M);
        dl[i] = __fsub_rn(z[i], f[i]);
        sum += f[i];                      // exact: small integers
    }
    const bool odd = ((int)sum) & 1;
    float best = fabsf(dl[0]), dj = dl[0];
    int j = 0;
#pragma unroll
    for (int i = 1; i < 8; ++i) {
        const float a = fabsf(dl[i]);
        const bool gt = a > best;
        best = gt ? a : best; dj = gt ? dl[i] : dj; j = gt ? i : j;
    }
    const float step = odd ? (dj < 0.0f ? -1.0f : 1.0f) : 0.0f;
#pragma unroll
    for (int i = 0; i < 8; ++i) f[i] += (i == j) ? step : 0.0f;
}
__device__ __forceinline__ void dither_e8_fast(const PhiloxKeys& rk, uint32_t blk, uint32_t token, uint32_t headrole, float* U) {
    uint32_t o[8];
    philox4x32_10_keys(2 * blk, token, headrole, 3u, rk, o);
    philox4x32_10_keys(2 * blk + 1, token, headrole, 3u, rk, o + 4);
    float y[8], za[8], zb[8], fa[8], fb[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const float wf = (float)(2u * (o[j] >> 9) + 1u);          // exact: < 2^24
        y[j] = __fsub_rn(__fmul_rn(wf, 0x1p-22f), 2.0f);
        za[j] = __fmul_rn(y[j], 0.5f);
        zb[j] = __fmul_rn(__fsub_rn(y[j], 1.0f), 0.5f);
    }
    nearest_d8_f32(za, fa);
    nearest_d8_f32(zb, fb);
    float da[8], db[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        fa[i] = fa[i] * 2.0f;                 // a = 2 Q(y/2)
        fb[i] = fb[i] * 2.0f + 1.0f;          // b = 2 Q((y-1)/2) + 1   (exact small integers)
        const float ea = __fsub_rn(y[i], fa[i]), eb = __fsub_rn(y[i], fb[i]);
        da[i] = __fmul_rn(ea, ea);
        db[i] = __fmul_rn(eb, eb);
    }
    const float dist_a = __fadd_rn(__fadd_rn(__fadd_rn(da[0], da[1]), __fadd_rn(da[2], da[3])),
                                   __fadd_rn(__fadd_rn(da[4], da[5]), __fadd_rn(da[6], da[7])));
    const float dist_b = __fadd_rn(__fadd_rn(__fadd_rn(db[0], db[1]), __fadd_rn(db[2], db[3])),
                                   __fadd_rn(__fadd_rn(db[4], db[5]), __fadd_rn(db[6], db[7])));
    const bool pa = dist_a <= dist_b;
#pragma unroll
    for (int i = 0; i < 8; ++i) U[i] = __fsub_rn(y[i], pa ? fa[i] : fb[i]);
}

// ---- the same dither with packed fp32 pairs (sm_100 add / mul / fma .f32x2): the kernel is issue bound and the E8 nearest
// point is 19 FADD + 6 FMUL per scalar, so two coordinates per instruction saves a sixth of all issue slots.  Pair k holds
// coordinates (k, k + 4): elementwise steps pair up trivially, and the canonical tree sum of the squared distances
// ((d0+d1)+(d2+d3)) + ((d4+d5)+(d6+d7)) is two packed levels and one scalar add.  Every operation is the same IEEE
// round-to-nearest fp32 operation on the same values as in dither_e8_fast: a - b is fma(b, -1, a) (the product is exact),
// y = w 2^-22 - 2 and (y - 1) / 2 are single fmas whose products are exact too.  Same decisions, same U.
__device__ __forceinline__ uint64_t pk2(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void up2(uint64_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) { uint64_t r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b) { uint64_t r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) { uint64_t r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }

// Q_{D8} on packed pairs: z2[k] = (z_k, z_{k+4}); returns f2 likewise
__device__ __forceinline__ void nearest_d8_p2(const uint64_t* z2, uint64_t* f2) {
    const uint64_t M2 = pk2(12582912.0f, 12582912.0f), NM2 = pk2(-12582912.0f, -12582912.0f), N1 = pk2(-1.0f, -1.0f);
    uint64_t dl2[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        f2[k] = add2(add2(z2[k], M2), NM2);    // rint: (z + M) - M
        dl2[k] = fma2(f2[k], N1, z2[k]);       // z - f
    }
    float slo, shi;
    up2(add2(add2(f2[0], f2[1]), add2(f2[2], f2[3])), slo, shi);
    const bool odd = ((int)(slo + shi)) & 1;   // exact: small integers
    float dl[8];
#pragma unroll
    for (int k = 0; k < 4; ++k) up2(dl2[k], dl[k], dl[k + 4]);
    float best = fabsf(dl[0]), dj = dl[0];
    int j = 0;
#pragma unroll
    for (int i = 1; i < 8; ++i) {
        const float a = fabsf(dl[i]);
        const bool gt = a > best;
        best = gt ? a : best; dj = gt ? dl[i] : dj; j = gt ? i : j;
    }
    const float step = odd ? (dj < 0.0f ? -1.0f : 1.0f) : 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k) f2[k] = add2(f2[k], pk2(j == k ? step : 0.0f, j == k + 4 ? step : 0.0f));
}
// U2[k] = (U_k, U_{k+4})
__device__ __forceinline__ void dither_e8_packed(const PhiloxKeys& rk, uint32_t blk, uint32_t token, uint32_t headrole, uint64_t* U2) {
    uint32_t o[8];
    philox4x32_10_keys(2 * blk, token, headrole, 3u, rk, o);
    philox4x32_10_keys(2 * blk + 1, token, headrole, 3u, rk, o + 4);
    const uint64_t C22 = pk2(0x1p-22f, 0x1p-22f), N2 = pk2(-2.0f, -2.0f), H2 = pk2(0.5f, 0.5f), NH2 = pk2(-0.5f, -0.5f),
                   T2 = pk2(2.0f, 2.0f), O2 = pk2(1.0f, 1.0f), N1 = pk2(-1.0f, -1.0f);
    uint64_t y2[4], za2[4], zb2[4], fa2[4], fb2[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint64_t w2 = pk2((float)(2u * (o[k] >> 9) + 1u), (float)(2u * (o[k + 4] >> 9) + 1u));   // exact: < 2^24
        y2[k] = fma2(w2, C22, N2);            // w 2^-22 - 2
        za2[k] = mul2(y2[k], H2);             // y / 2
        zb2[k] = fma2(y2[k], H2, NH2);        // (y - 1) / 2
    }
    nearest_d8_p2(za2, fa2);
    nearest_d8_p2(zb2, fb2);
    uint64_t da2[4], db2[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        fa2[k] = mul2(fa2[k], T2);            // a = 2 Q(y/2)
        fb2[k] = fma2(fb2[k], T2, O2);        // b = 2 Q((y-1)/2) + 1
        const uint64_t ea = fma2(fa2[k], N1, y2[k]), eb = fma2(fb2[k], N1, y2[k]);
        da2[k] = mul2(ea, ea);
        db2[k] = mul2(eb, eb);
    }
    float alo, ahi, blo, bhi;
    up2(add2(add2(da2[0], da2[1]), add2(da2[2], da2[3])), alo, ahi);   // ((d0+d1)+(d2+d3), (d4+d5)+(d6+d7))
    up2(add2(add2(db2[0], db2[1]), add2(db2[2], db2[3])), blo, bhi);
    const bool pa = __fadd_rn(alo, ahi) <= __fadd_rn(blo, bhi);
#pragma unroll
    for (int k = 0; k < 4; ++k) U2[k] = fma2(pa ? fa2[k] : fb2[k], N1, y2[k]);
}

// GP = query heads per KV head padded to 4 or 8 (vector loads of q' and p).
// Code size matters here (the dither regeneration is ~300 instructions per lattice block): a token's codes are decoded
// once into a byte row in shared memory, and ONE loop over the lattice blocks regenerates the dither and feeds the score
// (K) or the v' row (V); nothing is unrolled over blocks or duplicated per decoder path.
template <int LAT, int GP>
// 256 threads: threads 0..127 take the K rows of the block's 128 tokens (decode, dither, scores), threads 128..255 the V rows
// (decode, dither, v' rows) AT THE SAME TIME - half the serial latency per block of the one-role-after-the-other loop and
// 16 instead of 12 resident warps per SM; the P V product is then split over the two halves by tokens.
__global__ void __launch_bounds__(256, 2)
k_attend_split(AttendParams p) {
    extern __shared__ float sm[];
    const int d = p.d, G = p.G;
    float* qs = sm;                            // [d][GP]   q' of the G query heads, coordinate-major
    float* vt = qs + d * GP;                   // [128][d+1]
    float* ps = vt + 128 * (d + 1);            // [128][GP]  p of the block's tokens
    float* red = ps + 128 * GP;                // [GP][4] block reductions (score max)
    float* red2 = red + GP * 4;                // [GP][4] block reductions (sum of p)
    const int KC = d + 68;                     // bytes per token of the K threads' rows: d codes + 17 nibble words
    uint8_t* kc = (uint8_t*)(red2 + GP * 4);   // [128][KC]
    __shared__ uint32_t scan[8];               // [role][4]
    __shared__ uint32_t lut_s[512];    // phase-1 table of the E8 decoder, [parity][byte]
    const int tid = threadIdx.x, role = tid >> 7, tok = tid & 127, lane = tid & 31, warp = tok >> 5;   // warp: inside the role
    const int h = blockIdx.x / p.n_split, split = blockIdx.x % p.n_split;
    for (int i = tid; i < 512; i += 256) lut_s[i] = unary_lut_entry(i & 255, i >> 8);
    const uint32_t lut_a = smem_u32(lut_s);
    // nibble scratch of the E8 decoder: the last 17 words of this thread's (otherwise idle at that time) vt row
    const uint32_t scr_a = role ? smem_u32(vt + tok * (d + 1) + (d - 17)) : smem_u32(kc + tok * KC + d);
    // the token's INT8 codes: the last d bytes of its vt row.  The V loop overwrites the row with floats from the front
    // and reads the codes of a step before writing it, so the floats never reach codes still needed (4 j0 + 32 <= 3 d + 4 + j0 + 8)
    uint8_t* crow = role ? (uint8_t*)(vt + tok * (d + 1)) + (3 * d + 4) : kc + tok * KC;

    // q' = S RHT(q): transformed in the vt area (one row of d floats per head), then stored coordinate-major
    for (int i = tid; i < G * d; i += 256) vt[i] = __bfloat162float(p.q[(h * G) * d + i]);
    __syncthreads();
    for (int g = tid >> 5; g < G; g += 8) warp_query_transform(vt + g * d, d, p.dsign, p.ssign, p.rotation, p.qjl_t, lane);
    __syncthreads();
    for (int i = tid; i < d * GP; i += 256) {
        const int j = i / GP, g = i % GP;
        qs[i] = g < G ? vt[g * d + j] : 0.0f;
    }
    __syncthreads();

    const int64_t Tc = attend_tc(p);
    const int64_t nblk_total = (Tc + 127) / 128;
    const int64_t blk0 = (nblk_total * split) / p.n_split, blk1 = (nblk_total * (split + 1)) / p.n_split;   // balanced

    const PhiloxKeys rk = philox_round_keys(p.seed);
    float m_run[GP], l_run[GP], acc[GP], acc2[GP];  // thread (j, half) owns coordinate j (and j + 128 when d == 256) over its half of a block's tokens
#pragma unroll
    for (int g = 0; g < GP; ++g) { m_run[g] = -INFINITY; l_run[g] = 0.0f; acc[g] = 0.0f; acc2[g] = 0.0f; }

    for (int64_t blk = blk0; blk < blk1; ++blk) {
        const int64_t t = blk * 128 + tok;
        const bool valid = t < Tc;
        float pg[GP];
        {
            const uint32_t* rem = p.rem + ((int64_t)role * p.H + h) * p.rem_words;
            const uint32_t* una = p.una + ((int64_t)role * p.H + h) * p.una_words;
            const uint16_t* ulen = p.ulen + ((int64_t)role * p.H + h) * p.max_tokens;
            const uint16_t* norm = p.norm + ((int64_t)role * p.H + h) * p.max_tokens;
            const uint32_t* blkoff = p.blk_off + ((int64_t)role * p.H + h) * (p.n_blk + 1);
            // every token of the block has been appended (t < T), those >= Tc are simply masked
            uint32_t ul = (blk * 128 + tok < p.max_tokens) ? ulen[blk * 128 + tok] : 0;
            uint32_t us = blkoff[blk] + row_ustart_128(ul, scan + 4 * role, tok);
            const float scale = valid ? f16_bits_to_f32(norm[t]) * p.inv_A : 0.0f;
            // ---- decode the token's codes into its byte row
            if (valid) {
                decode_token<LAT>(rem, (uint32_t)(t * p.rbits), una, us, ul, d, p.k0, p.k1, lut_a, scr_a,
                                  [&](int b, const int* c) {
                                      if (LAT == LAT_E8) {
                                          uint32_t w0 = 0, w1 = 0;
#pragma unroll
                                          for (int e = 0; e < 4; ++e) {
                                              w0 |= (uint32_t)(uint8_t)(int8_t)c[e] << (8 * e);
                                              w1 |= (uint32_t)(uint8_t)(int8_t)c[4 + e] << (8 * e);
                                          }
                                          *(uint32_t*)(crow + b * 8) = w0;
                                          *(uint32_t*)(crow + b * 8 + 4) = w1;
                                      } else {
#pragma unroll
                                          for (int e = 0; e < LAT; ++e) crow[b * LAT + e] = (uint8_t)(int8_t)c[e];
                                      }
                                  });
            }
            uint64_t dot2[GP / 2];   // (head 2i, head 2i + 1)
#pragma unroll
            for (int g = 0; g < GP / 2; ++g) dot2[g] = 0ull;
            float* row = vt + tok * (d + 1);
            // ---- one loop over the lattice blocks: codes - regenerated dither -> score terms (K) or the v' row (V)
            if (valid) {
                constexpr int BL = LAT == LAT_E8 ? 8 : 4;   // coordinates per iteration (a multiple of the lattice dimension)
#pragma unroll 1
                for (int j0 = 0; j0 < d; j0 += BL) {
                    float v[BL];
                    const uint32_t w0 = *(const uint32_t*)(crow + j0);
                    const uint32_t w1 = BL == 8 ? *(const uint32_t*)(crow + j0 + 4) : 0u;
#pragma unroll
                    for (int e = 0; e < BL; ++e) v[e] = (float)(int)(int8_t)((e < 4 ? w0 : w1) >> (8 * (e & 3)));
                    if (LAT == LAT_A2) { v[0] *= HQ_S3; v[2] *= HQ_S3; }
                    if (p.dither) {
                        if (LAT == LAT_E8) {   // packed pairs (coordinate k, k + 4)
                            uint64_t U2[4];
                            dither_e8_packed(rk, (uint32_t)(j0 / LAT), (uint32_t)t, (uint32_t)h | ((uint32_t)role << 16), U2);
#pragma unroll
                            for (int k = 0; k < 4; ++k) up2(fma2(U2[k], pk2(-1.0f, -1.0f), pk2(v[k], v[k + 4])), v[k], v[k + 4]);
                        } else {
#pragma unroll
                            for (int sb = 0; sb < BL / LAT; ++sb) {
                                float U[LAT];
                                dither_block<LAT>(p.seed, (uint32_t)(j0 / LAT + sb), (uint32_t)t, (uint32_t)h, (uint32_t)role, U);
#pragma unroll
                                for (int e = 0; e < LAT; ++e) v[sb * LAT + e] -= U[e];
                            }
                        }
                    }
                    if (role == 0) {
#pragma unroll
                        for (int e = 0; e < BL; ++e) {
                            const uint64_t vv = pk2(v[e], v[e]);
#pragma unroll
                            for (int g4 = 0; g4 < GP; g4 += 4) {   // two query heads per packed fma
                                const ulonglong2 q2 = *(const ulonglong2*)(qs + (j0 + e) * GP + g4);
                                dot2[g4 / 2] = fma2(q2.x, vv, dot2[g4 / 2]);
                                dot2[g4 / 2 + 1] = fma2(q2.y, vv, dot2[g4 / 2 + 1]);
                            }
                        }
                    } else {
#pragma unroll
                        for (int e = 0; e < BL; ++e) row[j0 + e] = v[e] * scale;
                    }
                }
            } else if (role == 1) {
                for (int j = 0; j < d; ++j) row[j] = 0.0f;
            }
            if (role == 0) {
                // scores and the warps' maxima
#pragma unroll
                float dot[GP];
#pragma unroll
                for (int g = 0; g < GP / 2; ++g) up2(dot2[g], dot[2 * g], dot[2 * g + 1]);
#pragma unroll
                for (int g = 0; g < GP; ++g) {
                    float s = (valid && g < G) ? dot[g] * scale * p.inv_sqrt_d : -INFINITY;
                    float mx = s;
                    for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                    if (lane == 0) red[g * 4 + warp] = mx;
                    pg[g] = s;
                }
            }
            __syncthreads();   // the maxima and the v' rows are written
#pragma unroll
            for (int g = 0; g < GP; ++g) {
                float mb = fmaxf(fmaxf(red[g * 4], red[g * 4 + 1]), fmaxf(red[g * 4 + 2], red[g * 4 + 3]));
                float m_new = fmaxf(m_run[g], mb);
                float corr = (m_run[g] == -INFINITY) ? 0.0f : __expf(m_run[g] - m_new);
                if (role == 0) {
                    float pe = (valid && g < G) ? __expf(pg[g] - m_new) : 0.0f;
                    ps[tok * GP + g] = pe;
                    float psum = pe;   // the block's softmax denominator, once (not per coordinate in the P V loop)
                    for (int o = 16; o; o >>= 1) psum += __shfl_xor_sync(0xffffffffu, psum, o);
                    if (lane == 0) red2[g * 4 + warp] = psum;
                }
                // every thread keeps the same running stats; l gets the block sum below
                acc[g] *= corr; acc2[g] *= corr; l_run[g] *= corr; m_run[g] = m_new;
            }
            __syncthreads();   // p and its sums are written
            // P V: thread = (coordinate, half of the block's tokens); the halves meet after the last block
            for (int j = tok, jj = 0; j < d; j += 128, ++jj) {
                uint64_t a2[GP / 2];
#pragma unroll
                for (int g = 0; g < GP / 2; ++g) a2[g] = 0ull;
#pragma unroll 4
                for (int tt = 64 * role; tt < 64 * role + 64; ++tt) {
                    const float vf = vt[tt * (d + 1) + j];
                    const uint64_t vv = pk2(vf, vf);
#pragma unroll
                    for (int g4 = 0; g4 < GP; g4 += 4) {
                        const ulonglong2 p2 = *(const ulonglong2*)(ps + tt * GP + g4);
                        a2[g4 / 2] = fma2(p2.x, vv, a2[g4 / 2]);
                        a2[g4 / 2 + 1] = fma2(p2.y, vv, a2[g4 / 2 + 1]);
                    }
                }
#pragma unroll
                for (int g = 0; g < GP / 2; ++g) {
                    float lo, hi;
                    up2(a2[g], lo, hi);
                    if (jj == 0) { acc[2 * g] += lo; acc[2 * g + 1] += hi; } else { acc2[2 * g] += lo; acc2[2 * g + 1] += hi; }
                }
            }
#pragma unroll
            for (int g = 0; g < GP; ++g) l_run[g] += (red2[g * 4] + red2[g * 4 + 1]) + (red2[g * 4 + 2] + red2[g * 4 + 3]);
            __syncthreads();   // the block's rows, p and reductions may be overwritten
        }
    }
    // the two token halves of every coordinate meet (vt is free now)
    if (role == 1) {
#pragma unroll
        for (int g = 0; g < GP; ++g) { vt[(2 * g) * 128 + tok] = acc[g]; vt[(2 * g + 1) * 128 + tok] = acc2[g]; }
    }
    __syncthreads();
    if (role == 1) return;
#pragma unroll
    for (int g = 0; g < GP; ++g) { acc[g] += vt[(2 * g) * 128 + tok]; acc2[g] += vt[(2 * g + 1) * 128 + tok]; }
    // write partials: [h][split][g][d + 2] = acc..., m, l   (threads with tid < d hold valid m/l)
    float* out = p.ws + ((int64_t)(h * p.n_split + split) * G) * (d + 2);
#pragma unroll
    for (int g = 0; g < GP; ++g) {
        if (g < G) {
            if (tok < d) out[g * (d + 2) + tok] = acc[g];
            if (d > 128) out[g * (d + 2) + tok + 128] = acc2[g];
            if (tok == 0) { out[g * (d + 2) + d] = m_run[g]; out[g * (d + 2) + d + 1] = l_run[g]; }
        }
    }
}

// Combine the splits, add the exact window tokens, un-rotate: one block per query head, d threads.
__global__ void k_attend_combine(AttendParams p, const __nv_bfloat16* ring, int window, int64_t T,
                                 __nv_bfloat16* out_bf16, float* out_f32) {
    extern __shared__ float sm[];
    const int d = p.d, G = p.G;
    float* code = sm;        // [d] code-domain accumulator
    float* sc = code + d;    // [window] window scores
    float* qf = sc + (window > 0 ? window : 1);  // [d]
    float* fs = qf + d;      // [n_split] exp(m_s - m), 0 for an empty split
    float* ls = fs + p.n_split;   // [n_split] the split's softmax denominator
    float* red = ls + p.n_split;  // [d / 32] block reduction
    __shared__ float s_m, s_l;
    const int qh = blockIdx.x, h = qh / G, g = qh % G, j = threadIdx.x;
    if (p.pos_dev) T = (int64_t)__ldcg(p.pos_dev);
    const float* wbase = p.ws + ((int64_t)h * p.n_split * G + g) * (d + 2);   // split s at + s * G * (d + 2)
    const int64_t wstride = (int64_t)G * (d + 2);
    // this thread's coordinate of the first 64 splits' partial rows: issued now, needed after the max (one round trip for all)
    constexpr int PRE = 64;
    float pv[PRE];
#pragma unroll
    for (int u = 0; u < PRE; ++u) pv[u] = u < p.n_split ? __ldcg(wbase + u * wstride + j) : 0.0f;
    // global max over splits: thread j takes splits j, j + d, ... (independent loads), then a block reduction
    float m = -INFINITY;
    for (int s = j; s < p.n_split; s += d) {
        const float* w = wbase + s * wstride;
        const float ms = __ldcg(w + d), l = __ldcg(w + d + 1);
        fs[s] = ms;
        ls[s] = l;
        if (l > 0.0f) m = fmaxf(m, ms);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((j & 31) == 0) red[j >> 5] = m;
    // window scores (original domain, exact bf16 K)
    qf[j] = __bfloat162float(p.q[qh * d + j]);
    __syncthreads();
    for (int i = 0; i < d / 32; ++i) m = fmaxf(m, red[i]);
    const int64_t w0 = attend_tc(p);
    const int nw = (int)(T - w0);
    if (j < nw) {
        int64_t t = w0 + j;
        const uint4* kr = (const uint4*)(ring + ((int64_t)(0 * window + (t % window)) * p.H + h) * d);   // rows are 2 d bytes: 16-byte aligned
        float dot = 0.0f;
        for (int i8 = 0; i8 < d / 8; ++i8) {
            const uint4 v = __ldg(kr + i8);
            const uint32_t wv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                dot += qf[8 * i8 + 2 * e] * __uint_as_float(wv[e] << 16);
                dot += qf[8 * i8 + 2 * e + 1] * __uint_as_float(wv[e] & 0xffff0000u);
            }
        }
        sc[j] = dot * p.inv_sqrt_d;
    }
    __syncthreads();
    if (j == 0) {
        float mm = m;
        for (int i = 0; i < nw; ++i) mm = fmaxf(mm, sc[i]);
        s_m = mm;
    }
    __syncthreads();
    m = s_m;
    for (int s = j; s < p.n_split; s += d) fs[s] = ls[s] > 0.0f ? __expf(fs[s] - m) : 0.0f;
    __syncthreads();
    // the splits in split order (deterministic), eight loads in flight at a time
    float a = 0.0f, l = 0.0f;
#pragma unroll
    for (int u = 0; u < PRE; ++u)
        if (u < p.n_split && ls[u] > 0.0f) {
            const float f = fs[u];
            a += f * pv[u];
            l += f * ls[u];
        }
    for (int s0 = PRE; s0 < p.n_split; s0 += 8) {
        float v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = (s0 + u < p.n_split && ls[s0 + u] > 0.0f) ? __ldcg(wbase + (s0 + u) * wstride + j) : 0.0f;
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (s0 + u < p.n_split && ls[s0 + u] > 0.0f) {
                const float f = fs[s0 + u];
                a += f * v[u];
                l += f * ls[s0 + u];
            }
    }
    // un-rotate the code-domain sum: x = D H (S u) / sqrt(d)
    code[j] = (p.rotation == HQ_ROT_SIGNS && p.ssign[j] < 0) ? -a : a;
    __syncthreads();
    if (p.rotation == HQ_ROT_QJL) {   // S^T: code_j <- sum_i S_ij code_i (thread j walks column j of S: coalesced)
        float r = 0.0f;
        for (int i = 0; i < d; ++i) r = fmaf(__ldg(p.qjl + (int64_t)i * d + j), code[i], r);
        __syncthreads();
        code[j] = r;
        __syncthreads();
    }
    for (int hh = 1; hh < d; hh <<= 1) {
        float x = 0.0f, y = 0.0f;
        int i = 0;
        if (j < d / 2) {
            i = ((j / hh) * 2 * hh) + (j % hh);
            x = code[i];
            y = code[i + hh];
        }
        __syncthreads();
        if (j < d / 2) {
            code[i] = x + y;
            code[i + hh] = x - y;
        }
        __syncthreads();
    }
    float o = code[j] * rsqrtf((float)d) * (p.dsign[j] < 0 ? -1.0f : 1.0f);
    // window tokens: exact V
    for (int i = 0; i < nw; ++i) {
        int64_t t = w0 + i;
        float pe = __expf(sc[i] - m);
        const __nv_bfloat16* vr = ring + ((int64_t)(1 * window + (t % window)) * p.H + h) * d;
        o += pe * __bfloat162float(vr[j]);
        l += pe;
    }
    if (j == 0) s_l = l;
    __syncthreads();
    o = s_l > 0.0f ? o / s_l : 0.0f;   // an empty device-position cache attends to nothing: zeros, not NaN
    if (out_bf16) out_bf16[qh * d + j] = __float2bfloat16_rn(o);
    if (out_f32) out_f32[qh * d + j] = o;
}

static int attend_n_split(const hq_ctx* ctx, const hq_kv* kv) {
    int64_t window = kv->cfg.window;
    int64_t Tc = kv->n_tokens > window ? kv->n_tokens - window : 0;
    if (kv->pos_dev) Tc = kv->cfg.max_tokens;   // fixed for the life of the cache: a captured launch stays valid as tokens arrive
    int64_t nblk = (Tc + 127) / 128;
    int64_t want = (ctx->sm_count * 2) / kv->cfg.kv_heads;   // one wave of the 2 resident CTAs (256 threads) per SM
    if (want < 1) want = 1;
    int64_t ns = nblk < want ? nblk : want;
    return (int)(ns < 1 ? 1 : ns);
}

size_t attend_workspace_bytes(const hq_ctx* ctx, const hq_kv* kv) {
    // attend_n_split launches at most 4 CTAs per SM in total, each writing ATT_MAXG x (d + 2) floats
    return (size_t)(ctx->sm_count * 4 + kv->cfg.kv_heads) * ATT_MAXG * (size_t)(kv->cfg.head_dim + 2) * sizeof(float);
}

hq_status launch_attend(hq_ctx* ctx, const hq_kv* kv, const void* q, int q_heads, void* out_bf16, float* out_f32,
                        cudaStream_t st) {
    AttendParams p;
    int H = kv->cfg.kv_heads, d = kv->cfg.head_dim;
    p.rem = kv->rem; p.una = kv->una; p.blk_off = kv->blk_off; p.ulen = kv->ulen; p.norm = kv->norm;
    p.H = H; p.d = d; p.k0 = kv->k0; p.k1 = kv->k1; p.rbits = kv->rbits; p.G = q_heads / H;
    p.dither = kv->cfg.dither; p.rotation = kv->cfg.rotation;
    p.max_tokens = kv->cfg.max_tokens; p.rem_words = kv->rem_words; p.una_words = kv->una_words; p.n_blk = kv->n_blk;
    int64_t window = kv->cfg.window;
    p.Tc = kv->n_tokens > window ? kv->n_tokens - window : 0;
    p.n_split = attend_n_split(ctx, kv);
    p.pos_dev = kv->pos_dev; p.window = (int)window;
    p.inv_A = (float)(1.0 / (kv->alpha * sqrt((double)d)));
    p.inv_sqrt_d = (float)(1.0 / sqrt((double)d));
    p.seed = kv->cfg.codec.seed;
    p.q = (const __nv_bfloat16*)q; p.dsign = kv->dsign; p.ssign = kv->ssign; p.ws = kv->att_ws;
    p.qjl = kv->qjl; p.qjl_t = kv->qjl ? kv->qjl + (size_t)kv->cfg.head_dim * kv->cfg.head_dim : nullptr;
    const int GP = p.G <= 4 ? 4 : 8;
    size_t smem = ((size_t)GP * d + 128 * (size_t)(d + 1) + (size_t)GP * 128 + (size_t)GP * 8) * sizeof(float) + 128 * (size_t)(d + 68);
#define HQ_AT(L)                                                                                                   \
    do {                                                                                                           \
        if (GP == 4) {                                                                                             \
            HQ_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_attend_split<L, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
            k_attend_split<L, 4><<<H * p.n_split, 256, smem, st>>>(p);                                             \
        } else {                                                                                                   \
            HQ_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_attend_split<L, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
            k_attend_split<L, 8><<<H * p.n_split, 256, smem, st>>>(p);                                             \
        }                                                                                                          \
    } while (0)
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    const bool run_split = p.Tc > 0 || kv->pos_dev;   // a device-position cache always launches: the count may have grown
    if (ctx->prof && run_split) {
        HQ_CUDA_CHECK(ctx, cudaEventCreate(&e0));
        HQ_CUDA_CHECK(ctx, cudaEventCreate(&e1));
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e0, st));
    }
    if (run_split) {
        switch (kv->cfg.codec.lattice) {
            case LAT_Z: HQ_AT(LAT_Z); break;
            case LAT_A2: HQ_AT(LAT_A2); break;
            case LAT_D4: HQ_AT(LAT_D4); break;
            default: HQ_AT(LAT_E8); break;
        }
        HQ_CUDA_CHECK(ctx, cudaGetLastError());
        if (e0) {
            HQ_CUDA_CHECK(ctx, cudaEventRecord(e1, st));
            ctx->prof_ev.push_back(e0);
            ctx->prof_ev.push_back(e1);
        }
    } else {
        p.n_split = 0;
    }
#undef HQ_AT
    size_t smem2 = (size_t)(2 * d + (window > 0 ? window : 1) + 2 * p.n_split + d / 32) * sizeof(float);
    k_attend_combine<<<q_heads, d, smem2, st>>>(p, kv->ring, (int)window, kv->n_tokens, (__nv_bfloat16*)out_bf16, out_f32);
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    return HQ_OK;
}

}  // namespace hq
