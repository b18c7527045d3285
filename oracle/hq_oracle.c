/*
 * hq_oracle.c — the ORACLE for HyperQuant's inference hot path (arxiv/paper_2606_23406).
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  The product (paper_2606_23406_b200/)
 * never does and shares no code, header, table or generator with it.
 *
 * Plain, slow, obviously-correct C: scalar loops in the paper's order and notation, following
 * docs/FORMAT.md for everything the paper leaves open (readings G1..G18 in DESIGN.md).  Citations
 * are PAPER.md line numbers.  Encode-side floating point is IEEE binary32 without FMA contraction
 * (build: gcc -O2 -ffp-contract=off, no -ffast-math) because it decides integers; reconstruction /
 * attention / dense-RHT checks are in double.
 *
 * Parity pins (tests/test_oracle_*.py): Philox known-answer vectors; H·Hᵀ = n·I and the dense
 * double RHT; brute-force nearest point; Voronoi second moments vs Table 2 (L139-142); strip
 * bijection and Table 3 savings (L284); Rice round trip; printed rates at 21 dB (L289); Table 14
 * α (L887-890); Table 11 A2 SNRs (L550-552); dither moments and unbiasedness (L786-808);
 * the layer glue of FORMAT R8-R10 (RMSNorm, SiLU·mul, bf16 rounding) against numpy float64 / ml_dtypes-free
 * bit manipulation (tests/test_oracle_layer.py).
 * Parity unpinned: none.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define HQO_Z 1
#define HQO_A2 2
#define HQO_D4 4
#define HQO_E8 8

/* ------------------------------------------------------------------------------------------ */
/* Counter RNG: Philox4x32-10 (docs/FORMAT.md §1).                                              */
/* ------------------------------------------------------------------------------------------ */
void hqo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
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

/* sign d_i in {+1,-1}: stream 1 = RHT D (eq.(1)), stream 2 = KV rotation S (L216). */
void hqo_signs(uint64_t seed, uint32_t stream, int64_t n, int8_t* out) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    for (int64_t i = 0; i < n; ++i) {
        uint32_t ctr[4] = {(uint32_t)(i >> 7), 0u, 0u, stream}, o[4];
        hqo_philox4x32_10(ctr, key, o);
        out[i] = ((o[(i >> 5) & 3] >> (i & 31)) & 1u) ? -1 : 1;
    }
}

/* dither uniform e of (token, head, role): odd 24-bit integer w = 2r+1 (FORMAT §1). */
static uint32_t dither_w(uint64_t seed, uint32_t e, uint32_t token, uint32_t head, uint32_t role) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t ctr[4] = {e >> 2, token, head | (role << 16), 3u}, o[4];
    hqo_philox4x32_10(ctr, key, o);
    return 2u * (o[e & 3] >> 9) + 1u;
}

/* ------------------------------------------------------------------------------------------ */
/* fp16 (storage of the norm, L500), bf16 helpers.                                             */
/* ------------------------------------------------------------------------------------------ */
static uint16_t f32_to_f16_bits(float f) { /* RNE, saturating at 65504 (FORMAT R3) */
    if (!(f == f)) return 0x7e00;
    float a = fabsf(f);
    uint16_t sign = signbit(f) ? 0x8000 : 0;
    if (a >= 65520.0f) return sign | 0x7bff; /* would round to inf: saturate */
    if (a < 5.9604644775390625e-8f * 0.5f) return sign;
    int e;
    float m = frexpf(a, &e); /* a = m * 2^e, m in [0.5,1) */
    int E = e - 1;            /* a = (2m) * 2^E, 2m in [1,2) */
    if (E < -14) {            /* subnormal: units of 2^-24 */
        float q = rintf(ldexpf(a, 24));
        return sign | (uint16_t)q; /* q may be 1024 = smallest normal: bit pattern still right */
    }
    float q = rintf(ldexpf(m, 11)); /* mantissa in [1024, 2048] */
    if (q == 2048.0f) { q = 1024.0f; E += 1; }
    return sign | (uint16_t)(((E + 15) << 10) + ((int)q - 1024));
}
static float f16_bits_to_f32(uint16_t h) {
    int s = h >> 15, e = (h >> 10) & 31, m = h & 1023;
    float v;
    if (e == 0) v = ldexpf((float)m, -24);
    else if (e == 31) v = m ? NAN : INFINITY;
    else v = ldexpf((float)(m + 1024), e - 25);
    return s ? -v : v;
}
uint16_t hqo_f32_to_f16_bits(float f) { return f32_to_f16_bits(f); }
float hqo_f16_bits_to_f32(uint16_t h) { return f16_bits_to_f32(h); }

/* ------------------------------------------------------------------------------------------ */
/* RHT (§3.1 eq.(1), §4.1; FORMAT R1).                                               */
/* ------------------------------------------------------------------------------------------ */
void hqo_fwht_f32(float* v, int n) { /* unnormalized Sylvester butterfly, ascending stride */
    for (int h = 1; h < n; h <<= 1)
        for (int i = 0; i < n; ++i)
            if ((i & h) == 0) {
                float a = v[i], b = v[i + h];
                v[i] = a + b;
                v[i + h] = a - b;
            }
}
void hqo_rht_f32(const float* x, const int8_t* d, int n, float* u) {
    float cn = (float)(1.0 / sqrt((double)n));
    for (int i = 0; i < n; ++i) u[i] = (d[i] < 0) ? -x[i] : x[i];
    hqo_fwht_f32(u, n);
    for (int i = 0; i < n; ++i) u[i] = u[i] * cn;
}
/* the definition, dense and in double: u = (1/sqrt n) H D x, H[i][j] = (-1)^popcount(i&j). */
void hqo_rht_dense_f64(const double* x, const int8_t* d, int n, double* u) {
    for (int i = 0; i < n; ++i) {
        double s = 0.0;
        for (int j = 0; j < n; ++j) {
            int par = __builtin_popcount((unsigned)(i & j)) & 1;
            double t = (double)d[j] * x[j];
            s += par ? -t : t;
        }
        u[i] = s / sqrt((double)n);
    }
}
/* inverse of the orthonormal RHT in double: x = D H u / sqrt n. */
static void rht_inverse_f64(const double* u, const int8_t* d, int n, double* x) {
    for (int j = 0; j < n; ++j) {
        double s = 0.0;
        for (int i = 0; i < n; ++i) {
            int par = __builtin_popcount((unsigned)(i & j)) & 1;
            s += par ? -u[i] : u[i];
        }
        x[j] = (double)d[j] * s / sqrt((double)n);
    }
}

static float treesum_f32(float* a, int m) { /* FORMAT R2, destroys a */
    for (int h = 1; h < m; h <<= 1)
        for (int i = 0; i + h < m; i += 2 * h) a[i] = a[i] + a[i + h];
    return a[0];
}

/* ------------------------------------------------------------------------------------------ */
/* Scale α (eq.(9)) and lattice constants (Table 2, covolumes from L241).          */
/* ------------------------------------------------------------------------------------------ */
int hqo_dim(int lattice) { return lattice; }
double hqo_second_moment(int lattice) { /* M = G(Λ) · V^{2/N} of the integer realization */
    switch (lattice) {
        case HQO_Z: return 1.0 / 12.0;
        case HQO_A2: return 0.0802 * 2.0 * sqrt(3.0); /* V = 2·sqrt3, N = 2 */
        case HQO_D4: return 0.0766 * sqrt(2.0);       /* V = 2, N = 4 */
        case HQO_E8: return 0.0717 * 4.0;             /* V = 2^8, N = 8 */
    }
    return 0.0;
}
double hqo_alpha(int lattice, double snr_db) {
    return sqrt(pow(10.0, snr_db / 10.0) * hqo_second_moment(lattice));
}

/* ------------------------------------------------------------------------------------------ */
/* Nearest lattice point (§3.2, §4.5; FORMAT R5, R6).                                 */
/* ------------------------------------------------------------------------------------------ */
static const float S3 = 1.7320508075688772f; /* (float)sqrt(3.0) */

static void nearest_Dm(const float* z, int m, int32_t* f) { /* Conway–Sloane D_m */
    float delta[8];
    int sum = 0;
    for (int i = 0; i < m; ++i) {
        float r = rintf(z[i]);
        f[i] = (int32_t)r;
        delta[i] = z[i] - r;
        sum += f[i];
    }
    if (sum & 1) {
        int j = 0;
        for (int i = 1; i < m; ++i)
            if (fabsf(delta[i]) > fabsf(delta[j])) j = i;
        f[j] += (delta[j] < 0.0f) ? -1 : 1;
    }
}

/* Q_Λ(y) without the INT8 pre-clamp. For A2 the block is (y, x) and c = (n_y, n_x). */
static void nearest_noclamp(int lattice, const float* y, int32_t* c) {
    if (lattice == HQO_Z) {
        c[0] = (int32_t)rintf(y[0]);
    } else if (lattice == HQO_D4) {
        nearest_Dm(y, 4, c);
    } else if (lattice == HQO_E8) {
        float za[8], zb[8], da[8], db[8];
        int32_t a[8], b[8];
        for (int i = 0; i < 8; ++i) { za[i] = y[i] * 0.5f; zb[i] = (y[i] - 1.0f) * 0.5f; }
        nearest_Dm(za, 8, a);
        nearest_Dm(zb, 8, b);
        for (int i = 0; i < 8; ++i) {
            a[i] = 2 * a[i];
            b[i] = 2 * b[i] + 1;
            float ea = y[i] - (float)a[i], eb = y[i] - (float)b[i];
            da[i] = ea * ea;
            db[i] = eb * eb;
        }
        float dist_a = treesum_f32(da, 8), dist_b = treesum_f32(db, 8);
        memcpy(c, (dist_a <= dist_b) ? a : b, 8 * sizeof(int32_t));
    } else { /* A2 */
        float two_s3 = 2.0f * S3;
        int32_t ay = 2 * (int32_t)rintf(y[0] / two_s3), ax = 2 * (int32_t)rintf(y[1] * 0.5f);
        int32_t by = 2 * (int32_t)rintf((y[0] - S3) / two_s3) + 1;
        int32_t bx = 2 * (int32_t)rintf((y[1] - 1.0f) * 0.5f) + 1;
        float eay = y[0] - S3 * (float)ay, eax = y[1] - (float)ax;
        float eby = y[0] - S3 * (float)by, ebx = y[1] - (float)bx;
        float dist_a = eay * eay + eax * eax, dist_b = eby * eby + ebx * ebx;
        if (dist_a <= dist_b) { c[0] = ay; c[1] = ax; } else { c[0] = by; c[1] = bx; }
    }
}

/* with the INT8 pre-clamp of the quantizer input (G8 / FORMAT R5); returns #coordinates clamped */
static int clamp_block(int lattice, const float* y, float* z) {
    int n = lattice, cnt = 0;
    for (int i = 0; i < n; ++i) {
        float lim = (lattice == HQO_E8) ? 125.0f : (lattice == HQO_Z) ? 127.0f : 126.0f;
        if (lattice == HQO_A2 && i == 0) lim = 126.0f * S3;
        float v = y[i];
        if (v > lim) { v = lim; cnt++; }
        if (v < -lim) { v = -lim; cnt++; }
        z[i] = v;
    }
    return cnt;
}
int hqo_nearest(int lattice, const float* y, int32_t* c) {
    float z[8];
    int cnt = clamp_block(lattice, y, z);
    nearest_noclamp(lattice, z, c);
    return cnt;
}
void hqo_nearest_noclamp(int lattice, const float* y, int32_t* c) { nearest_noclamp(lattice, y, c); }

/* dither U = π_Λ(box-uniform) for block `blk` of a vector (A.6 L843-847; FORMAT R4). */
static void dither_block(int lattice, uint64_t seed, uint32_t blk, uint32_t token, uint32_t head,
                         uint32_t role, float* U) {
    int dim = lattice;
    float y[8];
    int32_t c[8];
    for (int j = 0; j < dim; ++j) {
        float w = (float)dither_w(seed, (uint32_t)dim * blk + (uint32_t)j, token, head, role);
        if (lattice == HQO_E8) y[j] = w * 0x1p-22f - 2.0f;
        else if (lattice == HQO_D4) y[j] = w * 0x1p-23f - 1.0f;
        else if (lattice == HQO_Z) y[j] = w * 0x1p-24f - 0.5f;
        else y[j] = (j == 0) ? (w * 0x1p-23f - 1.0f) * S3 : (w * 0x1p-23f - 1.0f);
    }
    nearest_noclamp(lattice, y, c);
    for (int j = 0; j < dim; ++j) {
        float p = (float)c[j];
        if (lattice == HQO_A2 && j == 0) p = S3 * p;
        U[j] = y[j] - p;
    }
}
void hqo_dither_block(int lattice, uint64_t seed, uint32_t blk, uint32_t token, uint32_t head,
                      uint32_t role, float* U) {
    dither_block(lattice, seed, blk, token, head, role, U);
}

/* ------------------------------------------------------------------------------------------ */
/* Strip / un-strip with zig-zag (§4.6; FORMAT §3).                                    */
/* ------------------------------------------------------------------------------------------ */
static int32_t zigzag(int32_t v) { return v >= 0 ? 2 * v : -2 * v - 1; }
static int32_t unzigzag(int32_t z) { return (z & 1) ? -((z + 1) >> 1) : (z >> 1); }
static int32_t half_exact(int32_t v) { return v >> 1; } /* callers guarantee v even */

void hqo_strip(int lattice, const int32_t* c, int32_t* z) {
    if (lattice == HQO_E8) {
        int32_t coset = c[0] & 1, s[8], sum = 0;
        for (int i = 0; i < 8; ++i) s[i] = half_exact(c[i] - coset);
        for (int i = 0; i < 7; ++i) sum += s[i];
        int32_t p = sum & 1, t = half_exact(s[7] - p);
        for (int i = 0; i < 7; ++i) z[i] = zigzag(s[i]);
        z[7] = 2 * zigzag(t) + coset; /* comb, L274 */
    } else if (lattice == HQO_D4) {
        int32_t p = (c[0] + c[1] + c[2]) & 1, t = half_exact(c[3] - p);
        z[0] = zigzag(c[0]); z[1] = zigzag(c[1]); z[2] = zigzag(c[2]); z[3] = zigzag(t);
    } else if (lattice == HQO_A2) {
        int32_t p = c[1] & 1, ty = half_exact(c[0] - p);
        z[0] = zigzag(ty); z[1] = zigzag(c[1]);
    } else {
        z[0] = zigzag(c[0]);
    }
}
void hqo_unstrip(int lattice, const int32_t* z, int32_t* c) {
    if (lattice == HQO_E8) {
        int32_t s[8], sum = 0, coset = z[7] & 1, t = unzigzag(z[7] >> 1);
        for (int i = 0; i < 7; ++i) { s[i] = unzigzag(z[i]); sum += s[i]; }
        s[7] = 2 * t + (sum & 1);
        for (int i = 0; i < 8; ++i) c[i] = 2 * s[i] + coset;
    } else if (lattice == HQO_D4) {
        c[0] = unzigzag(z[0]); c[1] = unzigzag(z[1]); c[2] = unzigzag(z[2]);
        c[3] = 2 * unzigzag(z[3]) + ((c[0] + c[1] + c[2]) & 1);
    } else if (lattice == HQO_A2) {
        c[1] = unzigzag(z[1]);
        c[0] = 2 * unzigzag(z[0]) + (c[1] & 1);
    } else {
        c[0] = unzigzag(z[0]);
    }
}
static int sym_class(int lattice, int j) {
    if (lattice == HQO_D4) return (j & 3) == 3;
    if (lattice == HQO_A2) return j & 1;
    return 0;
}
/* Stream order of a tile's symbols (FORMAT §3).  Position p of the tile stream holds the symbol of
 * lattice block blk, coordinate i, returned as the block-major index blk*dim + i.  D4, A2, Z:
 * block-major (identity).  E8: inside each run of 32 symbols (4 blocks) the order is coordinate-pair
 * major: p = 32c + 8w + 2b + e  <->  block 4c + b, coordinate 2w + e  (w = 0..3, b = 0..3, e = 0..1),
 * so that four consecutive even (odd) positions hold one coordinate of four consecutive blocks. */
static int stream_to_blockmajor(int lattice, int p) {
    if (lattice != HQO_E8) return p;
    int c = p >> 5, w = (p >> 3) & 3, b = (p >> 1) & 3, e = p & 1;
    return 8 * (4 * c + b) + 2 * w + e;
}
/* symbols of a whole tile of n codes, in stream order; cls[p] = Rice class of position p */
static void tile_symbols(int lattice, const int8_t* codes, int n, int32_t* z) {
    int dim = lattice;
    int32_t zb[1024];
    for (int b = 0; b < n / dim; ++b) {
        int32_t c[8];
        for (int i = 0; i < dim; ++i) c[i] = codes[b * dim + i];
        hqo_strip(lattice, c, zb + b * dim);
    }
    for (int p = 0; p < n; ++p) z[p] = zb[stream_to_blockmajor(lattice, p)];
}
/* inverse: stream-order symbols -> codes */
static void tile_codes(int lattice, const int32_t* z, int n, int8_t* codes) {
    int dim = lattice;
    int32_t zb[1024];
    for (int p = 0; p < n; ++p) zb[stream_to_blockmajor(lattice, p)] = z[p];
    for (int b = 0; b < n / dim; ++b) {
        int32_t c[8];
        hqo_unstrip(lattice, zb + b * dim, c);
        for (int i = 0; i < dim; ++i) codes[b * dim + i] = (int8_t)c[i];
    }
}
/* Rice class of stream position p: a function of the symbol's coordinate inside its block */
static int pos_class(int lattice, int p) { return sym_class(lattice, stream_to_blockmajor(lattice, p)); }

/* ------------------------------------------------------------------------------------------ */
/* Rice coding of a tile into the split-plane tile stream (§3.3, §4.7; FORMAT §3-4).   */
/* ------------------------------------------------------------------------------------------ */
static void put_bit(uint32_t* words, uint64_t p, uint32_t bit) { /* MSB-first */
    if (bit) words[p >> 5] |= 1u << (31 - (p & 31));
}
static uint32_t get_bit(const uint32_t* words, uint64_t p) {
    return (words[p >> 5] >> (31 - (p & 31))) & 1u;
}
static void put_word(uint32_t* words, uint64_t p, uint32_t v, int nbits) { /* v's bit nbits-1 first */
    for (int i = 0; i < nbits; ++i) put_bit(words, p + i, (v >> (nbits - 1 - i)) & 1u);
}

/* bit length of a tile: Σ (k_j + 1 + q_j) */
int64_t hqo_tile_bits(int lattice, const int8_t* codes, int n, const int* k) {
    int32_t z[1024];
    tile_symbols(lattice, codes, n, z);
    int64_t L = 0;
    for (int j = 0; j < n; ++j) {
        int kk = k[pos_class(lattice, j)];
        L += kk + 1 + (z[j] >> kk);
    }
    return L;
}

/* Field planes of a k-bit remainder (FORMAT §4): one plane of width w = 1, 2, 4 for each set bit
 * of k = b0 + 2·b1 + 4·b2, in that order, each covering the next w remainder bits from bit 0 up
 * (k = 3: a 1-bit plane holding bit 0, then a 2-bit plane holding bits 1-2). */
static int field_planes(int k, int* w, int* lo) {
    int np = 0, at = 0;
    for (int b = 0; b < 3; ++b)
        if (k & (1 << b)) { w[np] = 1 << b; lo[np] = at; at += 1 << b; ++np; }
    return np;
}
static int rbits_of(int lattice, int n, const int* k) {
    int r = 0;
    for (int j = 0; j < n; ++j) r += k[sym_class(lattice, j)];
    return r;
}
int hqo_rbits(int lattice, int n, const int* k) { return rbits_of(lattice, n, k); }

/* R-section of one tile at bit position pos of `words` (FORMAT §4); returns its length n_0 k_0 + n_1 k_1 */
static int64_t write_tile_R(int lattice, const int8_t* codes, int n, const int* k, uint32_t* words,
                            uint64_t pos) {
    int32_t z[1024];
    uint64_t p = pos;
    tile_symbols(lattice, codes, n, z);
    int nclass = (lattice == HQO_D4 || lattice == HQO_A2) ? 2 : 1;
    for (int a = 0; a < nclass; ++a) {
        int32_t r[1024];
        int na = 0, ka = k[a], w[3], lo[3];
        int np = field_planes(ka, w, lo);
        for (int j = 0; j < n; ++j)
            if (pos_class(lattice, j) == a) r[na++] = z[j] & ((1 << ka) - 1);
        for (int ch = 0; ch * 32 < na; ++ch) {
            int cnt = na - ch * 32 < 32 ? na - ch * 32 : 32;
            for (int pl = 0; pl < np; ++pl) {
                int wd = w[pl], per = 8 / wd; /* groups of 4 symbols per word */
                if (cnt == 32) {
                    for (int i = 0; i < wd; ++i) {
                        uint32_t V = 0;
                        for (int u = 0; u < 32; ++u) {
                            int g = 2 * (u >> 3) + (u & 1), lane = (u & 7) >> 1;
                            if (g / per != i) continue;
                            uint32_t f = (uint32_t)(r[ch * 32 + u] >> lo[pl]) & ((1u << wd) - 1u);
                            V |= f << (8 * lane + wd * (g % per));
                        }
                        put_word(words, p, V, 32);
                        p += 32;
                    }
                } else { /* partial chunk: fields in symbol order, each MSB-first */
                    for (int u = 0; u < cnt; ++u) {
                        uint32_t f = (uint32_t)(r[ch * 32 + u] >> lo[pl]) & ((1u << wd) - 1u);
                        put_word(words, p, f, wd);
                        p += wd;
                    }
                }
            }
        }
    }
    return (int64_t)(p - pos);
}

/* U-section: for j = 0..n-1, q_j zeros then a one (§3.3); returns its length n + Σ q_j */
static int64_t write_tile_U(int lattice, const int8_t* codes, int n, const int* k, uint32_t* words,
                            uint64_t pos) {
    int32_t z[1024];
    uint64_t p = pos;
    tile_symbols(lattice, codes, n, z);
    for (int j = 0; j < n; ++j) {
        int q = z[j] >> k[pos_class(lattice, j)];
        p += q;
        put_bit(words, p, 1u);
        p += 1;
    }
    return (int64_t)(p - pos);
}

/* decode one tile from its R-section (rwords, rpos) and U-section (uwords, upos); returns U bits used */
static int64_t read_tile_RU(int lattice, int n, const int* k, const uint32_t* rwords, uint64_t rpos,
                            const uint32_t* uwords, uint64_t upos, int8_t* codes) {
    int32_t z[1024], rem[1024];
    uint64_t p = rpos;
    int nclass = (lattice == HQO_D4 || lattice == HQO_A2) ? 2 : 1;
    for (int a = 0; a < nclass; ++a) {
        int idx[1024], na = 0, ka = k[a], w[3], lo[3];
        int np = field_planes(ka, w, lo);
        for (int j = 0; j < n; ++j)
            if (pos_class(lattice, j) == a) { idx[na++] = j; rem[j] = 0; }
        for (int ch = 0; ch * 32 < na; ++ch) {
            int cnt = na - ch * 32 < 32 ? na - ch * 32 : 32;
            for (int pl = 0; pl < np; ++pl) {
                int wd = w[pl], per = 8 / wd;
                if (cnt == 32) {
                    for (int i = 0; i < wd; ++i) {
                        for (int u = 0; u < 32; ++u) {
                            int g = 2 * (u >> 3) + (u & 1), lane = (u & 7) >> 1;
                            if (g / per != i) continue;
                            int sh = 8 * lane + wd * (g % per); /* field's bit 0 in V */
                            for (int b = 0; b < wd; ++b)
                                rem[idx[ch * 32 + u]] |= (int32_t)get_bit(rwords, p + (31 - (sh + b))) << (lo[pl] + b);
                        }
                        p += 32;
                    }
                } else {
                    for (int u = 0; u < cnt; ++u) {
                        for (int b = 0; b < wd; ++b)
                            rem[idx[ch * 32 + u]] |= (int32_t)get_bit(rwords, p + b) << (lo[pl] + wd - 1 - b);
                        p += wd;
                    }
                }
            }
        }
    }
    p = upos;
    for (int j = 0; j < n; ++j) {
        int q = 0;
        while (!get_bit(uwords, p)) { ++q; ++p; }
        ++p;
        z[j] = (q << k[pos_class(lattice, j)]) | rem[j];
    }
    tile_codes(lattice, z, n, codes);
    return (int64_t)(p - upos);
}

/* the logical tile stream = R-section ‖ U-section at one bit position; returns its length L */
static int64_t write_tile(int lattice, const int8_t* codes, int n, const int* k, uint32_t* words,
                          uint64_t pos) {
    int64_t R = write_tile_R(lattice, codes, n, k, words, pos);
    return R + write_tile_U(lattice, codes, n, k, words, pos + (uint64_t)R);
}
static int64_t read_tile(int lattice, int n, const int* k, const uint32_t* words, uint64_t pos,
                         int8_t* codes) {
    int R = rbits_of(lattice, n, k);
    return R + read_tile_RU(lattice, n, k, words, pos, words, pos + (uint64_t)R, codes);
}

/* single-tile entry points for the round-trip pins */
int64_t hqo_write_tile(int lattice, const int8_t* codes, int n, const int* k, uint32_t* words,
                       uint64_t pos) {
    return write_tile(lattice, codes, n, k, words, pos);
}
int64_t hqo_read_tile(int lattice, int n, const int* k, const uint32_t* words, uint64_t pos,
                      int8_t* codes) {
    return read_tile(lattice, n, k, words, pos, codes);
}

/* The textbook Rice code of the same symbols (q zeros, a one, k bits MSB-first), interleaved per
 * symbol: used only to pin that the split-plane stream has exactly the Rice code's length. */
int64_t hqo_rice_reference_bits(int lattice, const int8_t* codes, int n, const int* k,
                                uint32_t* words) {
    int32_t z[1024];
    uint64_t p = 0;
    tile_symbols(lattice, codes, n, z);
    for (int j = 0; j < n; ++j) {
        int kk = k[pos_class(lattice, j)], q = z[j] >> kk;
        p += q;
        put_bit(words, p++, 1u);
        put_word(words, p, (uint32_t)(z[j] & ((1 << kk) - 1)), kk);
        p += kk;
    }
    return (int64_t)p;
}

/* marginal symbol histograms of a code array (for the B.4 scalar_entropy pin, L908) */
void hqo_symbol_histogram(int lattice, const int8_t* codes, int64_t ntiles, int n, int64_t* hist
                          /* [dim][512] */) {
    int dim = lattice;
    int32_t z[1024];
    for (int64_t t = 0; t < ntiles; ++t) {
        tile_symbols(lattice, codes + t * n, n, z);
        for (int j = 0; j < n; ++j) hist[(stream_to_blockmajor(lattice, j) % dim) * 512 + z[j]]++;
    }
}

/* ------------------------------------------------------------------------------------------ */
/* O1 steps 1-5: quantize rows of a matrix tile by tile (weights: no rotation, no dither).       */
/* W [m, n_in] fp32 (bf16 inputs are passed already widened, exactly).                           */
/* ------------------------------------------------------------------------------------------ */
static int64_t quantize_tile(int lattice, int n, float A, const float* u, int with_dither,
                             uint64_t seed, uint32_t token, uint32_t head, uint32_t role,
                             int8_t* codes, uint16_t* norm_bits) {
    float sq[1024];
    int64_t clamps = 0;
    for (int i = 0; i < n; ++i) sq[i] = u[i] * u[i];
    float rho32 = sqrtf(treesum_f32(sq, n));
    uint16_t hb = f32_to_f16_bits(rho32);
    float rho = f16_bits_to_f32(hb);
    *norm_bits = hb;
    if (rho == 0.0f) { /* G18 */
        memset(codes, 0, (size_t)n);
        return 0;
    }
    float g = A / rho;
    int dim = lattice;
    for (int b = 0; b < n / dim; ++b) {
        float y[8], U[8];
        int32_t c[8];
        for (int i = 0; i < dim; ++i) y[i] = u[b * dim + i] * g;
        if (with_dither) {
            dither_block(lattice, seed, (uint32_t)b, token, head, role, U);
            for (int i = 0; i < dim; ++i) y[i] = y[i] + U[i];
        }
        clamps += hqo_nearest(lattice, y, c);
        for (int i = 0; i < dim; ++i) codes[b * dim + i] = (int8_t)c[i];
    }
    return clamps;
}

int64_t hqo_quantize_weights(const float* W, int64_t m, int64_t n_in, int64_t ld, int lattice,
                             int n, double snr_db, uint64_t seed, int8_t* codes /*[m,n_in]*/,
                             uint16_t* norms /*[m,n_in/n]*/) {
    int64_t n_kt = n_in / n, clamps = 0;
    float A = (float)(hqo_alpha(lattice, snr_db) * sqrt((double)n));
    int8_t* d = (int8_t*)malloc((size_t)n_in);
    hqo_signs(seed, 1u, n_in, d);
#pragma omp parallel for reduction(+ : clamps) schedule(static)
    for (int64_t r = 0; r < m; ++r) {
        float u[1024];
        for (int64_t kt = 0; kt < n_kt; ++kt) {
            hqo_rht_f32(W + r * ld + kt * n, d + kt * n, n, u);
            clamps += quantize_tile(lattice, n, A, u, 0, 0, 0, 0, 0, codes + r * n_in + kt * n,
                                    norms + r * n_kt + kt);
        }
    }
    free(d);
    return clamps;
}

/* total bits of a code array for given k (also used by auto-k, FORMAT §3) */
int64_t hqo_total_bits(const int8_t* codes, int64_t ntiles, int lattice, int n, const int* k) {
    int64_t total = 0;
#pragma omp parallel for reduction(+ : total) schedule(static)
    for (int64_t t = 0; t < ntiles; ++t) total += hqo_tile_bits(lattice, codes + t * n, n, k);
    return total;
}
void hqo_choose_k(const int8_t* codes, int64_t ntiles, int lattice, int n, int* k_out) {
    /* per-class totals for k = 0..7 */
    int64_t tot[2][8];
    memset(tot, 0, sizeof tot);
    for (int64_t t = 0; t < ntiles; ++t) {
        int32_t z[1024];
        tile_symbols(lattice, codes + t * n, n, z);
        for (int j = 0; j < n; ++j)
            for (int kk = 0; kk < 8; ++kk) tot[pos_class(lattice, j)][kk] += kk + 1 + (z[j] >> kk);
    }
    if (lattice == HQO_D4) { /* k_t = max(k_s - 1, 0), minimize the sum (L272, L295) */
        int best = 0;
        int64_t bv = -1;
        for (int ks = 0; ks < 8; ++ks) {
            int kt = ks > 0 ? ks - 1 : 0;
            int64_t v = tot[0][ks] + tot[1][kt];
            if (bv < 0 || v < bv) { bv = v; best = ks; }
        }
        k_out[0] = best;
        k_out[1] = best > 0 ? best - 1 : 0;
        return;
    }
    for (int a = 0; a < 2; ++a) {
        int best = 0;
        for (int kk = 1; kk < 8; ++kk)
            if (tot[a][kk] < tot[a][best]) best = kk;
        k_out[a] = best;
    }
    if (lattice != HQO_A2) k_out[1] = k_out[0];
}

/* ------------------------------------------------------------------------------------------ */
/* Weight container (FORMAT §5): pack / unpack.                                                */
/* ------------------------------------------------------------------------------------------ */
/* Sub-group sg = (rb * n_kt + kt) * 4 + w holds rows [128 rb + 32 w, +32) of K-tile kt:
 *   u16 ulen[32] | u16 norm[32] | u32 rarea[RW*32] | u32 uarea[sum_i nw_i] | zero pad to 16 bytes
 * RW = ceil(Rbits/32); word j of row i's R-section at rarea[j*32 + i]; row i's U-section starts at
 * bit 0 of its own word 0 and takes nw_i = ceil(ulen_i/32) words; "word-row" t of uarea holds word t
 * of every row with nw_i > t, in increasing row order.  Absent rows (>= m): ulen = 0, norm = 0.
 * returns blob size in bytes; if blob == NULL only sizes (group_off[4G+1], 16-byte units) are computed. */
int64_t hqo_pack_weights(const int8_t* codes, const uint16_t* norms, int64_t m, int64_t n_in,
                         int lattice, int n, const int* k, uint8_t* blob,
                         uint32_t* group_off /*[4G+1]*/) {
    int64_t n_kt = n_in / n, n_rb = (m + 127) / 128, off16 = 0;
    int64_t Rbits = rbits_of(lattice, n, k), RW = (Rbits + 31) / 32;
    for (int64_t rb = 0; rb < n_rb; ++rb)
        for (int64_t kt = 0; kt < n_kt; ++kt)
            for (int w = 0; w < 4; ++w) {
                int64_t sg = (rb * n_kt + kt) * 4 + w, uwords = 0;
                int64_t U[32], nw[32], maxnw = 0;
                group_off[sg] = (uint32_t)off16;
                for (int i = 0; i < 32; ++i) {
                    int64_t r = rb * 128 + w * 32 + i;
                    U[i] = (r < m) ? hqo_tile_bits(lattice, codes + r * n_in + kt * n, n, k) - Rbits : 0;
                    nw[i] = (U[i] + 31) / 32;
                    uwords += nw[i];
                    if (nw[i] > maxnw) maxnw = nw[i];
                }
                int64_t bytes = 128 + 4 * (RW * 32 + uwords);
                int64_t sz16 = (bytes + 15) / 16;
                if (blob) {
                    uint8_t* base = blob + 16 * off16;
                    memset(base, 0, (size_t)sz16 * 16);
                    uint16_t* ulen = (uint16_t*)base;
                    uint16_t* nrm = ulen + 32;
                    uint32_t* rarea = (uint32_t*)(base + 128);
                    uint32_t* uarea = rarea + RW * 32;
                    uint32_t tmp[32][256]; /* row streams: FORMAT §5 bounds a U-section by 8160 bits = 255 words */
                    for (int i = 0; i < 32; ++i) {
                        int64_t r = rb * 128 + w * 32 + i;
                        ulen[i] = (uint16_t)U[i];
                        nrm[i] = (r < m) ? norms[r * n_kt + kt] : 0;
                        if (r >= m) continue;
                        uint32_t rw[64];
                        memset(rw, 0, sizeof rw);
                        write_tile_R(lattice, codes + r * n_in + kt * n, n, k, rw, 0);
                        for (int64_t j = 0; j < RW; ++j) rarea[j * 32 + i] = rw[j];
                        if (nw[i] > 255) return -1; /* FORMAT error (the CUDA side reports HQ_ERR_FORMAT) */
                        memset(tmp[i], 0, sizeof tmp[i]);
                        write_tile_U(lattice, codes + r * n_in + kt * n, n, k, tmp[i], 0);
                    }
                    int64_t at = 0;
                    for (int64_t t = 0; t < maxnw; ++t)
                        for (int i = 0; i < 32; ++i)
                            if (nw[i] > t) uarea[at++] = tmp[i][t];
                }
                off16 += sz16;
            }
    group_off[n_rb * n_kt * 4] = (uint32_t)off16;
    return off16 * 16;
}

/* O2: decode the container back to codes and norms */
void hqo_unpack_weights(const uint8_t* blob, const uint32_t* group_off, int64_t m, int64_t n_in,
                        int lattice, int n, const int* k, int8_t* codes, uint16_t* norms) {
    int64_t n_kt = n_in / n, n_rb = (m + 127) / 128;
    int64_t Rbits = rbits_of(lattice, n, k), RW = (Rbits + 31) / 32;
#pragma omp parallel for schedule(static)
    for (int64_t sg = 0; sg < n_rb * n_kt * 4; ++sg) {
        int64_t g = sg / 4, w = sg % 4, rb = g / n_kt, kt = g % n_kt;
        const uint8_t* base = blob + 16 * (int64_t)group_off[sg];
        const uint16_t* ulen = (const uint16_t*)base;
        const uint16_t* nrm = ulen + 32;
        const uint32_t* rarea = (const uint32_t*)(base + 128);
        const uint32_t* uarea = rarea + RW * 32;
        int64_t nw[32], maxnw = 0;
        for (int i = 0; i < 32; ++i) {
            nw[i] = (ulen[i] + 31) / 32;
            if (nw[i] > maxnw) maxnw = nw[i];
        }
        for (int i = 0; i < 32; ++i) {
            int64_t r = rb * 128 + w * 32 + i;
            if (r >= m) continue;
            norms[r * n_kt + kt] = nrm[i];
            uint32_t rw[64], uw[258];
            for (int64_t j = 0; j < RW; ++j) rw[j] = rarea[j * 32 + i];
            int64_t at = 0;
            for (int64_t t = 0; t < maxnw; ++t)
                for (int i2 = 0; i2 < 32; ++i2)
                    if (nw[i2] > t) {
                        if (i2 == i) uw[t] = uarea[at];
                        ++at;
                    }
            uw[nw[i]] = 0xffffffffu; /* guard: a corrupt stream stops here */
            read_tile_RU(lattice, n, k, rw, 0, uw, 0, codes + r * n_in + kt * n);
        }
    }
}

/* ------------------------------------------------------------------------------------------ */
/* O3: activations (FORMAT R7) and the INT8 contraction (§4.8).                            */
/* ------------------------------------------------------------------------------------------ */
void hqo_act_quant(const float* x, int64_t B, int64_t n_in, int64_t ldx, int lattice, int n,
                   uint64_t seed, int8_t* q /*[B,n_in]*/, float* s_x /*[B,n_kt]*/,
                   float* u_out /*[B,n_in] or NULL: the fp32 RHT output*/) {
    int64_t n_kt = n_in / n;
    int8_t* d = (int8_t*)malloc((size_t)n_in);
    hqo_signs(seed, 1u, n_in, d);
    for (int64_t b = 0; b < B; ++b)
        for (int64_t kt = 0; kt < n_kt; ++kt) {
            float u[1024], amax = 0.0f;
            hqo_rht_f32(x + b * ldx + kt * n, d + kt * n, n, u);
            if (u_out) memcpy(u_out + b * n_in + kt * n, u, (size_t)n * sizeof(float));
            if (lattice == HQO_A2)
                for (int i = 0; i < n; i += 2) u[i] = u[i] * S3;
            for (int i = 0; i < n; ++i)
                if (fabsf(u[i]) > amax) amax = fabsf(u[i]);
            int8_t* qq = q + b * n_in + kt * n;
            if (amax == 0.0f) {
                memset(qq, 0, (size_t)n);
                s_x[b * n_kt + kt] = 0.0f;
                continue;
            }
            float inv = 127.0f / amax;
            for (int i = 0; i < n; ++i) {
                float v = rintf(u[i] * inv);
                if (v > 127.0f) v = 127.0f;
                if (v < -127.0f) v = -127.0f;
                qq[i] = (int8_t)v;
            }
            s_x[b * n_kt + kt] = amax / 127.0f;
        }
    free(d);
}

/* ------------------------------------------------------------------------------------------ */
/* The steps between the linears of a decoder layer that fold into the activation cast           */
/* (§4.1: "the butterfly folds into the preceding LayerNorm"; FORMAT R8-R10). */
/* They produce the bf16 activation vector that hqo_act_quant then takes, so they decide integers */
/* and are canonical fp32.                                                                        */
/* ------------------------------------------------------------------------------------------ */
float hqo_bf16_round(float v) { /* fp32 -> bf16 (round to nearest even) -> fp32 */
    uint32_t b;
    memcpy(&b, &v, 4);
    if ((b & 0x7f800000u) == 0x7f800000u) return v; /* inf / nan unchanged */
    b += 0x7fffu + ((b >> 16) & 1u);
    b &= 0xffff0000u;
    memcpy(&v, &b, 4);
    return v;
}

void hqo_bf16_round_array(const float* v, int64_t n, float* out) {
    for (int64_t i = 0; i < n; ++i) out[i] = hqo_bf16_round(v[i]);
}

/* FORMAT R8: x_i = bf16((h_i * r) * g_i), r = 1 / sqrt(treesum(h_i^2) / n + eps). */
void hqo_rmsnorm_bf16(const float* h, const float* g, int64_t n, float eps, float* x) {
    float* sq = (float*)malloc((size_t)n * sizeof(float));
    for (int64_t i = 0; i < n; ++i) sq[i] = h[i] * h[i];
    float s = treesum_f32(sq, (int)n);
    free(sq);
    float ms = s / (float)n;
    float r = 1.0f / sqrtf(ms + eps);
    for (int64_t i = 0; i < n; ++i) x[i] = hqo_bf16_round((h[i] * r) * g[i]);
}

/* FORMAT R9: the canonical exponential (range reduction by ln 2 in two parts, degree-7 Taylor polynomial in Horner
 * form with fused multiply-adds, scaling by the exponent bits). */
float hqo_exp_c(float t) {
    if (t < -87.0f) t = -87.0f;
    if (t > 88.0f) t = 88.0f;
    float m = rintf(t * 0x1.715476p+0f);
    float f = fmaf(m, -0x1.62e000p-1f, t);
    f = fmaf(m, -0x1.0bfbe8p-15f, f);
    static const float C[8] = {1.0f, 1.0f, 0.5f, 0x1.555556p-3f, 0x1.555556p-5f, 0x1.111112p-7f, 0x1.6c16c2p-10f, 0x1.a01a02p-13f};
    float p = C[7];
    for (int j = 6; j >= 0; --j) p = fmaf(p, f, C[j]);
    uint32_t eb = (uint32_t)((int)m + 127) << 23;
    float two_m;
    memcpy(&two_m, &eb, 4);
    return p * two_m;
}

/* FORMAT R9: x_i = bf16(silu_c(a_i) * b_i), silu_c(a) = a / (1 + exp_c(-a)). */
void hqo_silu_mul_bf16(const float* a, const float* b, int64_t n, float* x) {
    for (int64_t i = 0; i < n; ++i) {
        float e = hqo_exp_c(-a[i]);
        float s = a[i] / (1.0f + e);
        x[i] = hqo_bf16_round(s * b[i]);
    }
}

/* acc[kt,b,r] = Σ_{i in tile} c[r,i]·q[b,i];  y[b,r] = Σ_kt (ρ[r,kt]/(α√n))·s_x[b,kt]·acc  (double) */
void hqo_linear(const int8_t* codes, const uint16_t* norms, int64_t m, int64_t n_in, int lattice,
                int n, double snr_db, const int8_t* q, const float* s_x, int64_t B,
                int32_t* acc /*[n_kt,B,m] or NULL*/, double* y /*[B,m]*/) {
    int64_t n_kt = n_in / n;
    double inv_A = 1.0 / (hqo_alpha(lattice, snr_db) * sqrt((double)n));
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < m; ++r)
        for (int64_t b = 0; b < B; ++b) {
            double yy = 0.0;
            for (int64_t kt = 0; kt < n_kt; ++kt) {
                int32_t a = 0;
                for (int i = 0; i < n; ++i)
                    a += (int32_t)codes[r * n_in + kt * n + i] * (int32_t)q[b * n_in + kt * n + i];
                if (acc) acc[(kt * B + b) * m + r] = a;
                yy += (double)f16_bits_to_f32(norms[r * n_kt + kt]) * inv_A *
                      (double)s_x[b * n_kt + kt] * (double)a;
            }
            y[b * m + r] = yy;
        }
}

/* ------------------------------------------------------------------------------------------ */
/* §4.8 L299 / §6.3: the FP8-E4M3 cast of both MMA operands ("a per-tile FP8 or INT8 cast for the MMA");        */
/* FORMAT R12.  E4M3 (fn): 1 sign, 4 exponent (bias 7), 3 mantissa bits; normals 2^-6 .. 448, subnormal step 2^-9;   */
/* round to nearest even, magnitudes that would round above 448 saturate to 448.                                      */
/* ------------------------------------------------------------------------------------------ */
float hqo_e4m3_round(float v) {
    if (v != v) return v;
    float a = fabsf(v), r;
    if (a >= 448.0f) r = 448.0f;
    else if (a < 0x1p-6f) r = rintf(a * 512.0f) / 512.0f;          /* subnormals: multiples of 2^-9 */
    else {
        int e;
        (void)frexpf(a, &e);                                       /* a = f * 2^e, f in [0.5, 1): 2^(e-1) <= a */
        float step = ldexpf(1.0f, e - 1 - 3);                      /* 3 mantissa bits */
        r = rintf(a / step) * step;                                /* power-of-two division: exact; rintf = RNE */
        if (r > 448.0f) r = 448.0f;
    }
    return v < 0.0f ? -r : r;
}
void hqo_e4m3_round_array(const float* v, int64_t n, float* out) {
    for (int64_t i = 0; i < n; ++i) out[i] = hqo_e4m3_round(v[i]);
}

/* activations (R12): u by R1; amax; q8_i = e4m3(u_i * (448 / amax)); s_x = amax / 448.  E8 / D4 / Z (no sqrt 3 factor). */
void hqo_act_quant_fp8(const float* x, int64_t B, int64_t n_in, int64_t ldx, int n, uint64_t seed,
                       float* q8 /*[B,n_in] E4M3 values*/, float* s_x /*[B,n_kt]*/) {
    int64_t n_kt = n_in / n;
    int8_t* d = (int8_t*)malloc((size_t)n_in);
    hqo_signs(seed, 1u, n_in, d);
    for (int64_t b = 0; b < B; ++b)
        for (int64_t kt = 0; kt < n_kt; ++kt) {
            float u[1024], amax = 0.0f;
            hqo_rht_f32(x + b * ldx + kt * n, d + kt * n, n, u);
            for (int i = 0; i < n; ++i)
                if (fabsf(u[i]) > amax) amax = fabsf(u[i]);
            float* qq = q8 + b * n_in + kt * n;
            if (amax == 0.0f) {
                for (int i = 0; i < n; ++i) qq[i] = 0.0f;
                s_x[b * n_kt + kt] = 0.0f;
                continue;
            }
            float inv = 448.0f / amax;
            for (int i = 0; i < n; ++i) qq[i] = hqo_e4m3_round(u[i] * inv);
            s_x[b * n_kt + kt] = amax / 448.0f;
        }
    free(d);
}

/* y[b,r] = Σ_kt (ρ[r,kt]/(α√n))·s_x[b,kt]·Σ_{i in tile} e4m3(c[r,i])·q8[b,i]   (double; products of two E4M3 values are exact) */
void hqo_linear_fp8(const int8_t* codes, const uint16_t* norms, int64_t m, int64_t n_in, int lattice, int n,
                    double snr_db, const float* q8, const float* s_x, int64_t B, double* y /*[B,m]*/,
                    double* acc /*[n_kt,B,m] or NULL: the per-tile sums*/, double* acc_abs /*[n_kt,B,m] or NULL: sums of |products|*/) {
    int64_t n_kt = n_in / n;
    double inv_A = 1.0 / (hqo_alpha(lattice, snr_db) * sqrt((double)n));
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < m; ++r)
        for (int64_t b = 0; b < B; ++b) {
            double yy = 0.0;
            for (int64_t kt = 0; kt < n_kt; ++kt) {
                double a = 0.0, aa = 0.0;
                for (int i = 0; i < n; ++i) {
                    double t = (double)hqo_e4m3_round((float)codes[r * n_in + kt * n + i]) * (double)q8[b * n_in + kt * n + i];
                    a += t;
                    aa += fabs(t);
                }
                if (acc) acc[(kt * B + b) * m + r] = a;
                if (acc_abs) acc_abs[(kt * B + b) * m + r] = aa;
                yy += (double)f16_bits_to_f32(norms[r * n_kt + kt]) * inv_A * (double)s_x[b * n_kt + kt] * a;
            }
            y[b * m + r] = yy;
        }
}

/* sampled version for sizes where the full contraction is too slow on a CPU: outputs (b_s, r_s) */
void hqo_linear_sampled(const int8_t* codes, const uint16_t* norms, int64_t m, int64_t n_in,
                        int lattice, int n, double snr_db, const int8_t* q, const float* s_x,
                        int64_t B, int64_t ns, const int64_t* bs, const int64_t* rs,
                        int32_t* acc /*[ns,n_kt]*/, double* y /*[ns]*/) {
    int64_t n_kt = n_in / n;
    double inv_A = 1.0 / (hqo_alpha(lattice, snr_db) * sqrt((double)n));
    (void)B; (void)m;
    for (int64_t s = 0; s < ns; ++s) {
        int64_t b = bs[s], r = rs[s];
        double yy = 0.0;
        for (int64_t kt = 0; kt < n_kt; ++kt) {
            int32_t a = 0;
            for (int i = 0; i < n; ++i)
                a += (int32_t)codes[r * n_in + kt * n + i] * (int32_t)q[b * n_in + kt * n + i];
            acc[s * n_kt + kt] = a;
            yy += (double)f16_bits_to_f32(norms[r * n_kt + kt]) * inv_A *
                  (double)s_x[b * n_kt + kt] * (double)a;
        }
        y[s] = yy;
    }
}

/* Ŵ in the original (un-rotated) domain, double: Ŵ[r,tile] = RHT^{-1}( (ρ/(α√n))·c ).  Used for
 * the MSE / realized-SNR pins (L874) and y_exact = Ŵx. */
void hqo_dequant_weights(const int8_t* codes, const uint16_t* norms, int64_t m, int64_t n_in,
                         int lattice, int n, double snr_db, uint64_t seed, double* What) {
    int64_t n_kt = n_in / n;
    double inv_A = 1.0 / (hqo_alpha(lattice, snr_db) * sqrt((double)n));
    int8_t* d = (int8_t*)malloc((size_t)n_in);
    hqo_signs(seed, 1u, n_in, d);
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < m; ++r)
        for (int64_t kt = 0; kt < n_kt; ++kt) {
            double u[1024], x[1024];
            double sc = (double)f16_bits_to_f32(norms[r * n_kt + kt]) * inv_A;
            for (int i = 0; i < n; ++i) {
                double p = (double)codes[r * n_in + kt * n + i];
                if (lattice == HQO_A2 && (i & 1) == 0) p *= sqrt(3.0);
                u[i] = sc * p;
            }
            rht_inverse_f64(u, d + kt * n, n, x);
            for (int i = 0; i < n; ++i) What[r * n_in + kt * n + i] = x[i];
        }
    free(d);
}

/* ------------------------------------------------------------------------------------------ */
/* KV path (§5.2): encode vectors [n_tok, heads, d] of one role.                        */
/* rotation: 0 none, 1 signs, 2 qjl (dense Q).  token0 = index of the first token of this call.   */
/* ------------------------------------------------------------------------------------------ */
/* rotation 2 = qjl (§3.4, eq.(2); Table 4): a dense orthogonal S = Q [d][d] row-major, drawn Haar-uniform
 * once per layer by the caller and passed in; u'_i = sum_j Q_ij u_j accumulated in j order with one fused multiply-add
 * per term (FORMAT R11 - canonical because it decides the codes).                                                   */
static void qjl_apply_f32(const float* Q, int d, float* u) {
    float r[1024];
    for (int i = 0; i < d; ++i) {
        float acc = 0.0f;
        for (int j = 0; j < d; ++j) acc = fmaf(Q[i * d + j], u[j], acc);
        r[i] = acc;
    }
    memcpy(u, r, (size_t)d * sizeof(float));
}
int64_t hqo_kv_quantize_q(const float* kv, int64_t n_tok, int heads, int d, int64_t token0, int role,
                          int lattice, double snr_db, int rotation, int dither, uint64_t seed, const float* Q,
                          int8_t* codes /*[n_tok,heads,d]*/, uint16_t* norms /*[n_tok,heads]*/);
int64_t hqo_kv_quantize(const float* kv, int64_t n_tok, int heads, int d, int64_t token0, int role,
                        int lattice, double snr_db, int rotation, int dither, uint64_t seed,
                        int8_t* codes /*[n_tok,heads,d]*/, uint16_t* norms /*[n_tok,heads]*/) {
    return hqo_kv_quantize_q(kv, n_tok, heads, d, token0, role, lattice, snr_db, rotation, dither, seed, NULL, codes, norms);
}
int64_t hqo_kv_quantize_q(const float* kv, int64_t n_tok, int heads, int d, int64_t token0, int role,
                          int lattice, double snr_db, int rotation, int dither, uint64_t seed, const float* Q,
                          int8_t* codes /*[n_tok,heads,d]*/, uint16_t* norms /*[n_tok,heads]*/) {
    float A = (float)(hqo_alpha(lattice, snr_db) * sqrt((double)d));
    int8_t *D = (int8_t*)malloc((size_t)d), *S = (int8_t*)malloc((size_t)d);
    int64_t clamps = 0;
    hqo_signs(seed, 1u, d, D);
    hqo_signs(seed, 2u, d, S);
#pragma omp parallel for reduction(+ : clamps) schedule(static)
    for (int64_t t = 0; t < n_tok; ++t)
        for (int h = 0; h < heads; ++h) {
            float u[1024];
            hqo_rht_f32(kv + (t * heads + h) * d, D, d, u);
            if (rotation == 1)
                for (int i = 0; i < d; ++i) u[i] = (S[i] < 0) ? -u[i] : u[i];
            if (rotation == 2) qjl_apply_f32(Q, d, u);
            clamps += quantize_tile(lattice, d, A, u, dither, seed, (uint32_t)(token0 + t),
                                    (uint32_t)h, (uint32_t)role, codes + (t * heads + h) * d,
                                    norms + t * heads + h);
        }
    free(D); free(S);
    return clamps;
}

/* pack one (role, head) of the KV container (FORMAT §6): token t's R-section goes to bit
 * (t0 + t)·Rbits of `rem`, its U-section is appended to `una` after bit position upos0.
 * ulen[t] written; returns the new U position.  Both word arrays zero-initialized by the caller. */
int64_t hqo_kv_pack_head(const int8_t* codes /*[n_tok,heads,d]*/, int64_t n_tok, int heads, int d,
                         int head, int lattice, const int* k, int64_t t0, uint32_t* rem,
                         uint32_t* una, int64_t upos0, uint16_t* ulen /*[n_tok]*/) {
    uint64_t p = (uint64_t)upos0;
    int64_t Rbits = rbits_of(lattice, d, k);
    for (int64_t t = 0; t < n_tok; ++t) {
        const int8_t* c = codes + (t * heads + head) * d;
        write_tile_R(lattice, c, d, k, rem, (uint64_t)((t0 + t) * Rbits));
        int64_t U = write_tile_U(lattice, c, d, k, una, p);
        ulen[t] = (uint16_t)U;
        p += (uint64_t)U;
    }
    return (int64_t)p;
}
/* decode token t of a packed (role, head): R-section at t·Rbits of rem, U-section at upos of una */
int64_t hqo_kv_unpack_token(int lattice, int d, const int* k, const uint32_t* rem, int64_t t,
                            const uint32_t* una, int64_t upos, int8_t* codes) {
    int64_t Rbits = rbits_of(lattice, d, k);
    return read_tile_RU(lattice, d, k, rem, (uint64_t)(t * Rbits), una, (uint64_t)upos, codes);
}

/* reconstruct one cached vector the long way (O4): decode -> c - U -> un-normalize -> Sᵀ -> RHT⁻¹ */
static void kv_reconstruct(const int8_t* codes, uint16_t norm_bits, int d, int lattice, double inv_A,
                           int rotation, int dither, uint64_t seed, uint32_t token, uint32_t head,
                           uint32_t role, const int8_t* D, const int8_t* S, const float* Q, double* out) {
    double u[1024];
    double sc = (double)f16_bits_to_f32(norm_bits) * inv_A;
    int dim = lattice;
    for (int b = 0; b < d / dim; ++b) {
        float U[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        if (dither) dither_block(lattice, seed, (uint32_t)b, token, head, role, U);
        for (int i = 0; i < dim; ++i) {
            double p = (double)codes[b * dim + i];
            if (lattice == HQO_A2 && i == 0) p *= sqrt(3.0);
            u[b * dim + i] = sc * (p - (double)U[i]);
        }
    }
    if (norm_bits == 0) for (int i = 0; i < d; ++i) u[i] = 0.0;
    if (rotation == 1)
        for (int i = 0; i < d; ++i) u[i] = (S[i] < 0) ? -u[i] : u[i];
    if (rotation == 2) { /* S^T (eq.(2)): u_j <- sum_i Q_ij u_i */
        double r[1024];
        for (int j = 0; j < d; ++j) {
            double acc = 0.0;
            for (int i = 0; i < d; ++i) acc += (double)Q[i * d + j] * u[i];
            r[j] = acc;
        }
        memcpy(u, r, (size_t)d * sizeof(double));
    }
    rht_inverse_f64(u, D, d, out);
}
void hqo_kv_reconstruct_q(const int8_t* codes, const uint16_t* norms, int64_t n_tok, int heads, int d, int64_t token0,
                          int role, int lattice, double snr_db, int rotation, int dither, uint64_t seed, const float* Q,
                          double* out);
void hqo_kv_reconstruct(const int8_t* codes /*[n_tok,heads,d]*/, const uint16_t* norms, int64_t n_tok,
                        int heads, int d, int64_t token0, int role, int lattice, double snr_db,
                        int rotation, int dither, uint64_t seed, double* out /*[n_tok,heads,d]*/) {
    hqo_kv_reconstruct_q(codes, norms, n_tok, heads, d, token0, role, lattice, snr_db, rotation, dither, seed, NULL, out);
}
void hqo_kv_reconstruct_q(const int8_t* codes /*[n_tok,heads,d]*/, const uint16_t* norms, int64_t n_tok,
                          int heads, int d, int64_t token0, int role, int lattice, double snr_db,
                          int rotation, int dither, uint64_t seed, const float* Q, double* out /*[n_tok,heads,d]*/) {
    double inv_A = 1.0 / (hqo_alpha(lattice, snr_db) * sqrt((double)d));
    int8_t *D = (int8_t*)malloc((size_t)d), *S = (int8_t*)malloc((size_t)d);
    hqo_signs(seed, 1u, d, D);
    hqo_signs(seed, 2u, d, S);
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < n_tok; ++t)
        for (int h = 0; h < heads; ++h)
            kv_reconstruct(codes + (t * heads + h) * d, norms[t * heads + h], d, lattice, inv_A,
                           rotation, dither, seed, (uint32_t)(token0 + t), (uint32_t)h,
                           (uint32_t)role, D, S, Q, out + (t * heads + h) * d);
    free(D); free(S);
}

/* O4: textbook attention (L178) in double over reconstructed K̂,V̂ [T,heads,d]; the last `window`
 * tokens are taken from exact (bf16-valued) K,V instead (L562).  q [q_heads, d]. */
void hqo_attend(const double* Khat, const double* Vhat, const float* Kexact, const float* Vexact,
                int64_t T, int heads, int d, int window, const float* q, int q_heads,
                double* out /*[q_heads,d]*/) {
    int gsz = q_heads / heads;
    int64_t w0 = T - window < 0 ? 0 : T - window;
#pragma omp parallel for schedule(static)
    for (int qh = 0; qh < q_heads; ++qh) {
        int h = qh / gsz;
        double* s = (double*)malloc((size_t)T * sizeof(double));
        double mx = -INFINITY, den = 0.0;
        for (int64_t t = 0; t < T; ++t) {
            double dot = 0.0;
            for (int i = 0; i < d; ++i) {
                double kk = (t >= w0) ? (double)Kexact[(t * heads + h) * d + i]
                                      : Khat[(t * heads + h) * d + i];
                dot += (double)q[qh * d + i] * kk;
            }
            s[t] = dot / sqrt((double)d);
            if (s[t] > mx) mx = s[t];
        }
        for (int64_t t = 0; t < T; ++t) { s[t] = exp(s[t] - mx); den += s[t]; }
        for (int i = 0; i < d; ++i) {
            double a = 0.0;
            for (int64_t t = 0; t < T; ++t) {
                double vv = (t >= w0) ? (double)Vexact[(t * heads + h) * d + i]
                                      : Vhat[(t * heads + h) * d + i];
                a += s[t] * vv;
            }
            out[qh * d + i] = a / den;
        }
        free(s);
    }
}

/* ------------------------------------------------------------------------------------------ */
/* Calibration helper (B.1 L857): quantize iid-Gaussian tiles at one SNR; report realized SNR.   */
/* tiles [nt, n] fp32 ~ N(0,1) are the "post-RHT" vectors themselves (no RHT applied).          */
/* ------------------------------------------------------------------------------------------ */
void hqo_calib_quantize(const float* tiles, int64_t nt, int n, int lattice, double snr_db,
                        int8_t* codes, double* sig_pow, double* err_pow) {
    float A = (float)(hqo_alpha(lattice, snr_db) * sqrt((double)n));
    double inv_A = 1.0 / (hqo_alpha(lattice, snr_db) * sqrt((double)n));
    double sp = 0.0, ep = 0.0;
#pragma omp parallel for reduction(+ : sp, ep) schedule(static)
    for (int64_t t = 0; t < nt; ++t) {
        uint16_t nb;
        quantize_tile(lattice, n, A, tiles + t * n, 0, 0, 0, 0, 0, codes + t * n, &nb);
        double sc = (double)f16_bits_to_f32(nb) * inv_A;
        for (int i = 0; i < n; ++i) {
            double p = (double)codes[t * n + i];
            if (lattice == HQO_A2 && (i & 1) == 0) p *= sqrt(3.0);
            double x = (double)tiles[t * n + i], e = x - sc * p;
            sp += x * x;
            ep += e * e;
        }
    }
    *sig_pow = sp;
    *err_pow = ep;
}
