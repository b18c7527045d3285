// hq_encode.cu — the encode half of HyperQuant's hot path:
//   RHT (§3.1 eq.(1), §4.1) -> rotate (§4.2, KV) -> l2-normalize (§4.3) ->
//   subtractive dither (§4.4, KV) -> nearest lattice point (§4.5) -> strip + zig-zag
//   (§4.6) -> Rice code (§3.3, §4.7) into the FORMAT §5/§6 containers,
//   and the activation path RHT -> amax INT8 cast (FORMAT R7).
// All float arithmetic that decides an integer uses __f*_rn intrinsics (no FMA contraction) in
// the fixed operation order of docs/FORMAT.md §2.
#include "hq_common.cuh"
#include "hq_act.cuh"
#include "hq_internal.h"
#include "hq_tc.cuh"

namespace hq {

// ---------------------------------------------------------------------------------------------
__global__ void k_signs(uint64_t seed, uint32_t stream_id, int64_t n, int8_t* out) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) out[i] = sign_bit(seed, stream_id, (uint32_t)i) ? -1 : 1;
}
void launch_signs(uint64_t seed, uint32_t stream_id, int64_t n, int8_t* out, cudaStream_t st) {
    k_signs<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(seed, stream_id, n, out);
}

// ---------------------------------------------------------------------------------------------
// One warp transforms one tile held in shared memory: FORMAT R1 (butterflies, ascending stride).
// ---------------------------------------------------------------------------------------------
__device__ inline void warp_rht_inplace(float* s, int n, int lane) {
    for (int h = 1; h < n; h <<= 1) {
        __syncwarp();
        for (int p = lane; p < n / 2; p += 32) {
            int i = ((p / h) * 2 * h) + (p % h);
            float a = s[i], b = s[i + h];
            s[i] = __fadd_rn(a, b);
            s[i + h] = __fsub_rn(a, b);
        }
    }
    __syncwarp();
    float cn = (float)(1.0 / sqrt((double)n));
    for (int i = lane; i < n; i += 32) s[i] = __fmul_rn(s[i], cn);
    __syncwarp();
}

// FORMAT R2 tree sum of t[0..n) (destroys t); all lanes return the result.
__device__ inline float warp_treesum(float* t, int n, int lane) {
    for (int h = 1; h < n; h <<= 1) {
        __syncwarp();
        for (int p = lane; p * 2 * h < n; p += 32) {
            int i = p * 2 * h;
            t[i] = __fadd_rn(t[i], t[i + h]);
        }
    }
    __syncwarp();
    return t[0];
}

__device__ inline float load_elem(const void* p, int dtype, int64_t idx) {
    if (dtype == HQ_BF16) return __bfloat162float(((const __nv_bfloat16*)p)[idx]);
    return ((const float*)p)[idx];
}

// quantize the normalized tile u[0..n) (smem) into codes; lanes take lattice blocks round-robin.
// Returns per-lane clamp count; accumulates per-lane auto-k totals into tot[2][8] if tot != nullptr.
template <int LAT>
__device__ inline int quantize_blocks(const float* u, int n, float g, bool with_dither, uint64_t seed,
                                      uint32_t token, uint32_t head, uint32_t role, int8_t* codes, int lane,
                                      unsigned long long* tot) {
    int clamps = 0;
    for (int b = lane; b < n / LAT; b += 32) {
        float y[LAT];
        int c[LAT];
#pragma unroll
        for (int i = 0; i < LAT; ++i) y[i] = __fmul_rn(u[b * LAT + i], g);
        if (with_dither) {
            float U[LAT];
            dither_block<LAT>(seed, (uint32_t)b, token, head, role, U);
#pragma unroll
            for (int i = 0; i < LAT; ++i) y[i] = __fadd_rn(y[i], U[i]);
        }
        clamps += clamp_block<LAT>(y);
        nearest_noclamp<LAT>(y, c);
#pragma unroll
        for (int i = 0; i < LAT; ++i) codes[b * LAT + i] = (int8_t)c[i];
        if (tot) {
            int z[LAT];
            strip<LAT>(c, z);
#pragma unroll
            for (int i = 0; i < LAT; ++i) {
                int a = sym_class(LAT, i);
#pragma unroll
                for (int kk = 0; kk < 8; ++kk) tot[a * 8 + kk] += (unsigned long long)(kk + 1 + (z[i] >> kk));
            }
        }
    }
    return clamps;
}

constexpr int QW_WARPS = 4;

// FORMAT R11 (qjl rotation, eq.(2)): u'_i = sum_j Q_ij u_j, accumulated in increasing j with one fused
// multiply-add per term (canonical: the result decides the codes).  u[n] in shared memory, one warp;
// qt = S transposed ([j][i]: the lanes' loads are coalesced and hit L1 - the matrix is 64 KB at d = 128).
__device__ __forceinline__ void warp_qjl_apply(float* u, int n, const float* __restrict__ qt, int lane) {
    float acc[8];   // n <= 256: outputs lane, lane + 32, ...
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k] = 0.0f;
    for (int j = 0; j < n; ++j) {
        const float uj = u[j];
#pragma unroll
        for (int k = 0; k < 8; ++k)
            if (k * 32 < n) acc[k] = __fmaf_rn(__ldg(qt + (int64_t)j * n + k * 32 + lane), uj, acc[k]);
    }
    __syncwarp();
#pragma unroll
    for (int k = 0; k < 8; ++k)
        if (k * 32 < n) u[k * 32 + lane] = acc[k];
    __syncwarp();
}

__global__ void k_transpose_f32(const float* __restrict__ a, float* __restrict__ at, int n) {
    const int i = blockIdx.x, j = threadIdx.x;   // at[j][i] = a[i][j]
    at[(int64_t)j * n + i] = a[(int64_t)i * n + j];
}
__global__ void k_set_u32(uint32_t* dst, uint32_t v) { *dst = v; }
void launch_set_u32(uint32_t* dst, uint32_t v, cudaStream_t st) { k_set_u32<<<1, 1, 0, st>>>(dst, v); }
void launch_transpose_f32(const float* a, float* at, int n, cudaStream_t st) { k_transpose_f32<<<n, n, 0, st>>>(a, at, n); }

// mode 0: weights (tile = (row, kt));  mode 1: KV (tile = (token, head), rotation, dither)
template <int LAT, int MODE>
__global__ void __launch_bounds__(QW_WARPS * 32)
k_quantize(const void* X, int dtype, int64_t n_tiles, int64_t n_kt, int64_t ld, int n, float A,
           const int8_t* dsign, const int8_t* ssign, int rotation, int dither, uint64_t seed, int64_t token0,
           int role, int H, int64_t max_tokens, int8_t* codes, uint16_t* norms, unsigned long long* counters,
           int want_totals, const float* qjl_t) {
    extern __shared__ float smem[];
    int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* u = smem + warp * 2 * n;
    float* t = u + n;
    unsigned long long tot[16];
    if (want_totals)
        for (int i = 0; i < 16; ++i) tot[i] = 0;
    unsigned long long clamps = 0;
    for (int64_t tile = blockIdx.x * (int64_t)QW_WARPS + warp; tile < n_tiles; tile += (int64_t)gridDim.x * QW_WARPS) {
        int64_t row = tile / n_kt, kt = tile % n_kt;  // KV: row = token, kt = head, n_kt = H
        int64_t src = (MODE == 0) ? row * ld + kt * n : tile * (int64_t)n;
        int64_t sgn0 = (MODE == 0) ? kt * n : 0;
        for (int i = lane; i < n; i += 32) {
            float x = load_elem(X, dtype, src + i);
            u[i] = (dsign[sgn0 + i] < 0) ? -x : x;
        }
        warp_rht_inplace(u, n, lane);
        if (MODE == 1 && rotation == HQ_ROT_SIGNS)
            for (int i = lane; i < n; i += 32)
                if (ssign[i] < 0) u[i] = -u[i];
        if (MODE == 1 && rotation == HQ_ROT_QJL) {
            __syncwarp();
            warp_qjl_apply(u, n, qjl_t, lane);
        }
        for (int i = lane; i < n; i += 32) t[i] = __fmul_rn(u[i], u[i]);
        float ss = warp_treesum(t, n, lane);
        float rho32 = __fsqrt_rn(ss);
        uint16_t hb = f32_to_f16_bits_sat(rho32);
        float rho = f16_bits_to_f32(hb);
        int8_t* out = codes + tile * (int64_t)n;
        if (MODE == 0) out = codes + row * (n_kt * n) + kt * n;
        if (lane == 0) {
            if (MODE == 0) norms[row * n_kt + kt] = hb;
            else norms[kt * max_tokens + token0 + row] = hb;
        }
        if (rho == 0.0f) {  // G18
            for (int i = lane; i < n; i += 32) out[i] = 0;
            if (want_totals && lane == 0)  // n zero symbols: k+1 bits each
                for (int j = 0; j < n; ++j)
                    for (int kk = 0; kk < 8; ++kk) tot[sym_class(LAT, j % LAT) * 8 + kk] += kk + 1;
        } else {
            float g = __fdiv_rn(A, rho);
            clamps += quantize_blocks<LAT>(u, n, g, MODE == 1 && dither, seed, (uint32_t)(token0 + row),
                                           (uint32_t)kt, (uint32_t)role, out, lane, want_totals ? tot : nullptr);
        }
        __syncwarp();
    }
    // reduce counters over the warp, one atomic per warp per counter
    for (int o = 16; o; o >>= 1) clamps += __shfl_xor_sync(0xffffffffu, clamps, o);
    if (lane == 0 && clamps) atomicAdd(&counters[0], clamps);
    if (want_totals) {
        for (int i = 0; i < 16; ++i) {
            unsigned long long v = tot[i];
            for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0 && v) atomicAdd(&counters[1 + i], v);
        }
    }
}

template <int MODE>
static void launch_quantize_any(int lattice, dim3 grid, size_t smem, cudaStream_t st, const void* X, int dtype,
                                int64_t n_tiles, int64_t n_kt, int64_t ld, int n, float A, const int8_t* dsign,
                                const int8_t* ssign, int rotation, int dither, uint64_t seed, int64_t token0,
                                int role, int H, int64_t max_tokens, int8_t* codes, uint16_t* norms,
                                unsigned long long* counters, int want_totals, const float* qjl_t = nullptr) {
#define HQ_LAUNCH_Q(L)                                                                                        \
    k_quantize<L, MODE><<<grid, QW_WARPS * 32, smem, st>>>(X, dtype, n_tiles, n_kt, ld, n, A, dsign, ssign,   \
                                                           rotation, dither, seed, token0, role, H,           \
                                                           max_tokens, codes, norms, counters, want_totals, qjl_t)
    switch (lattice) {
        case LAT_Z: HQ_LAUNCH_Q(LAT_Z); break;
        case LAT_A2: HQ_LAUNCH_Q(LAT_A2); break;
        case LAT_D4: HQ_LAUNCH_Q(LAT_D4); break;
        default: HQ_LAUNCH_Q(LAT_E8); break;
    }
#undef HQ_LAUNCH_Q
}

void launch_quantize_weights(const void* W, int dtype, int64_t m, int64_t n_in, int64_t ld, int lattice, int n,
                             float A, const int8_t* dsign, int8_t* codes, uint16_t* norms,
                             unsigned long long* counters, cudaStream_t st) {
    int64_t n_kt = n_in / n, n_tiles = m * n_kt;
    int64_t blocks = (n_tiles + QW_WARPS - 1) / QW_WARPS;
    if (blocks > 148 * 16) blocks = 148 * 16;
    launch_quantize_any<0>(lattice, dim3((unsigned)blocks), QW_WARPS * 2 * n * sizeof(float), st, W, dtype, n_tiles,
                           n_kt, ld, n, A, dsign, nullptr, 0, 0, 0, 0, 0, 0, 0, codes, norms, counters, 1);
}

void launch_quantize_kv(const void* x, int64_t n_tok, int H, int d, int64_t token0, int role, int lattice,
                        float A, int rotation, int dither, uint64_t seed, const int8_t* dsign,
                        const int8_t* ssign, int8_t* codes, uint16_t* norm_out, int64_t max_tokens,
                        unsigned long long* counters, cudaStream_t st, const float* qjl_t) {
    int64_t n_tiles = n_tok * H;
    int64_t blocks = (n_tiles + QW_WARPS - 1) / QW_WARPS;
    if (blocks > 148 * 16) blocks = 148 * 16;
    launch_quantize_any<1>(lattice, dim3((unsigned)blocks), QW_WARPS * 2 * d * sizeof(float), st, x, HQ_BF16,
                           n_tiles, H, 0, d, A, dsign, ssign, rotation, dither, seed, token0, role, H, max_tokens,
                           codes, norm_out, counters, 0, qjl_t);
}

// ---------------------------------------------------------------------------------------------
// Activations (FORMAT R7): RHT, amax, INT8 cast.  One warp per (row, tile).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(QW_WARPS * 32)
k_act_quant(const void* X, int dtype, int64_t n_tiles, int64_t n_kt, int64_t ldx, int lattice, int n,
            const int8_t* dsign, int8_t* q, float* s_x, float* u_out) {
    extern __shared__ float smem[];
    int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* u = smem + warp * n;
    for (int64_t tile = blockIdx.x * (int64_t)QW_WARPS + warp; tile < n_tiles; tile += (int64_t)gridDim.x * QW_WARPS) {
        int64_t b = tile / n_kt, kt = tile % n_kt;
        for (int i = lane; i < n; i += 32) {
            float x = load_elem(X, dtype, b * ldx + kt * n + i);
            u[i] = (dsign[kt * n + i] < 0) ? -x : x;
        }
        warp_rht_inplace(u, n, lane);
        int64_t o = b * (n_kt * n) + kt * n;
        if (u_out)
            for (int i = lane; i < n; i += 32) u_out[o + i] = u[i];
        float amax = 0.0f;
        for (int i = lane; i < n; i += 32) {
            float v = u[i];
            if (lattice == LAT_A2 && (i & 1) == 0) { v = __fmul_rn(v, HQ_S3); u[i] = v; }
            amax = fmaxf(amax, fabsf(v));
        }
        for (int s = 16; s; s >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, s));
        __syncwarp();
        if (amax == 0.0f) {
            for (int i = lane; i < n; i += 32) q[o + i] = 0;
            if (lane == 0) s_x[b * n_kt + kt] = 0.0f;
        } else {
            float inv = __fdiv_rn(127.0f, amax);
            for (int i = lane; i < n; i += 32) {
                float v = rintf(__fmul_rn(u[i], inv));
                v = fminf(fmaxf(v, -127.0f), 127.0f);
                q[o + i] = (int8_t)(int)v;
            }
            if (lane == 0) s_x[b * n_kt + kt] = __fdiv_rn(amax, 127.0f);
        }
        __syncwarp();
    }
}

// Same arithmetic as k_act_quant, output as the B operand tiles of the E8 fused kernel: for batch tile bt and
// K-tile kt a blob of NB rows x 128 bytes in K-major SWIZZLE_128B order, the K index permuted like the decoded
// weights (e8_kcol: 32c + 4i + b for block 4c+b, coordinate i), followed by NB fp32 scales s_x.  n = 128.
__global__ void __launch_bounds__(QW_WARPS * 32)
k_act_blob(const void* X, int dtype, int64_t B, int64_t n_kt, int64_t ldx, const int8_t* dsign, int NB,
           uint8_t* bblob, int fp8) {
    // The tile lives in registers: lane l holds elements 4l .. 4l+3.  FORMAT R1's butterflies (ascending stride, a+b to
    // the lower index, a-b to the upper) are two in-register stages and five shuffle stages: the same additions on the
    // same pairs as warp_rht_inplace, so the result is bit-identical to k_act_quant.
    extern __shared__ float smem[];
    griddep_launch();
    griddep_wait();   // x comes from the previous kernel; the blob area is read by the previous hq_linear
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint8_t* srow = (uint8_t*)smem + warp * 128;          // one operand row, K order of the operand (e8_kcol)
    const int64_t n_bt = (B + NB - 1) / NB, n_tiles = n_bt * NB * n_kt;
    const uint32_t blob_bytes = (uint32_t)(NB * 128 + NB * 4);
    const bool vec = dtype == HQ_BF16 ? ((((uintptr_t)X) | (uintptr_t)(ldx * 2)) & 7) == 0
                                      : ((((uintptr_t)X) | (uintptr_t)(ldx * 4)) & 15) == 0;
    // the four codes of this lane go to operand columns colb + 4j (block l>>1, coordinates 4(l&1) .. +3)
    const int colb = act_col0(lane);
    const uint32_t n_kt32 = (uint32_t)n_kt, NB32 = (uint32_t)NB;   // n_tiles < 2^32 (see launch_act_blob)
    // (row, K-tile) of the tile advances by the grid stride without a division per tile
    const uint32_t stride = gridDim.x * (uint32_t)QW_WARPS;
    const uint32_t st_b = stride / n_kt32, st_k = stride - st_b * n_kt32;
    const int nb_sh = (NB32 & (NB32 - 1u)) == 0u ? __ffs((int)NB32) - 1 : -1;
    uint32_t b32 = (blockIdx.x * (uint32_t)QW_WARPS + warp) / n_kt32;   // b runs over the padded batch n_bt*NB
    uint32_t kt32 = (blockIdx.x * (uint32_t)QW_WARPS + warp) - b32 * n_kt32;
    for (int64_t tile = blockIdx.x * (int64_t)QW_WARPS + warp; tile < n_tiles; tile += stride,
                 kt32 += st_k, b32 += st_b + (kt32 >= n_kt32 ? 1u : 0u), kt32 -= (kt32 >= n_kt32 ? n_kt32 : 0u)) {
        const int64_t b = b32, kt = kt32;
        const int64_t bt = nb_sh >= 0 ? (b32 >> nb_sh) : (b32 / NB32);
        const int bb = (int)(b32 - (uint32_t)bt * NB32);
        uint8_t* blob = bblob + (bt * n_kt + kt) * (int64_t)blob_bytes;
        float x[4] = {0.0f, 0.0f, 0.0f, 0.0f};
        int qv4[4] = {0, 0, 0, 0};
        float sx = 0.0f;
        if (b < B) {
            const int64_t base = b * ldx + kt * 128 + 4 * lane;
            if (vec && dtype == HQ_BF16) {
                const uint2 v = __ldg((const uint2*)((const __nv_bfloat16*)X + base));
                x[0] = __uint_as_float(v.x << 16); x[1] = __uint_as_float(v.x & 0xffff0000u);
                x[2] = __uint_as_float(v.y << 16); x[3] = __uint_as_float(v.y & 0xffff0000u);
            } else if (vec) {
                const float4 v = __ldg((const float4*)((const float*)X + base));
                x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
            } else {
#pragma unroll
                for (int j = 0; j < 4; ++j) x[j] = load_elem(X, dtype, base + j);
            }
            const uint32_t sg = __ldg((const uint32_t*)(dsign + kt * 128) + lane);
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if ((sg >> (8 * j)) & 0x80u) x[j] = -x[j];
            sx = fp8 ? warp_act_tile128_fp8(x, lane, qv4) : warp_act_tile128(x, lane, qv4);   // FORMAT R7 or R12
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) srow[colb + 4 * j] = (uint8_t)qv4[j];
        __syncwarp();
        // one coalesced 128-byte row: lane l owns operand columns 4l .. 4l+3 = 16-byte chunk l>>2 (swizzled), word l&3
        const uint32_t w4 = ((const uint32_t*)srow)[lane];
        *(uint32_t*)(blob + (bb >> 3) * 1024 + (bb & 7) * 128 + ((((lane >> 2) ^ (bb & 7)) << 4) | ((lane & 3) << 2))) = w4;
        if (lane == 0) ((float*)(blob + NB * 128))[bb] = sx;
        __syncwarp();
    }
}

// The same for RHT tiles of 256 (the large-M path at n_tile = 256).  A half-warp owns one tile: lane l of the half holds the
// 16 contiguous elements 16l .. 16l+15 and runs the butterflies of strides 1, 2, 4, 8 in registers; a 16 x 16 transpose
// through shared memory gives it elements l, 16 + l, ..., 240 + l for the strides 16 .. 128 - the same pairs in the same
// ascending-stride order as FORMAT R1, so the fp32 results are bit-identical to the shuffle butterfly of k_act_blob.
// The 16 values live as eight f32x2 register pairs {v[j], v[j+8]} from the load to the INT8 cast: butterflies between
// pairs are packed adds (IEEE round-to-nearest per element), the one inside the pairs is scalar.  The tile leaves as TWO
// operand chunks of 128 K-bytes (chunk = block / 16; K index inside a chunk 32c + 4i + b for block 4c + b, coordinate i),
// each followed by the NB scales s_x of the whole tile: blob index = (bt * n_kt256 + kt) * 2 + chunk.  Lanes l and l ^ 8
// hold the four bytes of every operand word between them: one exchange of two registers.
constexpr int A256_WARPS = 8;
constexpr int A256_CTAS = 4;        // per SM (64 registers x 256 threads)
constexpr int A256_WFLOATS = 592;   // per warp: two 16 x 18 float transposition buffers, the second shifted by 16 banks
__device__ __forceinline__ uint64_t a256_pack(uint32_t lo, uint32_t hi) { uint64_t r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi)); return r; }
__device__ __forceinline__ void a256_unpack(uint64_t v, float& lo, float& hi) {
    uint32_t a, b;
    asm("mov.b64 {%0, %1}, %2;" : "=r"(a), "=r"(b) : "l"(v));
    lo = __uint_as_float(a); hi = __uint_as_float(b);
}
__device__ __forceinline__ uint64_t a256_add2(uint64_t a, uint64_t b) { uint64_t r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ uint64_t a256_sub2(uint64_t a, uint64_t b) { uint64_t r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ uint64_t a256_mul2(uint64_t a, uint64_t b) { uint64_t r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
// sign bytes (+-1 as int8) -> sign-bit masks: prmt's replicate mode turns the selected byte into 0x00 / 0xff
template <uint32_t SEL>
__device__ __forceinline__ uint32_t a256_signs(uint32_t sgw) { uint32_t r; asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(sgw), "r"(0u), "n"(SEL)); return r; }
// four butterfly stages on the 16 values {P[j].lo = v[j], P[j].hi = v[j+8]}: index bits 0, 1, 2 between pairs, bit 3 inside
__device__ __forceinline__ void a256_fwht16(uint64_t* P) {
#pragma unroll
    for (int h = 1; h < 8; h <<= 1)
#pragma unroll
        for (int i = 0; i < 8; ++i)
            if (!(i & h)) {
                const uint64_t a = P[i], c = P[i + h];
                P[i] = a256_add2(a, c); P[i + h] = a256_sub2(a, c);
            }
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        float a, c;
        a256_unpack(P[j], a, c);
        P[j] = a256_pack(__float_as_uint(__fadd_rn(a, c)), __float_as_uint(__fsub_rn(a, c)));
    }
}

struct A256Raw { uint4 a, b, sg; };   // a lane's 16 bf16 elements and their 16 sign bytes

template <bool FAST, bool FP8>   // FAST: bf16 rows whose 16-element groups can be read as 16-byte words; FP8: E4M3 cast (FORMAT R12)
__global__ void __launch_bounds__(A256_WARPS * 32, A256_CTAS)
k_act_blob256(const void* X, int dtype, int64_t B, int64_t n_kt, int64_t ldx, const int8_t* dsign, int NB, uint8_t* bblob) {
    extern __shared__ float smem[];
    griddep_launch();
    griddep_wait();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, half = lane >> 4, l = lane & 15, hi8 = (l >> 3) & 1;
    float* tr = smem + warp * A256_WFLOATS + half * 304;
    const uint32_t n_kt32 = (uint32_t)n_kt, npr = (n_kt32 + 1u) >> 1, NB32 = (uint32_t)NB;
    const uint32_t rows = (uint32_t)((B + NB - 1) / NB) * NB32;
    const uint32_t n_pairs = rows * npr, stride = gridDim.x * (uint32_t)A256_WARPS;   // < 2^32: checked by the launcher
    const uint32_t blob_bytes = NB32 * 128u + NB32 * 4u;
    constexpr bool fast = FAST;
    auto locate = [&](uint32_t pair, uint32_t& b32, uint32_t& kt) {
        b32 = pair / npr;
        kt = 2u * (pair - b32 * npr) + (uint32_t)half;
    };
    auto load_raw = [&](uint32_t b32, uint32_t kt, A256Raw& r) {
        if (fast && kt < n_kt32 && (int64_t)b32 < B) {
            const uint4* src = (const uint4*)((const __nv_bfloat16*)X + ((int64_t)b32 * ldx + (int64_t)kt * 256 + 16 * l));
            r.a = __ldg(src); r.b = __ldg(src + 1);
            r.sg = __ldg((const uint4*)(dsign + (int64_t)kt * 256) + l);
        }
    };
    uint32_t pair = blockIdx.x * (uint32_t)A256_WARPS + warp;
    uint32_t b32 = 0, kt = 0;
    A256Raw cur;
    cur.a = cur.b = cur.sg = make_uint4(0u, 0u, 0u, 0u);
    if (pair < n_pairs) { locate(pair, b32, kt); load_raw(b32, kt, cur); }
    while (pair < n_pairs) {
        const uint32_t pair_n = pair + stride < pair ? 0xffffffffu : pair + stride;
        uint32_t b32_n = 0, kt_n = 0;
        A256Raw nxt;
        nxt.a = nxt.b = nxt.sg = make_uint4(0u, 0u, 0u, 0u);
        if (pair_n < n_pairs) { locate(pair_n, b32_n, kt_n); load_raw(b32_n, kt_n, nxt); }   // in flight behind this pair's arithmetic
        const bool tile_on = kt < n_kt32;                        // an odd tile count leaves the last pair's second half idle
        const bool row_on = tile_on && (int64_t)b32 < B;         // rows past B pad the batch tile with zeros
        uint64_t P[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) P[j] = 0ull;
        if (row_on) {
            if (fast) {
                const uint32_t wa[4] = {cur.a.x, cur.a.y, cur.a.z, cur.a.w}, wb[4] = {cur.b.x, cur.b.y, cur.b.z, cur.b.w};
                const uint32_t sw[4] = {cur.sg.x, cur.sg.y, cur.sg.z, cur.sg.w};
#pragma unroll
                for (int e = 0; e < 4; ++e) {   // word e: elements 2e, 2e+1 (and 8 + 2e, 9 + 2e); sign bytes (2e) & 3, +1 of sw[e >> 1] (sw[2 + (e >> 1)])
                    uint32_t ma, mb;
                    if (e & 1) { ma = a256_signs<0xb4a4>(sw[e >> 1]); mb = a256_signs<0xb4a4>(sw[2 + (e >> 1)]); }
                    else       { ma = a256_signs<0x9484>(sw[e >> 1]); mb = a256_signs<0x9484>(sw[2 + (e >> 1)]); }
                    const uint32_t xa = wa[e] ^ (ma & 0x80008000u), xb = wb[e] ^ (mb & 0x80008000u);
                    P[2 * e] = a256_pack(xa << 16, xb << 16);
                    P[2 * e + 1] = a256_pack(xa & 0xffff0000u, xb & 0xffff0000u);
                }
            } else {
                const int64_t base = (int64_t)b32 * ldx + (int64_t)kt * 256 + 16 * l;
                const int8_t* sp = dsign + (int64_t)kt * 256 + 16 * l;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const float lo = load_elem(X, dtype, base + j), hi = load_elem(X, dtype, base + j + 8);
                    P[j] = a256_pack(__float_as_uint(sp[j] < 0 ? -lo : lo), __float_as_uint(sp[j + 8] < 0 ? -hi : hi));
                }
            }
        }
        a256_fwht16(P);                                          // strides 1, 2, 4, 8
        __syncwarp();                                            // the previous pair's reads of the buffer are done
#pragma unroll
        for (int j = 0; j < 8; ++j) *(uint64_t*)(tr + l * 18 + 2 * j) = P[j];   // value j at slot 2 (j & 7) + (j >> 3) of row l
        __syncwarp();
        {
            const float* col = tr + 2 * (l & 7) + (l >> 3);      // element 16 m + l: value l of row m
#pragma unroll
            for (int j = 0; j < 8; ++j) P[j] = a256_pack(__float_as_uint(col[j * 18]), __float_as_uint(col[(j + 8) * 18]));
        }
        a256_fwht16(P);                                          // strides 16, 32, 64, 128
        float amax = 0.0f;
        {
            const uint64_t cn = a256_pack(__float_as_uint(0.0625f), __float_as_uint(0.0625f));   // 1 / sqrt(256)
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                P[j] = a256_mul2(P[j], cn);
                float a, c;
                a256_unpack(P[j], a, c);
                amax = fmaxf(amax, fmaxf(fabsf(a), fabsf(c)));
            }
        }
#pragma unroll
        for (int sft = 8; sft; sft >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, sft));   // inside the half-warp
        uint32_t pk[2][2] = {{0u, 0u}, {0u, 0u}};                // pk[chunk][jj]: codes of elements m = 8 chunk + 4 jj .. + 3 (x 16 + l)
        float sx = 0.0f;
        if (amax != 0.0f) {
            const float inv = __fdiv_rn(FP8 ? 448.0f : 127.0f, amax);
            const uint64_t inv2 = a256_pack(__float_as_uint(inv), __float_as_uint(inv));
            uint32_t qlo[8], qhi[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                float a, c;
                a256_unpack(a256_mul2(P[j], inv2), a, c);
                if (FP8) {   // byte 0 of qlo / qhi = e4m3(a) / e4m3(c): the packing below takes byte 0 only
                    const uint32_t r = f32x2_to_e4m3x2(a, c);
                    qlo[j] = r; qhi[j] = r >> 8;
                    continue;
                }
                // rint + clamp to +-127 + cast in one instruction: |x| <= amax bounds |x * inv| by 127 (1 + 2^-23), which
                // rounds to 127, so the saturating convert can never return -128 and equals FORMAT R7's clamp(rint(.))
                asm("cvt.rni.sat.s8.f32 %0, %1;" : "=r"(qlo[j]) : "f"(a));
                asm("cvt.rni.sat.s8.f32 %0, %1;" : "=r"(qhi[j]) : "f"(c));
            }
#pragma unroll
            for (int jj = 0; jj < 2; ++jj) {
                pk[0][jj] = __byte_perm(__byte_perm(qlo[4 * jj], qlo[4 * jj + 1], 0x0040), __byte_perm(qlo[4 * jj + 2], qlo[4 * jj + 3], 0x0040), 0x5410);
                pk[1][jj] = __byte_perm(__byte_perm(qhi[4 * jj], qhi[4 * jj + 1], 0x0040), __byte_perm(qhi[4 * jj + 2], qhi[4 * jj + 3], 0x0040), 0x5410);
            }
            sx = __fdiv_rn(amax, FP8 ? 448.0f : 127.0f);
        }
        // lane l (bit 3 clear) and lane l + 8 hold bytes {0, 2} and {1, 3} of every word: the low lane assembles chunk 0, the
        // high lane chunk 1
        uint32_t A[2], Bv[2];
#pragma unroll
        for (int jj = 0; jj < 2; ++jj) {
            const uint32_t keep = hi8 ? pk[1][jj] : pk[0][jj], send = hi8 ? pk[0][jj] : pk[1][jj];
            const uint32_t recv = __shfl_xor_sync(0xffffffffu, send, 8);
            A[jj] = hi8 ? recv : keep; Bv[jj] = hi8 ? keep : recv;
        }
        if (tile_on) {
            const uint32_t bt = b32 / NB32, bb = b32 - bt * NB32;
            uint8_t* blob = bblob + (((uint64_t)bt * n_kt32 + kt) * 2 + (uint32_t)hi8) * (uint64_t)blob_bytes;
            uint8_t* rowp = blob + (bb >> 3) * 1024 + (bb & 7) * 128 + ((l & 3) << 2);
#pragma unroll
            for (int pm = 0; pm < 4; ++pm) {   // word 8 pm + (l & 7) of the chunk row: 16-byte unit 2 pm + ((l & 7) >> 2)
                const uint32_t unit = 2u * pm + ((l & 7) >> 2);
                *(uint32_t*)(rowp + ((unit ^ (bb & 7)) << 4)) = __byte_perm(A[pm >> 1], Bv[pm >> 1], (pm & 1) ? 0x7362 : 0x5140);
            }
            if ((l & 7) == 0) ((float*)(blob + NB32 * 128u))[bb] = sx;   // both chunks carry the tile's scale
        }
        cur = nxt; pair = pair_n; b32 = b32_n; kt = kt_n;
    }
}

void launch_act_blob256(const void* x, int dtype, int64_t B, int64_t n_in, int64_t ldx, const int8_t* dsign, int NB,
                        uint8_t* bblob, cudaStream_t st, int fp8) {
    const int64_t n_kt = n_in / 256, n_bt = (B + NB - 1) / NB, n_pairs = n_bt * NB * ((n_kt + 1) / 2);
    int64_t blocks = (n_pairs + A256_WARPS - 1) / A256_WARPS;
    if (blocks > 148 * A256_CTAS) blocks = 148 * A256_CTAS;
    // n_pairs < 2^32 always: 2^32 pairs of 512 bf16 activations would be 4.4 TB of x
    const bool fast = dtype == HQ_BF16 && ((((uintptr_t)x) | (uintptr_t)(ldx * 2)) & 15) == 0;
#define HQ_A256(FAST_, FP8_)                                                                                                     \
    launch_pdl(k_act_blob256<FAST_, FP8_>, dim3((unsigned)blocks), dim3(A256_WARPS * 32), A256_WARPS * A256_WFLOATS * sizeof(float), \
               st, x, dtype, B, n_kt, ldx, dsign, NB, bblob)
    if (fast) { if (fp8) HQ_A256(true, true); else HQ_A256(true, false); }
    else { if (fp8) HQ_A256(false, true); else HQ_A256(false, false); }
#undef HQ_A256
}

void launch_act_blob(const void* x, int dtype, int64_t B, int64_t n_in, int64_t ldx, const int8_t* dsign, int NB,
                     uint8_t* bblob, cudaStream_t st, int fp8) {
    int64_t n_kt = n_in / 128, n_bt = (B + NB - 1) / NB, n_tiles = n_bt * NB * n_kt;
    int64_t blocks = (n_tiles + QW_WARPS - 1) / QW_WARPS;
    if (blocks > 148 * 16) blocks = 148 * 16;
    // n_tiles < 2^32 always: 2^32 tiles of 128 bf16 activations would be 1.1 TB of x
    launch_pdl(k_act_blob, dim3((unsigned)blocks), dim3(QW_WARPS * 32), QW_WARPS * 128 * sizeof(float), st, x, dtype, B, n_kt, ldx,
               dsign, NB, bblob, fp8);
}

void launch_act_quant(const void* x, int dtype, int64_t B, int64_t n_in, int64_t ldx, int lattice, int n,
                      const int8_t* dsign, int8_t* q, float* s_x, float* u, cudaStream_t st) {
    int64_t n_kt = n_in / n, n_tiles = B * n_kt;
    int64_t blocks = (n_tiles + QW_WARPS - 1) / QW_WARPS;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_act_quant<<<(unsigned)blocks, QW_WARPS * 32, QW_WARPS * n * sizeof(float), st>>>(x, dtype, n_tiles, n_kt, ldx,
                                                                                      lattice, n, dsign, q, s_x, u);
}

// ---------------------------------------------------------------------------------------------
// Tile lengths: thread per tile; symbols from the codes, ulen = n + sum q_j (FORMAT §4).
// ---------------------------------------------------------------------------------------------
template <int LAT>
__device__ inline uint32_t tile_ulen(const int8_t* codes, int n, int k0, int k1) {
    uint32_t L = (uint32_t)n;
    for (int b = 0; b < n / LAT; ++b) {
        int c[LAT], z[LAT];
#pragma unroll
        for (int i = 0; i < LAT; ++i) c[i] = codes[b * LAT + i];
        strip<LAT>(c, z);
#pragma unroll
        for (int i = 0; i < LAT; ++i) L += (uint32_t)(z[i] >> (sym_class(LAT, i) ? k1 : k0));
    }
    return L;
}

constexpr uint32_t W_ULEN_MAX = 8160;  // FORMAT §5: 255 words per row

// ulen_tmp[sg*32 + i], sg = (rb*n_kt + kt)*4 + w, row = 128 rb + 32 w + i (0 for absent rows)
template <int LAT>
__global__ void k_tile_ulen(const int8_t* codes, int64_t m, int64_t n_kt, int n, int k0, int k1, int64_t G,
                            uint16_t* ulen_tmp, int* err_flag) {
    int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;  // g*128 + (w*32 + i)
    if (idx >= G * 128) return;
    int64_t g = idx >> 7;
    int i = (int)(idx & 127);
    int64_t rb = g / n_kt, kt = g % n_kt, r = rb * 128 + i;
    uint32_t L = 0;
    if (r < m) {
        L = tile_ulen<LAT>(codes + r * (n_kt * n) + kt * n, n, k0, k1);
        if (L > W_ULEN_MAX) { atomicExch(err_flag, 1); L = W_ULEN_MAX; }
        // err_flag[4] tracks 65535 - (shortest U-section of a present row), warp-aggregated
        const unsigned am = __activemask();
        const uint32_t inv = __reduce_max_sync(am, 65535u - L);
        const uint32_t mx = __reduce_max_sync(am, L);   // err_flag[5]: the longest U-section (hq_weight_stats)
        if ((threadIdx.x & 31) == (__ffs(am) - 1)) {
            atomicMax((unsigned int*)err_flag + 4, inv);
            atomicMax((unsigned int*)err_flag + 5, mx);
        }
    }
    ulen_tmp[idx] = (uint16_t)L;
}

void launch_tile_ulen(const int8_t* codes, int64_t m, int64_t n_in, int lattice, int n, int k0, int k1,
                      uint16_t* ulen_tmp, int* err_flag, cudaStream_t st) {
    int64_t n_kt = n_in / n, n_rb = (m + 127) / 128, G = n_rb * n_kt;
    unsigned blocks = (unsigned)((G * 128 + 127) / 128);
    switch (lattice) {
        case LAT_Z: k_tile_ulen<LAT_Z><<<blocks, 128, 0, st>>>(codes, m, n_kt, n, k0, k1, G, ulen_tmp, err_flag); break;
        case LAT_A2: k_tile_ulen<LAT_A2><<<blocks, 128, 0, st>>>(codes, m, n_kt, n, k0, k1, G, ulen_tmp, err_flag); break;
        case LAT_D4: k_tile_ulen<LAT_D4><<<blocks, 128, 0, st>>>(codes, m, n_kt, n, k0, k1, G, ulen_tmp, err_flag); break;
        default: k_tile_ulen<LAT_E8><<<blocks, 128, 0, st>>>(codes, m, n_kt, n, k0, k1, G, ulen_tmp, err_flag); break;
    }
}

// ---------------------------------------------------------------------------------------------
// Sub-group offsets: device prefix sum over the sub-groups' sizes (north_star (a); FORMAT §5).
// One block; each thread sizes one sub-group from its 32 ulen, block scan in chunks of 1024.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024)
k_group_offsets(const uint16_t* ulen_tmp, int64_t G4, int rw_words, uint32_t* group_off, unsigned long long* totals,
                uint32_t* max_group16) {
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t carry_s;
    __shared__ unsigned long long ubits_total;
    __shared__ uint32_t maxg;
    int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) { carry_s = 0; ubits_total = 0; maxg = 0; }
    __syncthreads();
    for (int64_t base = 0; base < G4; base += 1024) {
        int64_t g = base + tid;
        uint32_t size16 = 0, ub = 0, uw = 0;
        if (g < G4) {
            const uint4* p = (const uint4*)(ulen_tmp + g * 32);  // 64 bytes
            for (int v = 0; v < 4; ++v) {
                uint4 w = p[v];
                uint32_t ws[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    uint32_t a = ws[e] & 0xffffu, b = ws[e] >> 16;
                    ub += a + b;
                    uw += ((a + 31) >> 5) + ((b + 31) >> 5);
                }
            }
            size16 = (128 + 4 * ((uint32_t)rw_words * 32 + uw) + 15) / 16;
        }
        uint32_t x = size16;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_sums[warp] = x;
        __syncthreads();
        if (warp == 0) {
            uint32_t sv = warp_sums[lane];
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t y = __shfl_up_sync(0xffffffffu, sv, o);
                if (lane >= o) sv += y;
            }
            warp_sums[lane] = sv;
        }
        __syncthreads();
        uint32_t incl = x + (warp ? warp_sums[warp - 1] : 0) + carry_s;
        if (g < G4) {
            group_off[g] = incl - size16;
            atomicAdd(&ubits_total, (unsigned long long)ub);
            atomicMax(&maxg, size16);
        }
        __syncthreads();
        if (tid == 1023) carry_s = incl;
        __syncthreads();
    }
    if (tid == 0) {
        group_off[G4] = carry_s;
        totals[0] = ubits_total;
        *max_group16 = maxg;
    }
}

void launch_group_offsets(const uint16_t* ulen_tmp, int64_t G4, int rw_words, uint32_t* group_off,
                          unsigned long long* totals, uint32_t* max_group16, cudaStream_t st) {
    k_group_offsets<<<1, 1024, 0, st>>>(ulen_tmp, G4, rw_words, group_off, totals, max_group16);
}

// ---------------------------------------------------------------------------------------------
// Bit packing.  A per-thread writer that assembles the 32-bit words of an MSB-first stream and hands
// every non-zero word to `store(word_index, value)` exactly once (destinations are zero-initialized).
// ---------------------------------------------------------------------------------------------
template <class Store>
struct BitWriter {
    Store store;
    uint32_t pos;   // next stream bit
    uint32_t cur;   // bits of the current word accumulated so far (already positioned)
    __device__ BitWriter(Store s, uint32_t p) : store(s), pos(p), cur(0) {}
    __device__ inline void flush_word() {
        if (cur) store((pos - 1) >> 5, cur);
        cur = 0;
    }
    // append nb (1..32) bits, value MSB-first
    __device__ inline void put(uint32_t v, int nb) {
        int sft = pos & 31;
        int room = 32 - sft;
        if (nb <= room) {
            cur |= (nb == 32) ? v : (v << (room - nb));
            pos += nb;
            if ((pos & 31) == 0) flush_word();
        } else {
            cur |= v >> (nb - room);
            pos += room;
            flush_word();
            int rest = nb - room;
            cur = v << (32 - rest);
            pos += rest;
        }
    }
    __device__ inline void skip(uint32_t nzeros) {  // append zeros
        uint32_t np = pos + nzeros;
        if ((np >> 5) != (pos >> 5)) {
            if (pos & 31) { pos = (pos | 31) + 1; flush_word(); }
        }
        pos = np;
    }
    __device__ inline void finish() {
        if (pos & 31) { if (cur) store(pos >> 5, cur); cur = 0; }
    }
};
struct StoreAtomicOr {  // streams that share boundary words with their neighbours (KV container, FORMAT §6)
    uint32_t* area;
    __device__ inline void operator()(uint32_t i, uint32_t v) const { atomicOr(&area[i], v); }
};

// R-section of a tile (FORMAT §4 field planes) from its symbols z[0..n) in stream order.
template <int LAT, class BW>
__device__ inline void write_R(BW& bw, const uint8_t* z, int n, int k0, int k1) {
    const int nclass = (LAT == LAT_D4 || LAT == LAT_A2) ? 2 : 1;
    for (int a = 0; a < nclass; ++a) {
        int ka = a ? k1 : k0;
        if (ka == 0) continue;
        int na = class_count(LAT, n, a);
        // stream position of the m-th symbol of class a
        auto sym_at = [&](int mi) -> uint32_t {
            int j;
            if (LAT == LAT_D4) j = a ? 4 * mi + 3 : (mi / 3) * 4 + (mi % 3);
            else if (LAT == LAT_A2) j = 2 * mi + a;
            else j = mi;
            return (uint32_t)z[j] & ((1u << ka) - 1u);
        };
        for (int ch = 0; ch * 32 < na; ++ch) {
            int cnt = min(32, na - ch * 32);
            int lo = 0;
            for (int b = 0; b < 3; ++b) {
                int wd = 1 << b;
                if (!(ka & wd)) continue;
                if (cnt == 32) {
                    int per = 8 / wd;
                    for (int i = 0; i < wd; ++i) {
                        uint32_t V = 0;
                        for (int u = 0; u < 32; ++u) {
                            int g = 2 * (u >> 3) + (u & 1), lane = (u & 7) >> 1;
                            if (g / per != i) continue;
                            uint32_t f = (sym_at(ch * 32 + u) >> lo) & ((1u << wd) - 1u);
                            V |= f << (8 * lane + wd * (g % per));
                        }
                        bw.put(V, 32);
                    }
                } else {
                    for (int u = 0; u < cnt; ++u) bw.put((sym_at(ch * 32 + u) >> lo) & ((1u << wd) - 1u), wd);
                }
                lo += wd;
            }
        }
    }
    bw.finish();
}

template <int LAT, class BW>
__device__ inline void write_U(BW& bw, const uint8_t* z, int n, int k0, int k1) {
    for (int j = 0; j < n; ++j) {
        uint32_t q = (uint32_t)z[j] >> (sym_class(LAT, j) ? k1 : k0);
        bw.skip(q);
        bw.put(1u, 1);
    }
    bw.finish();
}

// symbols of a tile in stream order (FORMAT §3)
template <int LAT>
__device__ inline void tile_symbols(const int8_t* codes, int n, uint8_t* z) {
    for (int b = 0; b < n / LAT; ++b) {
        int c[LAT], zz[LAT];
#pragma unroll
        for (int i = 0; i < LAT; ++i) c[i] = codes[b * LAT + i];
        strip<LAT>(c, zz);
#pragma unroll
        for (int i = 0; i < LAT; ++i) {  // <= 255 by the INT8 pre-clamp (G8)
            int p = (LAT == LAT_E8) ? 32 * (b >> 2) + 8 * (i >> 1) + 2 * (b & 3) + (i & 1) : b * LAT + i;
            z[p] = (uint8_t)zz[i];
        }
    }
}

// one block (128 threads = 128 rows = four sub-groups, one per warp) per (rb, kt); blob zero-initialized
constexpr uint32_t PACK_UCAP = 24;  // U words per row gathered through shared memory; longer rows go the slow way
template <int LAT>
__global__ void __launch_bounds__(128)
k_pack_groups(const int8_t* codes, const uint16_t* norms, const uint16_t* ulen_tmp, int64_t m, int64_t n_kt,
              int n, int k0, int k1, const uint32_t* group_off, uint8_t* blob) {
    extern __shared__ uint8_t zs[];  // [128][n+4] symbols (+4: de-conflict banks) | [128][PACK_UCAP+1] U words
    int64_t g = blockIdx.x;
    int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    int64_t rb = g / n_kt, kt = g % n_kt, r = rb * 128 + t;
    int rbits = rbits_of(LAT, n, k0, k1);
    int rw_words = (rbits + 31) / 32;
    uint8_t* base = blob + 16 * (int64_t)group_off[g * 4 + warp];
    uint16_t* h_ulen = (uint16_t*)base;
    uint16_t* h_norm = h_ulen + 32;
    uint32_t* rarea = (uint32_t*)(base + 128);
    uint32_t* uarea = rarea + rw_words * 32;
    const uint16_t* ulen_sg = ulen_tmp + (g * 4 + warp) * 32;
    uint32_t ul = ulen_sg[lane];
    uint32_t nw = (ul + 31) >> 5;
    h_ulen[lane] = (uint16_t)ul;
    h_norm[lane] = (r < m) ? norms[r * n_kt + kt] : (uint16_t)0;
    uint32_t* urow = (uint32_t*)(zs + 128 * (size_t)(n + 4)) + t * (PACK_UCAP + 1);
    for (uint32_t i = 0; i < PACK_UCAP; ++i) urow[i] = 0;
    if (r < m) {
        uint8_t* z = zs + t * (n + 4);
        tile_symbols<LAT>(codes + r * (n_kt * n) + kt * n, n, z);
        auto store_r = [&](uint32_t i, uint32_t v) { rarea[i * 32 + lane] = v; };
        BitWriter<decltype(store_r)> bwr(store_r, 0u);
        write_R<LAT>(bwr, z, n, k0, k1);
        auto store_u = [&](uint32_t i, uint32_t v) {
            if (i < PACK_UCAP) urow[i] = v;
            else uarea[u_word_index_slow(ulen_sg, lane, i)] = v;
        };
        BitWriter<decltype(store_u)> bwu(store_u, 0u);
        write_U<LAT>(bwu, z, n, k0, k1);
    }
    __syncwarp();
    // scatter the gathered words into the compacted word-rows
    uint32_t maxnw = nw;
#pragma unroll
    for (int o = 16; o; o >>= 1) maxnw = max(maxnw, __shfl_xor_sync(0xffffffffu, maxnw, o));
    uint32_t at = 0;
    for (uint32_t w = 0; w < min(maxnw, PACK_UCAP); ++w) {
        const bool has = nw > w;
        const uint32_t mk = __ballot_sync(0xffffffffu, has);
        if (has) uarea[at + __popc(mk & ((1u << lane) - 1u))] = urow[w];
        at += __popc(mk);
    }
}

void launch_pack_groups(const int8_t* codes, const uint16_t* norms, const uint16_t* ulen_tmp, int64_t m,
                        int64_t n_in, int lattice, int n, int k0, int k1, const uint32_t* group_off,
                        uint8_t* blob, cudaStream_t st) {
    int64_t n_kt = n_in / n, n_rb = (m + 127) / 128, G = n_rb * n_kt;
    size_t smem = 128 * (size_t)(n + 4) + 128 * (size_t)(PACK_UCAP + 1) * 4;
#define HQ_LAUNCH_P(L)                                                                                          \
    k_pack_groups<L><<<(unsigned)G, 128, smem, st>>>(codes, norms, ulen_tmp, m, n_kt, n, k0, k1, group_off, blob)
    switch (lattice) {
        case LAT_Z: HQ_LAUNCH_P(LAT_Z); break;
        case LAT_A2: HQ_LAUNCH_P(LAT_A2); break;
        case LAT_D4: HQ_LAUNCH_P(LAT_D4); break;
        default: HQ_LAUNCH_P(LAT_E8); break;
    }
#undef HQ_LAUNCH_P
}

// ---------------------------------------------------------------------------------------------
// KV container (FORMAT §6).  Phase 1: per-vector ulen; phase 2: per (role, head) sequential-chunk
// prefix over the new tokens (one warp per head), block offsets; phase 3: bit packing.
// ---------------------------------------------------------------------------------------------
// the cache's error flag lives in mapped host memory (hq_kv::flag): the host reads it without synchronizing
__device__ inline void kv_raise(int* flag, int code) {
    *(volatile int*)flag = code;
    __threadfence_system();
}
constexpr uint32_t KV_NO_ROOM = 0xffffffffu;   // ustart of a vector whose U-section is not stored

template <int LAT>
__global__ void k_kv_ulen(const int8_t* codes, int64_t n_tok, int H, int d, int64_t token0, int k0, int k1,
                          int64_t max_tokens, uint16_t* ulen /*[H][max_tokens] of this role*/, int* err_flag) {
    int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;  // t*H + h
    if (idx >= n_tok * H) return;
    int64_t t = idx / H;
    int h = (int)(idx % H);
    uint32_t L = tile_ulen<LAT>(codes + idx * d, d, k0, k1);
    if (L >= 65535u) { kv_raise(err_flag, 1); L = 65535u; }   // 65535 marks "does not fit" for k_kv_offsets
    ulen[h * max_tokens + token0 + t] = (uint16_t)L;
}

// one warp per head: ustart_tmp[h*n_tok + t] = U-stream bit position of token token0+t;
// updates upos[h], writes blk_off for every 128-token block that starts inside the range.
__global__ void k_kv_offsets(const uint16_t* ulen, int64_t n_tok, int H, int64_t token0, int64_t max_tokens,
                             int64_t n_blk, uint32_t* upos, uint32_t* blk_off, uint32_t* ustart_tmp,
                             int64_t una_bits, int* err_flag) {
    int h = blockIdx.x;
    int lane = threadIdx.x;
    uint64_t pos = upos[h];
    bool bad = false;
    for (int64_t t0 = 0; t0 < n_tok; t0 += 32) {
        int64_t t = t0 + lane;
        uint32_t L = (t < n_tok) ? ulen[h * max_tokens + token0 + t] : 0;
        uint64_t x = L;
        for (int o = 1; o < 32; o <<= 1) {
            uint64_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        const uint64_t start = pos + x - L;
        if (t < n_tok) {
            // a vector that does not fit (stream capacity, or a U-section past 65534 bits) is not written at all
            const bool fits = L < 65535u && start + L <= (uint64_t)una_bits;
            bad |= !fits;
            ustart_tmp[h * n_tok + t] = fits ? (uint32_t)start : KV_NO_ROOM;
            if (((token0 + t) & 127) == 0) blk_off[h * (n_blk + 1) + ((token0 + t) >> 7)] = (uint32_t)min(start, (uint64_t)una_bits);
        }
        pos += __shfl_sync(0xffffffffu, x, 31);
    }
    if (__any_sync(0xffffffffu, bad) && lane == 0) kv_raise(err_flag, 2);
    if (lane == 0) upos[h] = (uint32_t)min(pos, (uint64_t)una_bits + 1u);
}

template <int LAT>
__global__ void __launch_bounds__(128)
k_kv_pack(const int8_t* codes, int64_t n_tok, int H, int d, int64_t token0, int k0, int k1, int rbits,
          int64_t rem_words, int64_t una_words, uint32_t* rem, uint32_t* una, const uint32_t* ustart_tmp) {
    extern __shared__ uint8_t zs[];
    int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;  // t*H + h
    if (idx >= n_tok * H) return;
    int64_t t = idx / H;
    int h = (int)(idx % H);
    uint8_t* z = zs + threadIdx.x * (d + 4);
    tile_symbols<LAT>(codes + idx * d, d, z);
    BitWriter<StoreAtomicOr> bwr(StoreAtomicOr{rem + h * rem_words}, (uint32_t)((token0 + t) * rbits));
    write_R<LAT>(bwr, z, d, k0, k1);
    const uint32_t ustart = ustart_tmp[h * n_tok + t];
    if (ustart == KV_NO_ROOM) return;   // flagged by k_kv_offsets: nothing is written past the stream's capacity
    BitWriter<StoreAtomicOr> bwu(StoreAtomicOr{una + h * una_words}, ustart);
    write_U<LAT>(bwu, z, d, k0, k1);
}

void launch_kv_pack(const int8_t* codes, int64_t n_tok, int H, int d, int64_t token0, int role, int lattice,
                    int k0, int k1, int rbits, int64_t max_tokens, int64_t rem_words, int64_t una_words,
                    int64_t n_blk, uint32_t* rem, uint32_t* una, uint16_t* ulen, uint32_t* blk_off, uint32_t* upos,
                    int* err_flag, cudaStream_t st) {
    // role slices
    uint32_t* rem_r = rem + (int64_t)role * H * rem_words;
    uint32_t* una_r = una + (int64_t)role * H * una_words;
    uint16_t* ulen_r = ulen + (int64_t)role * H * max_tokens;
    uint32_t* blk_r = blk_off + (int64_t)role * H * (n_blk + 1);
    uint32_t* upos_r = upos + (int64_t)role * H;
    // ustart scratch lives right after the codes scratch (caller reserves n_tok*H u32 per role): we
    // reuse the tail of the codes buffer: codes is [n_tok*H*d] int8 and d >= 64, so allocate separately.
    uint32_t* ustart_tmp = (uint32_t*)(codes + n_tok * (int64_t)H * d);
    unsigned blocks = (unsigned)((n_tok * H + 127) / 128);
    size_t smem = 128 * (size_t)(d + 4);
#define HQ_KV(L)                                                                                                  \
    k_kv_ulen<L><<<blocks, 128, 0, st>>>(codes, n_tok, H, d, token0, k0, k1, max_tokens, ulen_r, err_flag);       \
    k_kv_offsets<<<H, 32, 0, st>>>(ulen_r, n_tok, H, token0, max_tokens, n_blk, upos_r, blk_r, ustart_tmp,        \
                                   una_words * 32 - 64, err_flag);                                                \
    k_kv_pack<L><<<blocks, 128, smem, st>>>(codes, n_tok, H, d, token0, k0, k1, rbits, rem_words, una_words,      \
                                            rem_r, una_r, ustart_tmp)
    switch (lattice) {
        case LAT_Z: HQ_KV(LAT_Z); break;
        case LAT_A2: HQ_KV(LAT_A2); break;
        case LAT_D4: HQ_KV(LAT_D4); break;
        default: HQ_KV(LAT_E8); break;
    }
#undef HQ_KV
}

__global__ void k_kv_ring(const __nv_bfloat16* k, const __nv_bfloat16* v, int64_t n_tok, int H, int d,
                          int64_t token0, int window, __nv_bfloat16* ring) {
    int64_t per = (int64_t)H * d;
    int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (idx >= n_tok * per) return;
    int64_t t = idx / per, e = idx % per;
    if (n_tok - t > window) return;  // only the last `window` tokens of this call can survive
    int64_t slot = (token0 + t) % window;
    ring[(0 * (int64_t)window + slot) * per + e] = k[idx];
    ring[(1 * (int64_t)window + slot) * per + e] = v[idx];
}
void launch_kv_ring(const void* k, const void* v, int64_t n_tok, int H, int d, int64_t token0, int window,
                    __nv_bfloat16* ring, cudaStream_t st) {
    if (window <= 0) return;
    int64_t t_first = n_tok > window ? n_tok - window : 0;
    int64_t cnt = (n_tok - t_first) * H * d;
    const __nv_bfloat16* kk = (const __nv_bfloat16*)k + t_first * H * d;
    const __nv_bfloat16* vv = (const __nv_bfloat16*)v + t_first * H * d;
    k_kv_ring<<<(unsigned)((cnt + 255) / 256), 256, 0, st>>>(kk, vv, n_tok - t_first, H, d, token0 + t_first, window,
                                                            ring);
}


// ---------------------------------------------------------------------------------------------
// One appended token, one launch (the decode-step case of hq_kv_append; a 1-token append is launch-latency
// bound).  One warp per (head, role) runs the whole chain B1-B7 with the same device functions as the bulk kernels
// (bit-identical container): RHT -> rotate -> normalize -> dither -> nearest point -> strip -> U length -> running
// offset of the head's U stream -> pack R and U -> bf16 ring.
// ---------------------------------------------------------------------------------------------
struct KvAppend1 {
    const __nv_bfloat16 *k, *v;    // [H][d] of the new token
    int H, d, rotation, dither, k0, k1, rbits, window;
    int64_t token, max_tokens, rem_words, una_words, n_blk;
    float A;
    uint64_t seed;
    const int8_t *dsign, *ssign;
    const float* qjl_t;            // HQ_ROT_QJL: S transposed
    uint32_t *rem, *una, *blk_off, *upos;
    uint16_t *ulen, *norm;
    __nv_bfloat16* ring;
    unsigned long long* counters;   // [0] clamps
    int* flag;                      // mapped host memory: error flag of the cache
    uint32_t* pos_dev;              // device_position caches: [0] token count (read as this token's index, advanced by the
                                    // last of the 2 H warps to finish), [1] their arrival counter; null: p.token is used
};

template <int LAT>
__global__ void __launch_bounds__(32)
k_kv_append1(KvAppend1 p) {
    extern __shared__ float smf[];   // u[d] | t[d] | codes[d] (int8) | z[d] (u8)
    const int lane = threadIdx.x, h = blockIdx.x, role = blockIdx.y, d = p.d, H = p.H;
    // every warp reads the position before its own arrival below; the last arrival writes the new one: no warp sees it early
    const int64_t token = p.pos_dev ? (int64_t)*(volatile const uint32_t*)p.pos_dev : p.token;
    auto arrive = [&]() {   // the warp's writes are done (or it wrote nothing)
        __syncwarp();
        if (p.pos_dev && lane == 0) {
            __threadfence();
            const unsigned prev = atomicAdd(p.pos_dev + 1, 1u);
            if (prev == 2u * (unsigned)H - 1u) {
                p.pos_dev[1] = 0u;
                if (token < p.max_tokens) *(volatile uint32_t*)p.pos_dev = (uint32_t)token + 1u;
            }
        }
    };
    if (token >= p.max_tokens) {   // a replayed graph ran past the capacity: nothing is written, the cache turns sticky
        if (lane == 0) kv_raise(p.flag, 3);
        arrive();
        return;
    }
    float* u = smf;
    float* t = u + d;
    int8_t* codes = (int8_t*)(t + d);
    uint8_t* z = (uint8_t*)(codes + d);
    const __nv_bfloat16* x = (role ? p.v : p.k) + (int64_t)h * d;
    for (int i = lane; i < d; i += 32) {
        const float xv = __bfloat162float(x[i]);
        u[i] = (p.dsign[i] < 0) ? -xv : xv;
        if (p.window > 0) p.ring[((int64_t)(role * p.window + (token % p.window)) * H + h) * d + i] = x[i];
    }
    warp_rht_inplace(u, d, lane);
    if (p.rotation == HQ_ROT_SIGNS)
        for (int i = lane; i < d; i += 32)
            if (p.ssign[i] < 0) u[i] = -u[i];
    if (p.rotation == HQ_ROT_QJL) {
        __syncwarp();
        warp_qjl_apply(u, d, p.qjl_t, lane);
    }
    for (int i = lane; i < d; i += 32) t[i] = __fmul_rn(u[i], u[i]);
    const float ss = warp_treesum(t, d, lane);
    const uint16_t hb = f32_to_f16_bits_sat(__fsqrt_rn(ss));
    const float rho = f16_bits_to_f32(hb);
    const int64_t rh = (int64_t)role * H + h;
    if (lane == 0) p.norm[rh * p.max_tokens + token] = hb;
    unsigned long long clamps = 0;
    if (rho == 0.0f) {
        for (int i = lane; i < d; i += 32) codes[i] = 0;
    } else {
        const float g = __fdiv_rn(p.A, rho);
        clamps = (unsigned long long)quantize_blocks<LAT>(u, d, g, p.dither != 0, p.seed, (uint32_t)token, (uint32_t)h,
                                                          (uint32_t)role, codes, lane, nullptr);
    }
    for (int o = 16; o; o >>= 1) clamps += __shfl_xor_sync(0xffffffffu, clamps, o);
    if (lane == 0 && clamps) atomicAdd(&p.counters[0], clamps);
    __syncwarp();
    // symbols in stream order, U length
    uint32_t L = 0;
    for (int b = lane; b < d / LAT; b += 32) {
        int c[LAT], zz[LAT];
#pragma unroll
        for (int i = 0; i < LAT; ++i) c[i] = codes[b * LAT + i];
        strip<LAT>(c, zz);
#pragma unroll
        for (int i = 0; i < LAT; ++i) {
            const int pos = (LAT == LAT_E8) ? 32 * (b >> 2) + 8 * (i >> 1) + 2 * (b & 3) + (i & 1) : b * LAT + i;
            z[pos] = (uint8_t)zz[i];
            L += 1u + ((uint32_t)zz[i] >> (sym_class(LAT, i) ? p.k1 : p.k0));
        }
    }
    for (int o = 16; o; o >>= 1) L += __shfl_xor_sync(0xffffffffu, L, o);
    __syncwarp();
    uint32_t ustart = 0;
    if (lane == 0) {
        ustart = p.upos[rh];
        if ((token & 127) == 0) p.blk_off[rh * (p.n_blk + 1) + (token >> 7)] = ustart;
        if (L >= 65535u) { kv_raise(p.flag, 1); L = 65535u; ustart = KV_NO_ROOM; }
        else if ((int64_t)ustart + L > p.una_words * 32 - 64) { kv_raise(p.flag, 2); ustart = KV_NO_ROOM; }
        else p.upos[rh] = ustart + L;
        p.ulen[rh * p.max_tokens + token] = (uint16_t)L;
    }
    // pack: lane 0 writes the R-section, lane 1 the U-section (serial bit writers; 2 x 128 symbols)
    ustart = __shfl_sync(0xffffffffu, ustart, 0);
    if (lane == 0) {
        BitWriter<StoreAtomicOr> bwr(StoreAtomicOr{p.rem + rh * p.rem_words}, (uint32_t)(token * p.rbits));
        write_R<LAT>(bwr, z, d, p.k0, p.k1);
    }
    if (ustart != KV_NO_ROOM) {   // a vector that does not fit is not written (flag raised)
        // the U-section by all 32 lanes: lane l writes the unary codes of symbols [l d/32, (l+1) d/32) at the bit offset its
        // predecessors' lengths add up to (an exclusive warp scan); words shared between lanes are merged by atomicOr
        const int spl = d >> 5;
        uint32_t mine = 0;
        for (int j = lane * spl; j < (lane + 1) * spl; ++j) mine += 1u + ((uint32_t)z[j] >> (sym_class(LAT, j) ? p.k1 : p.k0));
        uint32_t incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        BitWriter<StoreAtomicOr> bwu(StoreAtomicOr{p.una + rh * p.una_words}, ustart + (incl - mine));
        for (int j = lane * spl; j < (lane + 1) * spl; ++j) {
            bwu.skip((uint32_t)z[j] >> (sym_class(LAT, j) ? p.k1 : p.k0));
            bwu.put(1u, 1);
        }
        bwu.finish();
    }
    arrive();
}

void launch_kv_append1(const hq_kv* kv, const void* k, const void* v, cudaStream_t st) {
    KvAppend1 p;
    p.k = (const __nv_bfloat16*)k; p.v = (const __nv_bfloat16*)v;
    p.H = kv->cfg.kv_heads; p.d = kv->cfg.head_dim; p.rotation = kv->cfg.rotation; p.dither = kv->cfg.dither;
    p.k0 = kv->k0; p.k1 = kv->k1; p.rbits = kv->rbits; p.window = kv->cfg.window;
    p.token = kv->n_tokens; p.max_tokens = kv->cfg.max_tokens; p.rem_words = kv->rem_words; p.una_words = kv->una_words;
    p.n_blk = kv->n_blk; p.A = kv->A; p.seed = kv->cfg.codec.seed; p.dsign = kv->dsign; p.ssign = kv->ssign;
    p.qjl_t = kv->qjl ? kv->qjl + (size_t)p.d * p.d : nullptr;
    p.rem = kv->rem; p.una = kv->una; p.blk_off = kv->blk_off; p.upos = kv->upos; p.ulen = kv->ulen; p.norm = kv->norm;
    p.ring = kv->ring; p.counters = kv->counters; p.flag = kv->flag_dev; p.pos_dev = kv->pos_dev;
    const size_t smem = (size_t)p.d * (4 + 4 + 1 + 1);
    dim3 grid((unsigned)p.H, 2);
    switch (kv->cfg.codec.lattice) {
        case LAT_Z: k_kv_append1<LAT_Z><<<grid, 32, smem, st>>>(p); break;
        case LAT_A2: k_kv_append1<LAT_A2><<<grid, 32, smem, st>>>(p); break;
        case LAT_D4: k_kv_append1<LAT_D4><<<grid, 32, smem, st>>>(p); break;
        default: k_kv_append1<LAT_E8><<<grid, 32, smem, st>>>(p); break;
    }
}

}  // namespace hq
