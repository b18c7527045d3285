// hq_linear.cu — half 1 of the hot path: per weight group (128 rows x one
// RHT tile) fetch the Rice stream (A3), decode unary + remainders (A4, §3.3), un-zig-zag and
// un-strip to INT8 lattice points (A5, §4.6), stage them in shared memory in the UMMA
// K-major SWIZZLE_128B layout and contract with the INT8 activations on the tensor core
// (A6, tcgen05.mma kind::i8 -> INT32 in TMEM, §4.8), then rescale per K-tile and accumulate (A7,
// §4.3).  Decoded weights never leave shared memory.
#include "hq_common.cuh"
#include "hq_e8_fast.cuh"
#include "hq_internal.h"
#include "hq_tc.cuh"

namespace hq {

// ---------------------------------------------------------------------------------------------
// Group view + row start offsets.
// ---------------------------------------------------------------------------------------------
struct GroupView {
    const uint16_t* ulen;
    const uint16_t* norm;
    const uint32_t* rarea;
    const uint32_t* uarea;
};
__device__ inline GroupView group_view(const uint8_t* base, int rbits) {
    uint32_t r16 = (uint32_t)((128 * rbits + 127) / 128);
    GroupView v;
    v.ulen = (const uint16_t*)base;
    v.norm = v.ulen + 128;
    v.rarea = (const uint32_t*)(base + 512);
    v.uarea = (const uint32_t*)(base + 512 + 16 * (size_t)r16);
    return v;
}

// ---------------------------------------------------------------------------------------------
// hq_decode_int8: block per group, thread per row, straight from global memory (parity tool).
// ---------------------------------------------------------------------------------------------
template <int LAT>
__global__ void __launch_bounds__(128)
k_decode_int8(const uint8_t* blob, const uint32_t* group_off, int64_t m, int64_t n_kt, int n, int k0, int k1,
              int8_t* codes, uint16_t* norms) {
    __shared__ uint32_t scan[4];
    int64_t g = blockIdx.x;
    int i = threadIdx.x;
    int64_t rb = g / n_kt, kt = g % n_kt, r = rb * 128 + i;
    int rbits = rbits_of(LAT, n, k0, k1);
    GroupView gv = group_view(blob + 16 * (size_t)group_off[g], rbits);
    uint32_t ul = gv.ulen[i];
    uint32_t ustart = row_ustart_128(ul, scan, i);
    if (r >= m) return;
    if (norms) norms[r * n_kt + kt] = gv.norm[i];
    int8_t* out = codes + r * (n_kt * n) + kt * n;
    decode_row_generic<LAT>(gv.rarea, (uint32_t)(i * rbits), gv.uarea, ustart, n, k0, k1,
                            [&](int b, const int* c) {
#pragma unroll
                                for (int e = 0; e < LAT; ++e) out[b * LAT + e] = (int8_t)c[e];
                            });
}

void launch_decode_int8(const hq_weight* w, int8_t* codes, uint16_t* norms, cudaStream_t st) {
#define HQ_D(L) \
    k_decode_int8<L><<<(unsigned)w->G, 128, 0, st>>>(w->blob, w->group_off, w->m, w->n_kt, w->n, w->k0, w->k1, codes, norms)
    switch (w->lattice) {
        case LAT_Z: HQ_D(LAT_Z); break;
        case LAT_A2: HQ_D(LAT_A2); break;
        case LAT_D4: HQ_D(LAT_D4); break;
        default: HQ_D(LAT_E8); break;
    }
#undef HQ_D
}

// ---------------------------------------------------------------------------------------------
// Fused decode + INT8 MMA, generic version (any lattice / tile / k):
// CTA = 128 threads = the 128 rows of a row block; loops over a range of K-tiles.
//   per K-tile: stage the group blob in smem -> each thread decodes its row into the A operand tile
//   -> B operand tile (activations) -> fence -> one thread issues n/32 tcgen05.mma -> commit ->
//   everybody reads its accumulator row from TMEM, rescales and accumulates in fp32 registers.
// NB = columns of the MMA (batch rows handled per pass, multiple of 16).
// ---------------------------------------------------------------------------------------------
struct LinearParams {
    const uint8_t* blob;
    const uint32_t* group_off;
    int64_t m, n_kt;
    int n, k0, k1, rbits;
    float inv_A;
    const int8_t* q;    // [B, n_in]
    const float* s_x;   // [B, n_kt]
    int64_t B;
    int n_split;        // K split
    float* partials;    // [n_split, B, m]
    int32_t* acc_i32;   // [n_kt, B, m] or null
    uint32_t stage_bytes;
};

template <int LAT, int NB>
__global__ void __launch_bounds__(128)
k_linear_generic(LinearParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    // carve: A tile | B tile | stage | small
    const int n = p.n;
    const int n_atoms = (n + 127) / 128;
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sA = smem;
    uint8_t* sB = sA + n_atoms * 128 * 128;
    uint8_t* stage = sB + n_atoms * NB * 128;
    float* s_sx = (float*)(stage + p.stage_bytes);  // [NB]
    uint32_t* scan = (uint32_t*)(s_sx + NB);        // [4]
    uint64_t* bar = (uint64_t*)(scan + 4);
    uint32_t* tmem_slot = (uint32_t*)(bar + 1);

    const int tid = threadIdx.x, warp = tid >> 5;
    const int64_t n_bt = (p.B + NB - 1) / NB;
    int64_t item = blockIdx.x;
    const int split = (int)(item % p.n_split); item /= p.n_split;
    const int64_t bt = item % n_bt;
    const int64_t rb = item / n_bt;
    const int64_t kt_per = (p.n_kt + p.n_split - 1) / p.n_split;
    const int64_t kt0 = split * kt_per, kt1 = min(p.n_kt, kt0 + kt_per);
    const int64_t b0 = bt * NB;
    const int64_t r = rb * 128 + tid;

    constexpr uint32_t TCOLS = NB < 32 ? 32 : NB;
    if (warp == 0) tmem_alloc(tmem_slot, TCOLS);
    if (tid == 0) { mbar_init(bar, 1); mbar_fence_init(); }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const uint32_t idesc = make_idesc_i8(128, NB);
    uint32_t phase = 0;

    float yacc[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) yacc[b] = 0.0f;

    for (int64_t kt = kt0; kt < kt1; ++kt) {
        const int64_t g = rb * p.n_kt + kt;
        const uint8_t* gsrc = p.blob + 16 * (size_t)p.group_off[g];
        const uint32_t gbytes = 16u * (p.group_off[g + 1] - p.group_off[g]);
        const bool staged = gbytes <= p.stage_bytes;
        if (staged) {
            const uint4* s4 = (const uint4*)gsrc;
            uint4* d4 = (uint4*)stage;
            for (uint32_t v = tid; v < gbytes / 16; v += 128) d4[v] = __ldg(s4 + v);
        }
        // B operand: NB rows x n K-bytes, 16-byte chunks
        {
            const int chunks_per_row = n / 16;
            for (int v = tid; v < NB * chunks_per_row; v += 128) {
                int bb = v / chunks_per_row, c16 = v % chunks_per_row;
                uint4 val = make_uint4(0, 0, 0, 0);
                if (b0 + bb < p.B) val = __ldg((const uint4*)(p.q + (b0 + bb) * (p.n_kt * n) + kt * n + c16 * 16));
                *(uint4*)(sB + sw128_offset(NB, bb, c16 * 16)) = val;
            }
            if (tid < NB) s_sx[tid] = (b0 + tid < p.B) ? p.s_x[(b0 + tid) * p.n_kt + kt] : 0.0f;
        }
        __syncthreads();
        GroupView gv = group_view(staged ? stage : gsrc, p.rbits);
        const uint32_t ul = gv.ulen[tid];
        const float rho = f16_bits_to_f32(gv.norm[tid]);
        const uint32_t ustart = row_ustart_128(ul, scan, tid);
        if (r < p.m) {
            decode_row_generic<LAT>(gv.rarea, (uint32_t)(tid * p.rbits), gv.uarea, ustart, n, p.k0, p.k1,
                                    [&](int b, const int* c) {
#pragma unroll
                                        for (int e = 0; e < LAT; ++e)
                                            sA[sw128_offset(128, tid, b * LAT + e)] = (uint8_t)(int8_t)c[e];
                                    });
        } else {
            for (int j = 0; j < n; j += 16) *(uint4*)(sA + sw128_offset(128, tid, j)) = make_uint4(0, 0, 0, 0);
        }
        fence_proxy_async_smem();
        __syncthreads();
        if (tid == 0) {
            tc_fence_after();
            const uint32_t a0 = smem_u32(sA), bb0 = smem_u32(sB);
            for (int ks = 0; ks < n / 32; ++ks) {
                uint32_t aoff = (uint32_t)((ks >> 2) * 128 * 128 + (ks & 3) * 32);
                uint32_t boff = (uint32_t)((ks >> 2) * NB * 128 + (ks & 3) * 32);
                mma_i8(tmem_base, make_desc_sw128(a0 + aoff), make_desc_sw128(bb0 + boff), idesc, ks > 0);
            }
            mma_commit(bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
        tc_fence_after();
        const float sw = rho * p.inv_A;
#pragma unroll
        for (int c0 = 0; c0 < NB; c0 += 16) {
            uint32_t v[16];
            tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + c0, v);
            tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                int a = (int)v[e];
                if (p.acc_i32 && r < p.m && b0 + c0 + e < p.B) p.acc_i32[(kt * p.B + b0 + c0 + e) * p.m + r] = a;
                yacc[c0 + e] += (sw * s_sx[c0 + e]) * (float)a;
            }
        }
        tc_fence_before();
        __syncthreads();
    }
    if (r < p.m) {
#pragma unroll
        for (int b = 0; b < NB; ++b)
            if (b0 + b < p.B) p.partials[((int64_t)split * p.B + b0 + b) * p.m + r] = yacc[b];
    }
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem_base, TCOLS);
}

// ---------------------------------------------------------------------------------------------
// Fused decode + INT8 MMA, E8 fast path (north_star (a)-(d)):
//   * group blobs arrive by TMA 1-D bulk copies (cp.async.bulk + mbarrier), NSTG groups in flight per CTA;
//   * each thread decodes its row with the LUT/SWAR decoder of hq_e8_fast.cuh straight into the
//     SWIZZLE_128B K-major A operand tile (decoded weights never leave shared memory);
//   * one thread issues the tcgen05.mma kind::i8 chain for the K-tile; accumulators sit in TMEM;
//   * every thread drains its accumulator row (tcgen05.ld), rescales by rho/(alpha sqrt n) * s_x (A7).
// Several CTAs per SM hide the decode's shared-memory latencies.
// ---------------------------------------------------------------------------------------------
constexpr int LIN_NSTG = 2;

template <int K, int NB>
__global__ void __launch_bounds__(128, 3)
k_linear_e8(LinearParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const int n = p.n;
    const int n_atoms = (n + 127) / 128;
    const int nblk = n / 8;
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sA = smem;
    uint8_t* sB = sA + n_atoms * 128 * 128;
    uint8_t* stage0 = sB + n_atoms * NB * 128;
    uint32_t* scr_all = (uint32_t*)(stage0 + LIN_NSTG * p.stage_bytes);  // [128][nblk + 1]
    uint32_t* lut = scr_all + 128 * (nblk + 1);                            // [512]
    float* s_sx = (float*)(lut + 512);                                     // [NB]
    uint32_t* scan = (uint32_t*)(s_sx + NB);                               // [4]
    uint64_t* bar_full = (uint64_t*)(scan + 4);                            // [LIN_NSTG]
    uint64_t* bar_mma = bar_full + LIN_NSTG;
    uint32_t* tmem_slot = (uint32_t*)(bar_mma + 1);

    const int tid = threadIdx.x, warp = tid >> 5;
    const int64_t n_bt = (p.B + NB - 1) / NB;
    int64_t item = blockIdx.x;
    const int split = (int)(item % p.n_split); item /= p.n_split;
    const int64_t bt = item % n_bt;
    const int64_t rb = item / n_bt;
    const int64_t kt_per = (p.n_kt + p.n_split - 1) / p.n_split;
    const int64_t kt0 = split * kt_per, kt1 = min(p.n_kt, kt0 + kt_per);
    const int64_t b0 = bt * NB;
    const int64_t r = rb * 128 + tid;

    constexpr uint32_t TCOLS = NB < 32 ? 32 : NB;
    if (warp == 0) tmem_alloc(tmem_slot, TCOLS);
    if (tid == 0) {
        for (int s = 0; s < LIN_NSTG; ++s) mbar_init(&bar_full[s], 1);
        mbar_init(bar_mma, 1);
        mbar_fence_init();
    }
    build_unary_lut(lut, tid, 128);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const uint32_t idesc = make_idesc_i8(128, NB);
    uint32_t mma_phase = 0;

    auto group_bytes = [&](int64_t kt) -> uint32_t {
        const int64_t g = rb * p.n_kt + kt;
        return 16u * (p.group_off[g + 1] - p.group_off[g]);
    };
    auto prefetch = [&](int64_t kt) {  // thread 0 only
        if (kt >= kt1) return;
        const uint32_t gb = group_bytes(kt);
        if (gb > p.stage_bytes) return;  // oversized group: decoded from global memory
        const int s = (int)((kt - kt0) % LIN_NSTG);
        const int64_t g = rb * p.n_kt + kt;
        mbar_arrive_expect_tx(&bar_full[s], gb);
        bulk_g2s(stage0 + (size_t)s * p.stage_bytes, p.blob + 16 * (size_t)p.group_off[g], gb, &bar_full[s]);
    };
    if (tid == 0)
        for (int s = 0; s < LIN_NSTG; ++s) prefetch(kt0 + s);

    float yacc[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) yacc[b] = 0.0f;
    uint32_t* scr = scr_all + tid * (nblk + 1);
    const uint32_t a_row = (uint32_t)((tid >> 3) * 1024 + (tid & 7) * 128);

    for (int64_t kt = kt0; kt < kt1; ++kt) {
        const int s = (int)((kt - kt0) % LIN_NSTG);
        const uint32_t full_parity = (uint32_t)(((kt - kt0) / LIN_NSTG) & 1);
        const int64_t g = rb * p.n_kt + kt;
        const uint32_t gbytes = group_bytes(kt);
        const bool staged = gbytes <= p.stage_bytes;
        // B operand (activations), permuted inside each 8-byte group to (0,2,4,6,1,3,5,7)
        {
            const int chunks_per_row = n / 16;
            for (int v = tid; v < NB * chunks_per_row; v += 128) {
                int bb = v / chunks_per_row, c16 = v % chunks_per_row;
                uint4 val = make_uint4(0, 0, 0, 0);
                if (b0 + bb < p.B) val = __ldg((const uint4*)(p.q + (b0 + bb) * (p.n_kt * n) + kt * n + c16 * 16));
                uint4 pv;
                pv.x = __byte_perm(val.x, val.y, 0x6420); pv.y = __byte_perm(val.x, val.y, 0x7531);
                pv.z = __byte_perm(val.z, val.w, 0x6420); pv.w = __byte_perm(val.z, val.w, 0x7531);
                *(uint4*)(sB + sw128_offset(NB, bb, c16 * 16)) = pv;
            }
            if (tid < NB) s_sx[tid] = (b0 + tid < p.B) ? p.s_x[(b0 + tid) * p.n_kt + kt] : 0.0f;
        }
        if (staged) mbar_wait(&bar_full[s], full_parity);
        GroupView gv = group_view(staged ? stage0 + (size_t)s * p.stage_bytes : p.blob + 16 * (size_t)p.group_off[g], p.rbits);
        const uint32_t ul = gv.ulen[tid];
        const float rho = f16_bits_to_f32(gv.norm[tid]);
        const uint32_t ustart = row_ustart_128(ul, scan, tid);
        auto store_block = [&](int b, uint32_t ce, uint32_t co) {
            uint32_t off = (uint32_t)((b >> 4) * 16384) + a_row + (uint32_t)(((((b & 15) >> 1) ^ (tid & 7)) << 4) + (b & 1) * 8);
            *(uint2*)(sA + off) = make_uint2(ce, co);
        };
        bool ok = false;
        if (r < p.m && ul > 0) {
            if (staged) ok = e8_decode_row_fast<K>(gv.uarea, ustart, ul, gv.rarea + tid * (p.rbits >> 5), lut, scr, n, store_block);
            if (!ok) {  // a quotient >= 16 somewhere in the row, or an oversized group: generic decoder
                decode_row_generic<LAT_E8>(gv.rarea, (uint32_t)(tid * p.rbits), gv.uarea, ustart, n, p.k0, p.k1,
                                           [&](int b, const int* c) {
                                               uint32_t ce = (uint32_t)(uint8_t)c[0] | ((uint32_t)(uint8_t)c[2] << 8) |
                                                             ((uint32_t)(uint8_t)c[4] << 16) | ((uint32_t)(uint8_t)c[6] << 24);
                                               uint32_t co = (uint32_t)(uint8_t)c[1] | ((uint32_t)(uint8_t)c[3] << 8) |
                                                             ((uint32_t)(uint8_t)c[5] << 16) | ((uint32_t)(uint8_t)c[7] << 24);
                                               store_block(b, ce, co);
                                           });
            }
        } else {
            for (int b = 0; b < nblk; ++b) store_block(b, 0u, 0u);
        }
        fence_proxy_async_smem();
        __syncthreads();
        if (tid == 0) {
            prefetch(kt + LIN_NSTG);  // stage s is free again
            tc_fence_after();
            const uint32_t a0 = smem_u32(sA), bb0 = smem_u32(sB);
            for (int ks = 0; ks < n / 32; ++ks) {
                uint32_t aoff = (uint32_t)((ks >> 2) * 128 * 128 + (ks & 3) * 32);
                uint32_t boff = (uint32_t)((ks >> 2) * NB * 128 + (ks & 3) * 32);
                mma_i8(tmem_base, make_desc_sw128(a0 + aoff), make_desc_sw128(bb0 + boff), idesc, ks > 0);
            }
            mma_commit(bar_mma);
        }
        mbar_wait(bar_mma, mma_phase);
        mma_phase ^= 1;
        tc_fence_after();
        const float sw = rho * p.inv_A;
#pragma unroll
        for (int c0 = 0; c0 < NB; c0 += 16) {
            uint32_t v[16];
            tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + c0, v);
            tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                int a = (int)v[e];
                if (p.acc_i32 && r < p.m && b0 + c0 + e < p.B) p.acc_i32[(kt * p.B + b0 + c0 + e) * p.m + r] = a;
                yacc[c0 + e] += (sw * s_sx[c0 + e]) * (float)a;
            }
        }
        tc_fence_before();
        __syncthreads();
    }
    if (r < p.m) {
#pragma unroll
        for (int b = 0; b < NB; ++b)
            if (b0 + b < p.B) p.partials[((int64_t)split * p.B + b0 + b) * p.m + r] = yacc[b];
    }
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem_base, TCOLS);
}

// y[b, r] = sum over splits (in order) -> fp32 and bf16
__global__ void k_linear_finalize(const float* partials, int n_split, int64_t B, int64_t m, __nv_bfloat16* y,
                                  int64_t ldy, float* y_f32) {
    int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (idx >= B * m) return;
    float s = 0.0f;
    for (int sp = 0; sp < n_split; ++sp) s += partials[(int64_t)sp * B * m + idx];
    int64_t b = idx / m, r = idx % m;
    if (y) y[b * ldy + r] = __float2bfloat16_rn(s);
    if (y_f32) y_f32[idx] = s;
}

static uint32_t stage_bytes_for(const hq_weight* w) {
    // header + R area + room for ~3 unary bits per symbol; larger groups are read from global memory
    uint32_t r16 = (uint32_t)((128 * (int64_t)w->rbits + 127) / 128);
    uint32_t cap = 512 + 16 * r16 + 128 * (uint32_t)(w->n * 3 / 8) + 256;
    return (cap + 127) & ~127u;
}

int linear_choose_split(const hq_ctx* ctx, const hq_weight* w, int64_t B) {
    int NB = B <= 16 ? 16 : 64;
    int64_t n_bt = (B + NB - 1) / NB;
    int64_t items = w->n_rb * n_bt;
    int target = ctx->sm_count * 4;
    int split = 1;
    while (items * split < target && split * 2 <= w->n_kt) split *= 2;
    return split;
}

template <int NB>
static hq_status launch_linear_nb(hq_ctx* ctx, const hq_weight* w, LinearParams& p, cudaStream_t st) {
    int n_atoms = (w->n + 127) / 128;
    int64_t n_bt = (p.B + NB - 1) / NB;
    int64_t grid = w->n_rb * n_bt * p.n_split;
    if (w->lattice == LAT_E8) {
        size_t smem = 1024 + (size_t)n_atoms * 128 * 128 + (size_t)n_atoms * NB * 128 + (size_t)LIN_NSTG * p.stage_bytes +
                      128 * (size_t)(w->n / 8 + 1) * 4 + 2048 + NB * 4 + 16 + 8 * (LIN_NSTG + 1) + 16;
#define HQ_LE(KK)                                                                                                   \
    case KK:                                                                                                        \
        HQ_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_linear_e8<KK, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        k_linear_e8<KK, NB><<<(unsigned)grid, 128, smem, st>>>(p);                                                  \
        break
        switch (w->k0) {
            HQ_LE(0); HQ_LE(1); HQ_LE(2); HQ_LE(3); HQ_LE(4); HQ_LE(5); HQ_LE(6); HQ_LE(7);
        }
#undef HQ_LE
        HQ_CUDA_CHECK(ctx, cudaGetLastError());
        return HQ_OK;
    }
    size_t smem = 1024 + (size_t)n_atoms * 128 * 128 + (size_t)n_atoms * NB * 128 + p.stage_bytes + NB * 4 + 16 + 8 + 8;
#define HQ_L(L)                                                                                                   \
    do {                                                                                                          \
        HQ_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_linear_generic<L, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        k_linear_generic<L, NB><<<(unsigned)grid, 128, smem, st>>>(p);                                            \
    } while (0)
    switch (w->lattice) {
        case LAT_Z: HQ_L(LAT_Z); break;
        case LAT_A2: HQ_L(LAT_A2); break;
        case LAT_D4: HQ_L(LAT_D4); break;
        default: HQ_L(LAT_E8); break;
    }
#undef HQ_L
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    return HQ_OK;
}

hq_status launch_linear(hq_ctx* ctx, const hq_weight* w, const int8_t* q, const float* s_x, int64_t B,
                        void* y_bf16, int64_t ldy, float* y_f32, int32_t* acc_i32, float* partials, int n_split,
                        cudaStream_t st) {
    LinearParams p;
    p.blob = w->blob; p.group_off = w->group_off; p.m = w->m; p.n_kt = w->n_kt;
    p.n = w->n; p.k0 = w->k0; p.k1 = w->k1; p.rbits = w->rbits;
    p.inv_A = (float)(1.0 / (w->alpha * sqrt((double)w->n)));
    p.q = q; p.s_x = s_x; p.B = B; p.n_split = n_split; p.partials = partials; p.acc_i32 = acc_i32;
    p.stage_bytes = stage_bytes_for(w);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (ctx->prof) {
        HQ_CUDA_CHECK(ctx, cudaEventCreate(&e0));
        HQ_CUDA_CHECK(ctx, cudaEventCreate(&e1));
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e0, st));
    }
    hq_status s = (B <= 16) ? launch_linear_nb<16>(ctx, w, p, st) : launch_linear_nb<64>(ctx, w, p, st);
    if (s != HQ_OK) return s;
    if (ctx->prof) {
        HQ_CUDA_CHECK(ctx, cudaEventRecord(e1, st));
        ctx->prof_ev.push_back(e0);
        ctx->prof_ev.push_back(e1);
    }
    int64_t tot = B * w->m;
    k_linear_finalize<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(partials, n_split, B, w->m, (__nv_bfloat16*)y_bf16,
                                                                    ldy, y_f32);
    HQ_CUDA_CHECK(ctx, cudaGetLastError());
    return HQ_OK;
}

}  // namespace hq
