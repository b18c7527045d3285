// hq_e8_ceiling.cuh — measurement kernel: the issue-slot ceiling of the E8 Rice decode ("measure the
// issue-slot ceiling first: decode-only kernel, no loads, and report %HBM and %issue together"; PAPER.md:L355 names the
// serial unary scan as the central obstacle).
//
// Same CTA shape as the fused kernel (NWG warp groups of 128 threads, lane = weight row, one CTA per SM, the phase-1
// table and the nibble scratch in shared memory), same phase 1 + phase 2 code (hq_e8_decode.cuh), same 128-bit stores
// into a SWIZZLE_128B A tile.  What is left out: global loads inside the loop (every warp keeps ONE sub-group of the
// tensor in registers and decodes it `reps` times), the MMA, the accumulator drain, split-K, barriers.  So the rate it
// reaches is what the decode arithmetic alone allows on this SM: an upper bound for any kernel built on this decoder.
#pragma once
#include "hq_common.cuh"
#include "hq_e8_decode.cuh"
#include "hq_linear_e8.cuh"
#include "hq_tc.cuh"

namespace hq {

struct E8CeilParams {
    const uint8_t* blob;
    const uint32_t* sub_off;
    const uint32_t* lut;
    int64_t n_groups;     // sub-groups of the tensor (4 G)
    int reps;
    unsigned int* sink;   // one word per thread: keeps the decode alive
};

template <int K, int NWG>
__global__ void __launch_bounds__(NWG * 128, 1) k_e8_decode_ceiling(E8CeilParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    constexpr int KW = 4 * K;
    const int tid = threadIdx.x, wg = tid >> 7, t = tid & 127, warp = t >> 5, lane = t & 31;
    uint32_t* lut_s = (uint32_t*)smem;
    for (int i = tid; i < E8_LUT_WORDS; i += NWG * 128) lut_s[i] = __ldg(p.lut + i);
    __syncthreads();
    const uint32_t smem_a = smem_u32(smem);
    const uint32_t wg_a = smem_a + E8_LUT_BYTES + (uint32_t)wg * (16384u + 128u * E8_SCR_STRIDE * 4u);
    const uint32_t sA_a = wg_a + (uint32_t)((t >> 3) * 1024 + (t & 7) * 128);
    const uint32_t scr_a = wg_a + 16384u + (uint32_t)t * E8_SCR_STRIDE * 4;
    const uint32_t lut_lane = smem_a + (uint32_t)(lane & (E8_LUT_COPIES - 1)) * 4;
    const uint32_t lane_lt = (1u << lane) - 1u;
    // one full sub-group per warp (any: they are statistically alike), loaded once
    const int64_t sg = ((int64_t)blockIdx.x * (NWG * 4) + wg * 4 + warp) % p.n_groups;
    const uint8_t* sgp = p.blob + 16 * (size_t)__ldg(p.sub_off + sg);
    const uint32_t ul = __ldg((const uint16_t*)sgp + lane);
    const uint32_t* rarea = (const uint32_t*)(sgp + 128);
    const uint32_t* uarea = rarea + KW * 32;
    uint32_t Rw[KW > 0 ? KW : 1], Uw[E8_NW];
#pragma unroll
    for (int j = 0; j < KW; ++j) Rw[j] = __ldg(rarea + j * 32 + lane);
    const uint32_t nw = (ul + 31) >> 5;
    {
        uint32_t base = 0;
#pragma unroll
        for (int w = 0; w < E8_NW; ++w) {
            const bool has = nw > (uint32_t)w;
            const uint32_t mk = __ballot_sync(0xffffffffu, has);
            Uw[w] = has ? __ldg(uarea + base + __popc(mk & lane_lt)) : 0u;
            base += __popc(mk);
        }
    }
    const uint32_t maxul = __reduce_max_sync(0xffffffffu, ul);
    const uint32_t maxnw = (maxul + 31) >> 5;
    uint32_t sink = 0;
    for (int rep = 0; rep < p.reps; ++rep) {
        // the compiler must not hoist the decode of loop-invariant inputs: make them opaque every iteration
#pragma unroll
        for (int w = 0; w < E8_NW; ++w) asm volatile("" : "+r"(Uw[w]));
#pragma unroll
        for (int j = 0; j < KW; ++j) asm volatile("" : "+r"(Rw[j]));
        {
            uint32_t T = 0, acc = 0, wo = scr_a;
#pragma unroll
            for (int w = 0; w < E8_NW; ++w) {
                if (w < E8_DENSE) {
                    e8_unary_word(Uw[w], lut_lane, T, acc, wo);
                } else if ((uint32_t)w < maxnw) {
                    const int nb = (int)min(4u, (maxul - 32u * (uint32_t)w + 7u) >> 3);
                    e8_unary_word(Uw[w], lut_lane, T, acc, wo, nb);
                }
            }
        }
        uint32_t total = 0, prevWo = 15u << 24;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            uint32_t W[4], C[8];
#pragma unroll
            for (int w = 0; w < 4; ++w) W[w] = lds32(scr_a + (c * 4 + w) * 4);
            e8_run<K>(W, Rw + c * K, prevWo, total, C);
            const uint32_t u0 = (uint32_t)(((2 * c) ^ (t & 7)) << 4), u1 = (uint32_t)(((2 * c + 1) ^ (t & 7)) << 4);
            sts128(sA_a + u0, C[0], C[1], C[2], C[3]);
            sts128(sA_a + u1, C[4], C[5], C[6], C[7]);
        }
        sink += total;
    }
    p.sink[(size_t)blockIdx.x * (NWG * 128) + tid] = sink + lds32(sA_a);
}

}  // namespace hq
