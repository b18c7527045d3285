// hq_act.cuh — one activation tile of 128 through the RHT and the INT8 cast, by one warp, in registers
// (FORMAT R1, R7; §3.1 eq.(1), §4.8).  Shared by k_act_blob (hq_encode.cu) and the
// batch-1 fused kernel (hq_gemv_e8.cuh), which quantizes x itself instead of reading operand tiles from global memory.
//
// Lane l holds elements 4l .. 4l+3.  FORMAT R1's butterflies (ascending stride, a+b to the lower index, a-b to the upper)
// are two in-register stages and five shuffle stages: the same additions on the same pairs as the shared-memory
// butterfly of k_act_quant, so the result is bit-identical.  Every operation is an explicit round-to-nearest intrinsic
// (no contraction whatever the translation unit's -fmad setting).
#pragma once
#include <cuda_bf16.h>
#include <stdint.h>

namespace hq {

// x[4]: the lane's four elements already multiplied by the RHT signs.  On return q[4] = INT8 codes (as int), and the
// function's value is the tile scale s_x = amax / 127 (0 for an all-zero tile).  All 32 lanes must call it.
__device__ __forceinline__ float warp_act_tile128(float* x, int lane, int* q) {
    {   // strides 1 and 2: inside the lane
        float a = x[0], c = x[1];
        x[0] = __fadd_rn(a, c); x[1] = __fsub_rn(a, c);
        a = x[2]; c = x[3];
        x[2] = __fadd_rn(a, c); x[3] = __fsub_rn(a, c);
        a = x[0]; c = x[2];
        x[0] = __fadd_rn(a, c); x[2] = __fsub_rn(a, c);
        a = x[1]; c = x[3];
        x[1] = __fadd_rn(a, c); x[3] = __fsub_rn(a, c);
    }
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) {   // strides 4 .. 64: lane ^ m holds the partner
        const float sg1 = (lane & m) ? -1.0f : 1.0f;   // upper index of the pair: a - b = o - x, else x + o
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float o = __shfl_xor_sync(0xffffffffu, x[j], m);
            x[j] = __fmaf_rn(x[j], sg1, o);            // the product is exact: one rounding, that of the sum
        }
    }
    const float cn = (float)(1.0 / sqrt(128.0));   // FORMAT R1 (folded at compile time)
    float amax = 0.0f;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        x[j] = __fmul_rn(x[j], cn);
        amax = fmaxf(amax, fabsf(x[j]));
    }
#pragma unroll
    for (int sft = 16; sft; sft >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, sft));
    const float inv = (amax == 0.0f) ? 0.0f : __fdiv_rn(127.0f, amax);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        int qv = 0;
        if (amax != 0.0f) {
            float v = rintf(__fmul_rn(x[j], inv));
            v = fminf(fmaxf(v, -127.0f), 127.0f);
            qv = (int)v;
        }
        q[j] = qv;
    }
    return (amax == 0.0f) ? 0.0f : __fdiv_rn(amax, 127.0f);
}

// The FP8-E4M3 cast of the same tile (FORMAT R12; §4.8): identical RHT, then q8 = e4m3(u * 448 / amax) as
// bytes (in q[], low 8 bits) and s_x = amax / 448.
__device__ __forceinline__ float warp_act_tile128_fp8(float* x, int lane, int* q) {
    {
        float a = x[0], c = x[1];
        x[0] = __fadd_rn(a, c); x[1] = __fsub_rn(a, c);
        a = x[2]; c = x[3];
        x[2] = __fadd_rn(a, c); x[3] = __fsub_rn(a, c);
        a = x[0]; c = x[2];
        x[0] = __fadd_rn(a, c); x[2] = __fsub_rn(a, c);
        a = x[1]; c = x[3];
        x[1] = __fadd_rn(a, c); x[3] = __fsub_rn(a, c);
    }
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) {
        const float sg1 = (lane & m) ? -1.0f : 1.0f;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float o = __shfl_xor_sync(0xffffffffu, x[j], m);
            x[j] = __fmaf_rn(x[j], sg1, o);
        }
    }
    const float cn = (float)(1.0 / sqrt(128.0));
    float amax = 0.0f;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        x[j] = __fmul_rn(x[j], cn);
        amax = fmaxf(amax, fabsf(x[j]));
    }
#pragma unroll
    for (int sft = 16; sft; sft >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, sft));
    if (amax == 0.0f) {
#pragma unroll
        for (int j = 0; j < 4; ++j) q[j] = 0;
        return 0.0f;
    }
    const float inv = __fdiv_rn(448.0f, amax);
#pragma unroll
    for (int j = 0; j < 4; j += 2) {
        uint16_t r;
        asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(__fmul_rn(x[j + 1], inv)), "f"(__fmul_rn(x[j], inv)));
        q[j] = (int)(r & 0xffu);
        q[j + 1] = (int)(r >> 8);
    }
    return __fdiv_rn(amax, 448.0f);
}

// NT tiles at once, stage by stage (the tiles are independent: their shuffles and roundings interleave, so the latency
// is that of one tile); per tile the same operations in the same order as warp_act_tile128: bit-identical.
// x[i][4], q[i][4], sx[i] for tile i; tiles with on[i] == false (warp-uniform) are skipped.
template <int NT>
__device__ __forceinline__ void warp_act_tiles128(float (*x)[4], const bool* on, int lane, int (*q)[4], float* sx) {
#pragma unroll
    for (int i = 0; i < NT; ++i) {
        float a = x[i][0], c = x[i][1];
        x[i][0] = __fadd_rn(a, c); x[i][1] = __fsub_rn(a, c);
        a = x[i][2]; c = x[i][3];
        x[i][2] = __fadd_rn(a, c); x[i][3] = __fsub_rn(a, c);
        a = x[i][0]; c = x[i][2];
        x[i][0] = __fadd_rn(a, c); x[i][2] = __fsub_rn(a, c);
        a = x[i][1]; c = x[i][3];
        x[i][1] = __fadd_rn(a, c); x[i][3] = __fsub_rn(a, c);
    }
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) {
        const float sg1 = (lane & m) ? -1.0f : 1.0f;
#pragma unroll
        for (int i = 0; i < NT; ++i) {
            if (!on[i]) continue;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float o = __shfl_xor_sync(0xffffffffu, x[i][j], m);
                x[i][j] = __fmaf_rn(x[i][j], sg1, o);
            }
        }
    }
    const float cn = (float)(1.0 / sqrt(128.0));
    float amax[NT];
#pragma unroll
    for (int i = 0; i < NT; ++i) {
        amax[i] = 0.0f;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            x[i][j] = __fmul_rn(x[i][j], cn);
            amax[i] = fmaxf(amax[i], fabsf(x[i][j]));
        }
    }
#pragma unroll
    for (int sft = 16; sft; sft >>= 1)
#pragma unroll
        for (int i = 0; i < NT; ++i)
            if (on[i]) amax[i] = fmaxf(amax[i], __shfl_xor_sync(0xffffffffu, amax[i], sft));
#pragma unroll
    for (int i = 0; i < NT; ++i) {
        const float inv = (amax[i] == 0.0f) ? 0.0f : __fdiv_rn(127.0f, amax[i]);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int qv = 0;
            if (amax[i] != 0.0f) {
                float v = rintf(__fmul_rn(x[i][j], inv));
                v = fminf(fmaxf(v, -127.0f), 127.0f);
                qv = (int)v;
            }
            q[i][j] = qv;
        }
        sx[i] = (amax[i] == 0.0f) ? 0.0f : __fdiv_rn(amax[i], 127.0f);
    }
}

// operand column (K index inside the tile, e8_kcol order: 32c + 4i + b for block 4c+b, coordinate i) of element 4*lane
// of the tile; the lane's four codes go to columns act_col0(lane) + 4j
__device__ __forceinline__ int act_col0(int lane) {
    const int blk = lane >> 1;
    return 32 * (blk >> 2) + 16 * (lane & 1) + (blk & 3);
}

}  // namespace hq
