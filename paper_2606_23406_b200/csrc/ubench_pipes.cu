// ubench_pipes.cu — issue-rate microbenchmark behind DESIGN.md §6 (ALU / FMA / XU pipe rates on sm_100a).  A
// stand-alone developer tool, not part of libhq.so:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/ubench_pipes paper_2606_23406_b200/csrc/ubench_pipes.cu && /tmp/ubench_pipes
// Results of round 1: profiles/r01_issue_rates.md.
// Each kernel: 8 independent dependency chains per thread, ITER iterations, all 148 SMs x 2 CTAs x 1024 threads.
// Prints warp-instructions per clock64 tick per SM; clock64 ticked at HALF the SM clock on the measured boxes
// ("implied MHz" ~ 975 at 1965 MHz), so halve the printed rates: see profiles/r01_issue_rates.md.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#define ITER 4096
#define CH 8

template <int OP>
__global__ void __launch_bounds__(1024) k(uint32_t* out, uint32_t seed, long long* clk) {
    __shared__ uint32_t lut[1024];
    for (int i = threadIdx.x; i < 1024; i += blockDim.x) lut[i] = (i * 2654435761u) ^ seed;
    __syncthreads();
    uint32_t a[CH], b = seed | 1, c = seed * 3 + 7;
#pragma unroll
    for (int i = 0; i < CH; ++i) a[i] = threadIdx.x * 31 + i * 7 + seed;
    long long t0 = clock64();
    for (int it = 0; it < ITER; ++it) {
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            if (OP == 0) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(b), "r"(c));
            if (OP == 1) asm volatile("shf.l.wrap.b32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
            if (OP == 2) asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
            if (OP == 3) asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(b));
            if (OP == 4) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
            if (OP == 5) asm volatile("popc.b32 %0, %0;" : "+r"(a[i]));
            if (OP == 6) asm volatile("clz.b32 %0, %0;" : "+r"(a[i]));
            if (OP == 7) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"((uint32_t)__cvta_generic_to_shared(&lut[a[i] & 1023]))); a[i] = v; }
            if (OP == 8) { float f; asm volatile("cvt.rn.f32.s32 %0, %1;" : "=f"(f) : "r"(a[i])); a[i] = __float_as_uint(f); }
            if (OP == 9) {  // mix: lop3 + imad alternating
                if (i & 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(b), "r"(c));
                else asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
            }
            if (OP == 10) {  // mix: shf + prmt + lop3 + imad
                if ((i & 3) == 0) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(b), "r"(c));
                if ((i & 3) == 1) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
                if ((i & 3) == 2) asm volatile("shf.l.wrap.b32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
                if ((i & 3) == 3) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
            }
            if (OP == 11) asm volatile("shl.b32 %0, %0, 3;" : "+r"(a[i]));
            if (OP == 12) asm volatile("and.b32 %0, %0, 0x0f0f0f0f;" : "+r"(a[i]));
            if (OP == 13) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"((uint32_t)__cvta_generic_to_shared(&lut[(threadIdx.x + i) & 1023]))); a[i] ^= v; }
            if (OP == 14) asm volatile("shf.r.clamp.b32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
            if (OP == 15) asm volatile("vabsdiff4.u32.u32.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
            if (OP == 16) asm volatile("dp4a.u32.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
            if (OP == 17) asm volatile("mul.wide.u16 %0, %1, %2;" : "=r"(a[i]) : "h"((unsigned short)a[i]), "h"((unsigned short)b));
            if (OP == 18) { float f = __uint_as_float(a[i]); asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(__uint_as_float(b)), "f"(__uint_as_float(c))); a[i] = __float_as_uint(f); }
            if (OP == 19) asm volatile("bfe.u32 %0, %0, %1, 8;" : "+r"(a[i]) : "r"(b));
            if (OP == 21) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(b));
            if (OP == 22) asm volatile("mad.hi.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
            if (OP == 23) asm volatile("shr.u32 %0, %0, 7;" : "+r"(a[i]));
            if (OP == 24) { if (i&1) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(b)); else asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(b), "r"(c)); }
            if (OP == 25) asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(*(unsigned long long*)&a[i&~1]) : "r"(b), "r"(c));
            if (OP == 26) asm volatile("slct.u32.s32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"((int)c - (int)a[i]));
            if (OP == 27) { if (i&1) asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(b)); else asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(b), "r"(c)); }
            if (OP == 28) { if (i&1) asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(b)); else asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c)); }
            if (OP == 20) asm volatile("bfi.b32 %0, %1, %0, %2, 8;" : "+r"(a[i]) : "r"(b), "r"(c));
        }
    }
    long long t1 = clock64();
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < CH; ++i) s ^= a[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *clk = t1 - t0;
}

template <int OP>
void run(const char* name, uint32_t* out, long long* clk) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    int grid = 148 * 2;
    k<OP><<<grid, 1024>>>(out, 12345u, clk);
    cudaDeviceSynchronize();
    cudaEventRecord(e0);
    k<OP><<<grid, 1024>>>(out, 12345u, clk);
    cudaEventRecord(e1);
    cudaDeviceSynchronize();
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    long long c; cudaMemcpy(&c, clk, 8, cudaMemcpyDeviceToHost);
    double winstr_per_sm = (double)ITER * CH * 32 /*warps per CTA*/ * 2 /*CTAs per SM*/;
    printf("%-28s %8.3f ms  block0 clks %10lld  warp-instr/clk/SM (by block0 clk) %6.3f   implied MHz %7.1f  err=%s\n", name, ms, c,
           winstr_per_sm / (double)c, (double)c / ms / 1e3, cudaGetErrorString(cudaGetLastError()));
}

int main() {
    uint32_t* out; long long* clk;
    cudaMalloc(&out, 148 * 2 * 1024 * 4); cudaMalloc(&clk, 8);
    run<0>("lop3", out, clk);
    run<1>("shf.l.wrap (funnel)", out, clk);
    run<14>("shf.r.clamp (funnel)", out, clk);
    run<2>("prmt (reg selector)", out, clk);
    run<3>("iadd", out, clk);
    run<4>("imad", out, clk);
    run<5>("popc", out, clk);
    run<6>("clz", out, clk);
    run<7>("lds random (dependent)", out, clk);
    run<13>("lds conflict-free", out, clk);
    run<8>("i2f", out, clk);
    run<9>("mix lop3+imad", out, clk);
    run<10>("mix lop3/shf + imad", out, clk);
    run<11>("shl imm", out, clk);
    run<12>("and imm", out, clk);
    run<15>("vabsdiff4", out, clk);
    run<16>("dp4a", out, clk);
    run<17>("mul.wide.u16", out, clk);
    run<18>("ffma", out, clk);
    run<19>("bfe", out, clk);
    run<20>("bfi", out, clk);
    run<21>("mul.hi.u32", out, clk);
    run<22>("mad.hi.u32", out, clk);
    run<23>("shr imm", out, clk);
    run<24>("mix mul.hi + lop3", out, clk);
    run<26>("sel? (slct)", out, clk);
    run<27>("mix iadd + lop3", out, clk);
    run<28>("mix iadd + imad", out, clk);
    return 0;
}
