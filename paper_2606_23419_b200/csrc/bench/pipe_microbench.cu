// pipe_microbench.cu — issue rate (warp-instr/clk/SM) of the instructions the VMM inner loop uses; not part of libgrinqh.so.
// nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/pipe_microbench paper_2606_23419_b200/csrc/bench/pipe_microbench.cu && /tmp/pipe_microbench
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define ITERS 4096
template <int MODE>
__global__ void k(uint32_t* out, uint32_t seed, long long* cyc) {
    uint32_t a[8]; float f[8];
    uint16_t xh = (uint16_t)(0x3c00 + (seed & 3));
    for (int i = 0; i < 8; ++i) { a[i] = seed * (i + 1) + threadIdx.x; f[i] = (float)i; }
    long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (MODE == 0) asm volatile("fma.rn.f32 %0, %0, %1, %0;" : "+f"(f[i]) : "f"(f[(i + 1) & 7]));
            if (MODE == 1) asm volatile("{.reg .b16 lo,hi; mov.b32 {lo,hi}, %1; fma.rn.f32.f16 %0, lo, %2, %0;}" : "+f"(f[i]) : "r"(a[i]), "h"(xh));
            if (MODE == 2) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]), "r"(seed));
            if (MODE == 3) asm volatile("prmt.b32 %0, %0, %1, 0x4140;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]));
            if (MODE == 4) asm volatile("shf.l.wrap.b32 %0, %0, %1, 3;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]));
            if (MODE == 5) { // FFMA2
                asm volatile("{.reg .b64 d, s; mov.b64 d, {%0,%1}; mov.b64 s, {%2,%2}; fma.rn.f32x2 d, d, s, d; mov.b64 {%0,%1}, d;}"
                    : "+f"(f[i]), "+f"(f[(i + 4) & 7]) : "f"(1.0001f));
            }
            if (MODE == 6) { // mix 1 LOP3 + 1 FHFMA
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]), "r"(seed));
                asm volatile("{.reg .b16 lo,hi; mov.b32 {lo,hi}, %1; fma.rn.f32.f16 %0, lo, %2, %0;}" : "+f"(f[i]) : "r"(a[(i+3)&7]), "h"(xh));
            }
            if (MODE == 7) { // mix 1 PRMT + 2 FHFMA (the accumulate pattern)
                uint32_t h; asm volatile("prmt.b32 %0, %1, 0, 0x4140;" : "=r"(h) : "r"(a[i]));
                asm volatile("{.reg .b16 lo,hi; mov.b32 {lo,hi}, %1; fma.rn.f32.f16 %0, lo, %2, %0;}" : "+f"(f[i]) : "r"(h), "h"(xh));
                asm volatile("{.reg .b16 lo,hi; mov.b32 {lo,hi}, %1; fma.rn.f32.f16 %0, hi, %2, %0;}" : "+f"(f[(i+4)&7]) : "r"(h), "h"(xh));
            }
            if (MODE == 8) asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(f[i]) : "f"(f[(i + 1) & 7]), "f"(1.5f)); // imm? (reg const)
            if (MODE == 9) { // HFMA2
                asm volatile("fma.rn.f16x2 %0, %0, %1, %0;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]));
            }
            if (MODE == 10) { // IMAD
                asm volatile("mad.lo.u32 %0, %0, %1, %0;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]));
            }
            if (MODE == 11) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]));
            if (MODE == 12) { // IMAD.WIDE: 64-bit product + 64-bit addend
                asm volatile("{.reg .b64 d; mov.b64 d, {%0,%1}; mad.wide.u32 d, %0, %2, d; mov.b64 {%0,%1}, d;}" : "+r"(a[i]), "+r"(a[(i + 4) & 7]) : "r"(seed));
            }
            if (MODE == 13) asm volatile("shr.u32 %0, %0, 1;" : "+r"(a[i]));
            if (MODE == 14) asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]));
            if (MODE == 15) { // 2 LOP3 + 1 mul.hi + 1 IMAD (a transpose pair with the right shift on the fma pipe)
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]), "r"(seed));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0xE4;" : "+r"(a[(i+2)&7]) : "r"(a[(i + 3) & 7]), "r"(seed));
                asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(a[(i+4)&7]) : "r"(seed));
                asm volatile("mad.lo.u32 %0, %0, %1, %0;" : "+r"(a[(i+5)&7]) : "r"(seed));
            }
            if (MODE == 16) { // 2 LOP3 + 1 SHF + 1 IMAD (the pair as committed)
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]), "r"(seed));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0xE4;" : "+r"(a[(i+2)&7]) : "r"(a[(i + 3) & 7]), "r"(seed));
                asm volatile("shf.l.wrap.b32 %0, %0, %1, 3;" : "+r"(a[(i+4)&7]) : "r"(a[(i + 1) & 7]));
                asm volatile("mad.lo.u32 %0, %0, %1, %0;" : "+r"(a[(i+5)&7]) : "r"(seed));
            }
        }
    }
    long long t1 = clock64();
    uint32_t r = 0; for (int i = 0; i < 8; ++i) r ^= a[i] ^ __float_as_uint(f[i]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}
template <int MODE> void run(const char* name, int per_iter) {
    uint32_t* out; long long* cyc; cudaMalloc(&out, 148 * 1024 * 4); cudaMalloc(&cyc, 8);
    for (int warps : {4, 8, 16, 32}) {
        k<MODE><<<148, warps * 32>>>(out, 12345, cyc); cudaDeviceSynchronize();
        k<MODE><<<148, warps * 32>>>(out, 12345, cyc); cudaDeviceSynchronize();
        long long c; cudaMemcpy(&c, cyc, 8, cudaMemcpyDeviceToHost);
        double warp_inst = (double)ITERS * 8 * per_iter * warps;
        printf("%-28s warps/SM %2d  cycles %8lld  warp-inst/clk/SM %.3f\n", name, warps, c, warp_inst / c);
    }
    cudaFree(out); cudaFree(cyc);
}
int main() {
    run<0>("FFMA 3reg", 1); run<1>("FHFMA (f32+=f16*f16)", 1); run<2>("LOP3", 1); run<3>("PRMT", 1); run<4>("SHF", 1);
    run<5>("FFMA2 (counts as 1 inst)", 1); run<6>("LOP3+FHFMA", 2); run<7>("PRMT+2FHFMA", 3); run<8>("FFMA reg*const", 1);
    run<9>("HFMA2", 1); run<10>("IMAD", 1); run<11>("IMAD.HI", 1); run<12>("IMAD.WIDE", 1); run<13>("SHR", 1); run<14>("IADD", 1); run<15>("2LOP3+HI+IMAD", 4); run<16>("2LOP3+SHF+IMAD", 4);
    cudaError_t e = cudaGetLastError(); printf("err %s\n", cudaGetErrorString(e));
    return 0;
}
