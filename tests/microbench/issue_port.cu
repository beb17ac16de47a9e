// issue-port micro-benchmark: does FFMA2 / MUFU block the issue port for a 2nd cycle?
#include <cstdio>
#include <cuda_runtime.h>
typedef unsigned long long f2;
#define FMA2(d,a,b) asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b))
#define FMA1(d,a,b) asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(d) : "f"(a), "f"(b))
#define MNMX(d,a) asm volatile("max.f32 %0, %0, %1;" : "+f"(d) : "f"(a))
#define IADD(d,a) asm volatile("add.s32 %0, %0, %1;" : "+r"(d) : "r"(a))
#define LOP(d,a) asm volatile("xor.b32 %0, %0, %1;" : "+r"(d) : "r"(a))
#define EX2(d) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(d))
#define SETP_SEL(d,a,b) asm volatile("{ .reg .pred p; setp.gt.f32 p, %1, %2; selp.f32 %0, %1, %0, p; }" : "+f"(d) : "f"(a), "f"(b))
template <int MODE> __global__ void k(float* out, int iters, float seed, long long* cyc)
{
    f2 p[8]; float s[8]; int r[8];
    for (int i = 0; i < 8; ++i) { p[i] = __float_as_uint(seed + i) | ((f2)__float_as_uint(seed * 2 + i) << 32); s[i] = seed + i; r[i] = threadIdx.x + i; }
    f2 a = p[0], b = p[1]; float fa = seed * 0.5f, fb = seed * 0.25f; int ia = threadIdx.x | 1;
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (MODE == 0) { FMA2(p[i], a, b); }                                  // 8 FFMA2
            if (MODE == 1) { FMA1(s[i], fa, fb); }                                // 8 FFMA
            if (MODE == 2) { FMA2(p[i], a, b); MNMX(s[i], fa); }                  // 8 FFMA2 + 8 FMNMX
            if (MODE == 3) { FMA2(p[i], a, b); IADD(r[i], ia); }                  // 8 FFMA2 + 8 IADD
            if (MODE == 4) { FMA2(p[i], a, b); IADD(r[i], ia); LOP(r[(i + 4) & 7], ia); }   // 8 FFMA2 + 16 ALU
            if (MODE == 5) { FMA1(s[i], fa, fb); IADD(r[i], ia); }                // 8 FFMA + 8 IADD
            if (MODE == 6) { FMA2(p[i], a, b); FMA1(s[i], fa, fb); }              // 8 FFMA2 + 8 FFMA
            if (MODE == 7) { EX2(s[i]); }                                         // 8 MUFU
            if (MODE == 8) { EX2(s[i]); IADD(r[i], ia); IADD(r[(i+1)&7], ia); IADD(r[(i+2)&7], ia); IADD(r[(i+3)&7], ia); IADD(r[(i+4)&7], ia); IADD(r[(i+5)&7], ia); IADD(r[(i+6)&7], ia); }   // 8 MUFU + 56 IADD
            if (MODE == 9) { EX2(s[i]); FMA2(p[i], a, b); FMA2(p[(i+1)&7], a, b); FMA2(p[(i+2)&7], a, b); }   // 8 MUFU + 24 FFMA2
            if (MODE == 10) { FMA2(p[i], a, b); SETP_SEL(s[i], fa, fb); }         // 8 FFMA2 + 8 (FSETP+FSEL)
            if (MODE == 11) { IADD(r[i], ia); }                                   // 8 IADD
            if (MODE == 12) { EX2(s[i]); FMA1(s[(i+1)&7], fa, fb); FMA1(s[(i+2)&7], fa, fb); FMA1(s[(i+3)&7], fa, fb); FMA1(s[(i+4)&7], fa, fb); FMA1(s[(i+5)&7], fa, fb); FMA1(s[(i+6)&7], fa, fb); FMA1(s[(i+7)&7], fa, fb); }  // 8 MUFU + 56 FFMA
        }
    }
    long long t1 = clock64();
    float acc = 0; for (int i = 0; i < 8; ++i) acc += s[i] + __uint_as_float((unsigned)p[i]) + __uint_as_float((unsigned)(p[i] >> 32)) + r[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}
template <int MODE> void run(const char* name, int n_instr, int warps_per_smsp)
{
    float* out; long long* cyc; cudaMalloc(&out, 148 * 1024 * 4); cudaMalloc(&cyc, 8);
    const int iters = 4000, threads = warps_per_smsp * 4 * 32;
    k<MODE><<<148, threads>>>(out, 10, 1.0f, cyc);
    k<MODE><<<148, threads>>>(out, iters, 1.0f, cyc);
    long long h; cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
    // cycles per group (8 x the pattern) per SMSP = elapsed / iters ; each SMSP runs warps_per_smsp warps
    printf("%-28s warps/SMSP %d: %.2f cycles per group per warp-slot -> %.2f cycles per warp-group, %.3f instr/clk\n", name, warps_per_smsp,
           (double)h / iters, (double)h / iters / warps_per_smsp, n_instr * (double)warps_per_smsp * iters / h);
    cudaFree(out); cudaFree(cyc);
}
int main()
{
    for (int w : {4, 8}) {
        run<0>("8 FFMA2", 8, w); run<1>("8 FFMA", 8, w); run<11>("8 IADD", 8, w); run<2>("8 FFMA2 + 8 FMNMX", 16, w); run<3>("8 FFMA2 + 8 IADD", 16, w);
        run<4>("8 FFMA2 + 16 ALU", 24, w); run<5>("8 FFMA + 8 IADD", 16, w); run<6>("8 FFMA2 + 8 FFMA", 16, w); run<10>("8 FFMA2 + 8 FSETP+SEL", 24, w);
        run<7>("8 MUFU", 8, w); run<8>("8 MUFU + 56 IADD", 64, w); run<12>("8 MUFU + 56 FFMA", 64, w); run<9>("8 MUFU + 24 FFMA2", 32, w);
    }
    return 0;
}
