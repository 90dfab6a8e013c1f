// pipes.cu -- pipe microbenchmarks behind the half-precision kernel design (profiles/r2_pipes.md):
// cycles per warp instruction per SM sub-partition for FFMA2 / PRMT / integer / I2F streams and their mixes.
// Not part of libtm_b200.so.  Build and run:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/pipes paper_1311_4462_b200/csrc/microbench/pipes.cu && /tmp/pipes
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#define ITER 512
typedef unsigned long long u64;
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 d; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
// d = (s, s) * b + c with the scalar broadcast operand the kernels use (SASS: FFMA2 Rd, Rs.F32, Rb.F32x2, Rc.F32x2)
__device__ __forceinline__ u64 fma2s(float s, u64 b, u64 c) { u64 d; asm volatile("{.reg .b64 t; mov.b64 t, {%1, %1}; fma.rn.f32x2 %0, t, %2, %3;}" : "=l"(d) : "f"(s), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t s) { uint32_t d; asm volatile("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(s)); return d; }
__device__ __forceinline__ float i2f_lo(uint32_t w) { float f; asm volatile("{.reg .b16 l, h; mov.b32 {l, h}, %1; cvt.rn.f32.s16 %0, l;}" : "=f"(f) : "r"(w)); return f; }
__device__ __forceinline__ float i2f_hi(uint32_t w) { float f; asm volatile("{.reg .b16 l, h; mov.b32 {l, h}, %1; cvt.rn.f32.s16 %0, h;}" : "=f"(f) : "r"(w)); return f; }
__device__ __forceinline__ float i2fp(int w) { float f; asm volatile("cvt.rn.f32.s32 %0, %1;" : "=f"(f) : "r"(w)); return f; }
__device__ __forceinline__ uint32_t iadd(uint32_t a, uint32_t b) { uint32_t d; asm volatile("add.u32 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b)); return d; }
__device__ __forceinline__ uint32_t imad(uint32_t a, uint32_t b, uint32_t c) { uint32_t d; asm volatile("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c)); return d; }
__device__ __forceinline__ float ffma(float a, float b, float c) { float d; asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c)); return d; }
__device__ __forceinline__ uint32_t lop(uint32_t a, uint32_t b, uint32_t c) { uint32_t d; asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(d) : "r"(a), "r"(b), "r"(c)); return d; }

template <int T> __global__ void __launch_bounds__(512, 1) kern(u64 *cyc, float *sink, const uint32_t *in)
{
    u64 a[8]; uint32_t r[8]; float f[8];
    for (int i = 0; i < 8; i++) { a[i] = ((u64)in[i] << 32) | in[i + 8]; r[i] = in[16 + i] + threadIdx.x; f[i] = (T >= 16 && T <= 18) ? __uint_as_float(in[40 + i]) : 0.f; }
    const u64 b = ((u64)in[24] << 32) | in[25], c = ((u64)in[26] << 32) | in[27];
    const u64 b2 = ((u64)in[28] << 32) | in[29], c2 = ((u64)in[30] << 32) | in[31];
    const uint32_t m = in[32], s = in[33];
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < ITER; it++) {
        if constexpr (T == 0) {            // FFMA2 x8, shared b,c
#pragma unroll
            for (int i = 0; i < 8; i++) a[i] = fma2(a[i], b, c);
        } else if constexpr (T == 1) {     // PRMT x8
#pragma unroll
            for (int i = 0; i < 8; i++) r[i] = prmt(r[i], m, s);
        } else if constexpr (T == 2) {     // I2F.S16 x8
#pragma unroll
            for (int i = 0; i < 8; i++) r[i] = __float_as_uint((i & 1) ? i2f_hi(r[i]) : i2f_lo(r[i]));
        } else if constexpr (T == 3) {     // FFMA2 + PRMT 1:1
#pragma unroll
            for (int i = 0; i < 8; i++) { a[i] = fma2(a[i], b, c); r[i] = prmt(r[i], m, s); }
        } else if constexpr (T == 4) {     // FFMA2 + I2F 1:1
#pragma unroll
            for (int i = 0; i < 8; i++) { a[i] = fma2(a[i], b, c); r[i] = __float_as_uint((i & 1) ? i2f_hi(r[i]) : i2f_lo(r[i])); }
        } else if constexpr (T == 5) {     // FFMA2 + I2F 2:1 (8 + 4)
#pragma unroll
            for (int i = 0; i < 8; i++) { a[i] = fma2(a[i], b, c); if (i & 1) r[i] = __float_as_uint(i2f_hi(r[i])); }
        } else if constexpr (T == 6) {     // I2FP.S32 x8
#pragma unroll
            for (int i = 0; i < 8; i++) r[i] = __float_as_uint(i2fp((int)r[i]));
        } else if constexpr (T == 7) {     // FFMA2 + IADD 1:1
#pragma unroll
            for (int i = 0; i < 8; i++) { a[i] = fma2(a[i], b, c); r[i] = iadd(r[i], m); }
        } else if constexpr (T == 8) {     // IADD x8
#pragma unroll
            for (int i = 0; i < 8; i++) r[i] = iadd(r[i], m);
        } else if constexpr (T == 9) {     // IMAD x8
#pragma unroll
            for (int i = 0; i < 8; i++) r[i] = imad(r[i], m, s);
        } else if constexpr (T == 10) {    // FFMA2 3 distinct operands per instr (a[i] = a[i]*a[i+1] + a[i+2])
#pragma unroll
            for (int i = 0; i < 8; i++) a[i] = fma2(a[(i + 1) & 7], a[(i + 2) & 7], a[i]);
        } else if constexpr (T == 11) {    // FFMA2 + PRMT 2:1
#pragma unroll
            for (int i = 0; i < 8; i++) { a[i] = fma2(a[i], b, c); if (i & 1) r[i] = prmt(r[i], m, s); }
        } else if constexpr (T == 12) {    // FFMA x8 scalar
#pragma unroll
            for (int i = 0; i < 8; i++) f[i] = ffma(f[i], __uint_as_float(m), __uint_as_float(s));
        } else if constexpr (T == 13) {    // FFMA2 + PRMT + I2F  (8 + 4 + 4)
#pragma unroll
            for (int i = 0; i < 8; i++) { a[i] = fma2(a[i], b, c); if (i & 1) r[i] = prmt(r[i], m, s); else r[i] = __float_as_uint(i2f_lo(r[i])); }
        } else if constexpr (T == 14) {    // LOP3 x8
#pragma unroll
            for (int i = 0; i < 8; i++) r[i] = lop(r[i], m, s);
        } else if constexpr (T == 16) {    // the kernels' form, nothing shared: scalar x pair + accumulator pair, all distinct
#pragma unroll
            for (int i = 0; i < 8; i++) a[i] = fma2s(f[i], a[(i + 3) & 7], a[i]);
        } else if constexpr (T == 17) {    // the same scalar in all 8 (reuse of the scalar operand)
#pragma unroll
            for (int i = 0; i < 8; i++) a[i] = fma2s(f[0], a[(i + 3) & 7], a[i]);
        } else if constexpr (T == 18) {    // the same pair in all 8, distinct scalars (reuse of the pair operand)
#pragma unroll
            for (int i = 0; i < 8; i++) a[i] = fma2s(f[i], b, a[i]);
        } else if constexpr (T == 15) {    // FFMA2 alternating two operand sets + I2F 4:1
#pragma unroll
            for (int i = 0; i < 8; i++) { a[i] = fma2(a[i], (i & 1) ? b : b2, (i & 2) ? c : c2); if ((i & 3) == 3) r[i] = __float_as_uint(i2f_hi(r[i])); }
        }
    }
    const long long t1 = clock64();
    float acc = 0.f;
    for (int i = 0; i < 8; i++) acc += f[i] + __uint_as_float(r[i]) + __uint_as_float((uint32_t)a[i]) + __uint_as_float((uint32_t)(a[i] >> 32));
    sink[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (threadIdx.x == 0) cyc[blockIdx.x] = (u64)(t1 - t0);
}
template <int T> void run(const char *name, int per_iter, u64 *cyc, float *sink, uint32_t *in)
{
    for (int warps = 4; warps <= 16; warps *= 2) {
        kern<T><<<148, warps * 32>>>(cyc, sink, in);
        kern<T><<<148, warps * 32>>>(cyc, sink, in);
        cudaDeviceSynchronize();
        u64 h[148]; cudaMemcpy(h, cyc, sizeof(h), cudaMemcpyDeviceToHost);
        double avg = 0; for (int i = 0; i < 148; i++) avg += h[i]; avg /= 148;
        printf("%-34s warps/SM %2d  cycles/inst/SMSP %.3f  (per group of %d: %.2f)\n", name, warps, avg / ((double)ITER * per_iter * (warps / 4)), per_iter,
               avg / ((double)ITER * (warps / 4)));
    }
}
int main()
{
    u64 *cyc; float *sink; uint32_t *in;
    cudaMalloc(&cyc, 148 * 8); cudaMalloc(&sink, 148 * 512 * 4); cudaMalloc(&in, 64 * 4);
    uint32_t h[64]; for (int i = 0; i < 64; i++) h[i] = 0x3f800000u + i * 12345u;
    for (int i = 40; i < 48; i++) h[i] = 0x3f000000u + i * 77u;     // scalars ~0.5: the chains stay finite h[32] = 0x4B000000u; h[33] = 0x7610;
    cudaMemcpy(in, h, sizeof(h), cudaMemcpyHostToDevice);
    run<0>("FFMA2", 8, cyc, sink, in);
    run<10>("FFMA2 3 distinct regs", 8, cyc, sink, in);
    run<16>("FFMA2 scalar x pair + pair, distinct", 8, cyc, sink, in);
    run<17>("FFMA2 scalar x pair + pair, same scalar", 8, cyc, sink, in);
    run<18>("FFMA2 scalar x pair + pair, same pair", 8, cyc, sink, in);
    run<12>("FFMA scalar", 8, cyc, sink, in);
    run<1>("PRMT", 8, cyc, sink, in);
    run<14>("LOP3", 8, cyc, sink, in);
    run<8>("IADD", 8, cyc, sink, in);
    run<9>("IMAD", 8, cyc, sink, in);
    run<2>("I2F.S16", 8, cyc, sink, in);
    run<6>("I2FP.S32", 8, cyc, sink, in);
    run<3>("FFMA2+PRMT 1:1", 16, cyc, sink, in);
    run<11>("FFMA2+PRMT 2:1", 12, cyc, sink, in);
    run<4>("FFMA2+I2F 1:1", 16, cyc, sink, in);
    run<5>("FFMA2+I2F 2:1", 12, cyc, sink, in);
    run<15>("FFMA2(4 opsets)+I2F 4:1", 10, cyc, sink, in);
    run<13>("FFMA2+PRMT+I2F 8+4+4", 16, cyc, sink, in);
    run<7>("FFMA2+IADD 1:1", 16, cyc, sink, in);
    return 0;
}
