// tm_f2.cuh -- packed-FP32 (Blackwell FFMA2 / FADD2 / FMUL2, PTX *.f32x2) building blocks.
//
// B200 issues at most one warp instruction per SM sub-partition per clock; a scalar FFMA stream therefore tops
// out at the FP32 peak with every issue slot taken.  The f32x2 forms do two lanes per instruction at the same
// pipe rate (measured: 74 TFLOP/s at 2 warp-inst/clk/SM), which halves the issue pressure of the dslash
// arithmetic and leaves slots for address, conversion and load instructions.  ptxas folds scalar broadcasts
// (R.F32), lane swaps (.F32x2.LO_HI) and negations into the FFMA2 operands, so none of the helpers below costs a
// MOV (checked with cuobjdump -sass).
//
// A pair always holds the SAME (color, re/im) of the two spin components of one half of the spinor:
//   (spin 0, spin 1) for the upper half, (spin 2, spin 3) for the lower half   (basis: DESIGN.md C5).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define TM_DEV __device__ __forceinline__

struct __align__(8) f2 {
    float x, y;
};

TM_DEV f2 mk2(float a, float b)
{
    f2 r;
    r.x = a;
    r.y = b;
    return r;
}
TM_DEV f2 bc2(float a) { return mk2(a, a); }          // scalar broadcast (free: R.F32 operand)
TM_DEV f2 sw2(f2 a) { return mk2(a.y, a.x); }         // lane swap (free: .F32x2.LO_HI operand)
TM_DEV f2 neg2(f2 a) { return mk2(-a.x, -a.y); }      // free: operand negation

TM_DEV unsigned long long pk2(f2 a)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
    return r;
}
TM_DEV f2 up2(unsigned long long r)
{
    f2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(r));
    return d;
}
TM_DEV f2 fma2(f2 a, f2 b, f2 c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(pk2(a)), "l"(pk2(b)), "l"(pk2(c)));
    return up2(d);
}
TM_DEV f2 mul2(f2 a, f2 b)
{
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk2(a)), "l"(pk2(b)));
    return up2(d);
}
TM_DEV f2 add2(f2 a, f2 b)
{
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk2(a)), "l"(pk2(b)));
    return up2(d);
}
TM_DEV f2 sub2(f2 a, f2 b) { return add2(a, neg2(b)); }

// ---- 16-bit fixed point <-> float without the (quarter-rate) conversion unit --------------------------
// Stored int16 are OFFSET BINARY: u = q + 32768.  A 32-bit word holds the pair's two lanes.
//   float bits 0x4B000000 | u  =  2^23 + u   ->   q = that - (2^23 + 32768), exact.
#define TM_CVT_MAGIC 8421376.0f            /* 2^23 + 2^15 */
// The biased pair (2^23 + u_lo, 2^23 + u_hi) = (M + q_lo, M + q_hi), M = TM_CVT_MAGIC: 2 PRMT, no arithmetic.
// Sums and differences of biased values in which the M cancel are exact (project_f2 uses this).
TM_DEV f2 cvt_pair_biased(uint32_t w)
{
    return mk2(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7610)), __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7632)));
}
TM_DEV f2 cvt_pair(uint32_t w)             // -> (q_lo, q_hi) as integer-valued floats: 2 PRMT + 1 FADD2
{
    const float lo = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7610));
    const float hi = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7632));
    return add2(mk2(lo, hi), bc2(-TM_CVT_MAGIC));
}
// rint(v * s) for |v * s| <= 32767 as offset binary, two lanes packed into one word: 1 FFMA2 + 1 PRMT.
//   v*s + (1.5 * 2^23 + 32768): the low 16 mantissa bits are q + 32768 (round to nearest even by the FMA).
#define TM_RND_MAGIC 12615680.0f           /* 1.5 * 2^23 + 2^15 */
TM_DEV uint32_t quant_pair(f2 v, float s)
{
    const f2 t = fma2(v, bc2(s), bc2(TM_RND_MAGIC));
    return __byte_perm(__float_as_uint(t.x), __float_as_uint(t.y), 0x5410);
}
