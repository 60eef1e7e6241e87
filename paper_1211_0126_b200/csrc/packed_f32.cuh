// packed_f32.cuh -- complex fp32 arithmetic on Blackwell's packed FP32 pipe (PTX add/mul/fma.rn.f32x2, SASS FADD2 /
// FMUL2 / FFMA2).  A complex number is one 64-bit register pair (re, im).  The SASS forms take a scalar register
// broadcast to both halves (R.F32) and a swapped and half-negated pair (-R.F32x2.LO_HI.NP) as operand modifiers, so
//     a + i b,    a + z w  (complex z, w)  =  fma2(z, w.re, fma2(i z, w.im, a))
// cost one and two instructions with no data movement: the SU(3) x half-spinor multiply of the stencil is 36 FFMA2
// instead of 72 FFMA / FMUL, the spin projection 6 FADD2 instead of 12 FADD.  Each half of a packed operation is the
// IEEE fp32 operation (round to nearest), so the 1e-5 parity bar of the fp32 stencil is untouched.
#pragma once

typedef unsigned long long f2;   // (lo, hi) = (re, im)

__device__ __forceinline__ f2 pk(float a, float b)
{
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void upk(f2 v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f2 add2(f2 a, f2 b)
{
    f2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b)
{
    f2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c)
{
    f2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f2 bc(float s) { return pk(s, s); }                     // scalar broadcast (an operand modifier in SASS)
// (re, im) of i^k z for the operand of a packed add / fma (sign and swap are operand modifiers in SASS)
__device__ __forceinline__ f2 c_pos(float re, float im) { return pk(re, im); }      //  z
__device__ __forceinline__ f2 c_neg(float re, float im) { return pk(-re, -im); }    // -z
__device__ __forceinline__ f2 c_i(float re, float im) { return pk(-im, re); }       //  i z
__device__ __forceinline__ f2 c_mi(float re, float im) { return pk(im, -re); }      // -i z
