// cdmt_fft2.cuh -- packed-FP32 (f32x2) butterflies for sm_100a.
//
// Blackwell's FADD2 / FMUL2 / FFMA2 work on an aligned register pair and deliver two FP32
// results per issue slot and per 64-bit operand read.  A "P2" is such a pair; a "C2" is a pair
// of complex numbers held as (re_lo, re_hi), (im_lo, im_hi): the two lanes carry two
// independent transforms (the even-bin and the odd-bin half of one backward FFT), so every
// butterfly, twiddle and constant below is applied to both at once.  Scalars broadcast to
// both lanes (ptxas folds the {w, w} pack into an .F32 operand) and negations fold into
// operand modifiers, so none of the helpers costs an extra instruction.
//
// Transform: X[k] = sum_n x[n] exp(+2 pi i k n / R)  (the backward FFT of PAPER.md:119).
#pragma once
#include <cuda_runtime.h>

namespace cdmt {

typedef unsigned long long P2;

__device__ __forceinline__ P2 pk(float lo, float hi)
{
    P2 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void upk(P2 v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ float lo_of(P2 v) { float a, b; upk(v, a, b); return a; }
__device__ __forceinline__ float hi_of(P2 v) { float a, b; upk(v, a, b); return b; }
__device__ __forceinline__ P2 bc(float s) { return pk(s, s); }
__device__ __forceinline__ P2 neg2(P2 a)
{
    float x, y;
    upk(a, x, y);
    return pk(-x, -y);
}
__device__ __forceinline__ P2 add2(P2 a, P2 b)
{
    P2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ P2 sub2(P2 a, P2 b)
{
    P2 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ P2 mul2(P2 a, P2 b)
{
    P2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ P2 fma2(P2 a, P2 b, P2 c)
{
    P2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}

struct C2 {
    P2 re, im;
};

__device__ __forceinline__ C2 cadd(C2 a, C2 b) { return C2{add2(a.re, b.re), add2(a.im, b.im)}; }
__device__ __forceinline__ C2 csub(C2 a, C2 b) { return C2{sub2(a.re, b.re), sub2(a.im, b.im)}; }
// multiply by +i
__device__ __forceinline__ C2 roti(C2 a) { return C2{neg2(a.im), a.re}; }
// multiply both lanes by the same scalar c + i s
__device__ __forceinline__ C2 cmuls(C2 a, float c, float s)
{
    return C2{fma2(neg2(a.im), bc(s), mul2(a.re, bc(c))), fma2(a.im, bc(c), mul2(a.re, bc(s)))};
}
// multiply lane-wise by (hr + i hi)
__device__ __forceinline__ C2 cmulp(C2 a, P2 hr, P2 hi)
{
    return C2{fma2(neg2(a.im), hi, mul2(a.re, hr)), fma2(a.im, hr, mul2(a.re, hi))};
}

constexpr float kP_R2 = 0.70710678118654752440f;  // cos(pi/4)
constexpr float kP_C8 = 0.92387953251128675613f;  // cos(pi/8)
constexpr float kP_S8 = 0.38268343236508977173f;  // sin(pi/8)

// multiply by exp(+2 pi i e / 8), e = 1, 3: three instructions each
__device__ __forceinline__ C2 mulw8_1(C2 a)
{
    const P2 t = mul2(a.im, bc(kP_R2));
    return C2{fma2(a.re, bc(kP_R2), neg2(t)), fma2(a.re, bc(kP_R2), t)};
}
__device__ __forceinline__ C2 mulw8_3(C2 a)
{
    const P2 t = mul2(a.im, bc(kP_R2));
    return C2{fma2(a.re, bc(-kP_R2), neg2(t)), fma2(a.re, bc(kP_R2), neg2(t))};
}

__device__ __forceinline__ void pdft2(C2 &a, C2 &b)
{
    const C2 t = a;
    a = cadd(t, b);
    b = csub(t, b);
}
__device__ __forceinline__ void pdft4(C2 &v0, C2 &v1, C2 &v2, C2 &v3)
{
    const C2 a = cadd(v0, v2), b = csub(v0, v2);
    const C2 c = cadd(v1, v3), d = roti(csub(v1, v3));
    v0 = cadd(a, c);
    v1 = cadd(b, d);
    v2 = csub(a, c);
    v3 = csub(b, d);
}

template <int R>
struct PDft;

template <>
struct PDft<2> {
    static __device__ __forceinline__ void run(C2 *v) { pdft2(v[0], v[1]); }
};
template <>
struct PDft<4> {
    static __device__ __forceinline__ void run(C2 *v) { pdft4(v[0], v[1], v[2], v[3]); }
};
template <>
struct PDft<8> {
    // n = 2 n1 + n2, k = k1 + 4 k2
    static __device__ __forceinline__ void run(C2 *v)
    {
        pdft4(v[0], v[2], v[4], v[6]);
        pdft4(v[1], v[3], v[5], v[7]);
        v[3] = mulw8_1(v[3]);
        v[5] = roti(v[5]);
        v[7] = mulw8_3(v[7]);
        const C2 x0 = cadd(v[0], v[1]), x4 = csub(v[0], v[1]);
        const C2 x1 = cadd(v[2], v[3]), x5 = csub(v[2], v[3]);
        const C2 x2 = cadd(v[4], v[5]), x6 = csub(v[4], v[5]);
        const C2 x3 = cadd(v[6], v[7]), x7 = csub(v[6], v[7]);
        v[0] = x0; v[1] = x1; v[2] = x2; v[3] = x3;
        v[4] = x4; v[5] = x5; v[6] = x6; v[7] = x7;
    }
};
template <>
struct PDft<16> {
    // n = 4 n1 + n2, k = k1 + 4 k2; natural-order output
    static __device__ __forceinline__ void run(C2 *v)
    {
        pdft4(v[0], v[4], v[8], v[12]);
        pdft4(v[1], v[5], v[9], v[13]);
        pdft4(v[2], v[6], v[10], v[14]);
        pdft4(v[3], v[7], v[11], v[15]);
        v[5] = cmuls(v[5], kP_C8, kP_S8);     // w16^1
        v[6] = mulw8_1(v[6]);                 // w16^2
        v[7] = cmuls(v[7], kP_S8, kP_C8);     // w16^3
        v[9] = mulw8_1(v[9]);                 // w16^2
        v[10] = roti(v[10]);                  // w16^4
        v[11] = mulw8_3(v[11]);               // w16^6
        v[13] = cmuls(v[13], kP_S8, kP_C8);   // w16^3
        v[14] = mulw8_3(v[14]);               // w16^6
        v[15] = cmuls(v[15], -kP_C8, -kP_S8); // w16^9
        pdft4(v[0], v[1], v[2], v[3]);
        pdft4(v[4], v[5], v[6], v[7]);
        pdft4(v[8], v[9], v[10], v[11]);
        pdft4(v[12], v[13], v[14], v[15]);
        C2 t;
        t = v[1]; v[1] = v[4]; v[4] = t;
        t = v[2]; v[2] = v[8]; v[8] = t;
        t = v[3]; v[3] = v[12]; v[12] = t;
        t = v[6]; v[6] = v[9]; v[9] = t;
        t = v[7]; v[7] = v[13]; v[13] = t;
        t = v[11]; v[11] = v[14]; v[14] = t;
    }
};

}  // namespace cdmt
