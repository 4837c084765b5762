// cdmt_fft.cuh -- register/shared-memory Stockham FFT building blocks (sm_100a).
//
// Every thread owns 16 complex points per pass: one radix-16 butterfly, or 16/R butterflies
// of radix R for the remainder pass.  A length-L transform is the radix sequence
// 16,16,..,rest (L = 16^a * rest, rest in {1,2,4,8}); passes exchange data through shared
// memory in natural (autosort) order, so the last pass leaves X[j + q L/R] in registers.
//
// Transform computed: X[k] = sum_n x[n] exp(SIGN 2 pi i k n / L)   (SIGN=-1: PAPER.md:115
// forward FFT; SIGN=+1: PAPER.md:119 backward FFT), unnormalised.
#pragma once
#include <cuda_runtime.h>

namespace cdmt {

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// multiply by exp(SIGN i pi/2) = SIGN * i
template <int SIGN>
__device__ __forceinline__ float2 rot90(float2 a)
{
    return SIGN > 0 ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}
// multiply by cos + SIGN i sin with compile-time cos, sin
template <int SIGN>
__device__ __forceinline__ float2 cmulc(float2 a, float c, float s)
{
    const float ss = SIGN > 0 ? s : -s;
    return make_float2(a.x * c - a.y * ss, a.x * ss + a.y * c);
}

constexpr float kR2 = 0.70710678118654752440f;  // cos(pi/4)
constexpr float kC8 = 0.92387953251128675613f;  // cos(pi/8)
constexpr float kS8 = 0.38268343236508977173f;  // sin(pi/8)

template <int SIGN>
__device__ __forceinline__ void dft2(float2 &a, float2 &b)
{
    float2 t = a;
    a = cadd(t, b);
    b = csub(t, b);
}

template <int SIGN>
__device__ __forceinline__ void dft4(float2 &v0, float2 &v1, float2 &v2, float2 &v3)
{
    float2 a = cadd(v0, v2), b = csub(v0, v2);
    float2 c = cadd(v1, v3), d = rot90<SIGN>(csub(v1, v3));
    v0 = cadd(a, c);
    v1 = cadd(b, d);
    v2 = csub(a, c);
    v3 = csub(b, d);
}

// multiply by exp(SIGN 2 pi i e / 8), e = 1, 3 (e = 2 is rot90)
template <int SIGN>
__device__ __forceinline__ float2 mulw8_1(float2 a)
{
    return SIGN > 0 ? make_float2((a.x - a.y) * kR2, (a.x + a.y) * kR2)
                    : make_float2((a.x + a.y) * kR2, (a.y - a.x) * kR2);
}
template <int SIGN>
__device__ __forceinline__ float2 mulw8_3(float2 a)
{
    return SIGN > 0 ? make_float2((-a.x - a.y) * kR2, (a.x - a.y) * kR2)
                    : make_float2((a.y - a.x) * kR2, (-a.x - a.y) * kR2);
}

template <int R, int SIGN>
struct Dft;

template <int SIGN>
struct Dft<2, SIGN> {
    static __device__ __forceinline__ void run(float2 *v) { dft2<SIGN>(v[0], v[1]); }
};

template <int SIGN>
struct Dft<4, SIGN> {
    static __device__ __forceinline__ void run(float2 *v) { dft4<SIGN>(v[0], v[1], v[2], v[3]); }
};

template <int SIGN>
struct Dft<8, SIGN> {
    // n = 2 n1 + n2, k = k1 + 4 k2
    static __device__ __forceinline__ void run(float2 *v)
    {
        dft4<SIGN>(v[0], v[2], v[4], v[6]);  // A[k1][0]
        dft4<SIGN>(v[1], v[3], v[5], v[7]);  // A[k1][1]
        v[3] = mulw8_1<SIGN>(v[3]);
        v[5] = rot90<SIGN>(v[5]);
        v[7] = mulw8_3<SIGN>(v[7]);
        float2 x0 = cadd(v[0], v[1]), x4 = csub(v[0], v[1]);
        float2 x1 = cadd(v[2], v[3]), x5 = csub(v[2], v[3]);
        float2 x2 = cadd(v[4], v[5]), x6 = csub(v[4], v[5]);
        float2 x3 = cadd(v[6], v[7]), x7 = csub(v[6], v[7]);
        v[0] = x0; v[1] = x1; v[2] = x2; v[3] = x3;
        v[4] = x4; v[5] = x5; v[6] = x6; v[7] = x7;
    }
};

template <int SIGN>
struct Dft<16, SIGN> {
    // n = 4 n1 + n2, k = k1 + 4 k2; A[k1][n2] is left in v[4 k1 + n2]
    static __device__ __forceinline__ void run(float2 *v)
    {
        dft4<SIGN>(v[0], v[4], v[8], v[12]);
        dft4<SIGN>(v[1], v[5], v[9], v[13]);
        dft4<SIGN>(v[2], v[6], v[10], v[14]);
        dft4<SIGN>(v[3], v[7], v[11], v[15]);
        // twiddles w16^(n2 k1)
        v[5] = cmulc<SIGN>(v[5], kC8, kS8);    // e = 1
        v[6] = mulw8_1<SIGN>(v[6]);            // e = 2
        v[7] = cmulc<SIGN>(v[7], kS8, kC8);    // e = 3
        v[9] = mulw8_1<SIGN>(v[9]);            // e = 2
        v[10] = rot90<SIGN>(v[10]);            // e = 4
        v[11] = mulw8_3<SIGN>(v[11]);          // e = 6
        v[13] = cmulc<SIGN>(v[13], kS8, kC8);  // e = 3
        v[14] = mulw8_3<SIGN>(v[14]);          // e = 6
        v[15] = cmulc<SIGN>(v[15], -kC8, -kS8);  // e = 9
        dft4<SIGN>(v[0], v[1], v[2], v[3]);      // k1 = 0 -> X[0,4,8,12]
        dft4<SIGN>(v[4], v[5], v[6], v[7]);      // k1 = 1 -> X[1,5,9,13]
        dft4<SIGN>(v[8], v[9], v[10], v[11]);    // k1 = 2
        dft4<SIGN>(v[12], v[13], v[14], v[15]);  // k1 = 3
        // v[4 k1 + k2] = X[k1 + 4 k2] -> transpose to natural order
        float2 t;
        t = v[1]; v[1] = v[4]; v[4] = t;
        t = v[2]; v[2] = v[8]; v[8] = t;
        t = v[3]; v[3] = v[12]; v[12] = t;
        t = v[6]; v[6] = v[9]; v[9] = t;
        t = v[7]; v[7] = v[13]; v[13] = t;
        t = v[11]; v[11] = v[14]; v[14] = t;
    }
};

// ---- radix plan: L = 16^a * rest -------------------------------------------------------
template <int L>
struct RadixPlan {
    static_assert(L >= 16 && (L & (L - 1)) == 0, "L must be a power of two >= 16");
    static constexpr int log2L()
    {
        int n = 0;
        for (int l = L; l > 1; l >>= 1) ++n;
        return n;
    }
    static constexpr int n16 = log2L() / 4;
    static constexpr int rest = 1 << (log2L() % 4);
    static constexpr int npass = n16 + (rest > 1 ? 1 : 0);
    static constexpr int radix(int p) { return p < n16 ? 16 : rest; }
    static constexpr int ns(int p)
    {
        int n = 1;
        for (int q = 0; q < p; ++q) n *= radix(q);
        return n;
    }
    // twiddle table: pass p >= 1 stores (R-1) * NS entries tw[(r-1) NS + k] = exp(SIGN 2 pi i k r/(NS R))
    static constexpr int tw_offset(int p)
    {
        int o = 0;
        for (int q = 1; q < p; ++q) o += (radix(q) - 1) * ns(q);
        return o;
    }
    static constexpr int tw_size = tw_offset(npass);
    static constexpr int last_radix = radix(npass - 1);
    static constexpr int last_ns = ns(npass - 1);
};

// Shared-memory addressing. Batched tiles: [elem][batch] with a padded pitch. Single
// transform: one pad element per 16 so that the stride-16 stores of pass 0 hit 16 banks.
template <int BATCH>
struct SmemAddr {
    static constexpr int PITCH = BATCH + 1;
    static __device__ __forceinline__ int at(int elem, int batch) { return elem * PITCH + batch; }
    static constexpr int size(int L) { return L * PITCH; }
};
template <>
struct SmemAddr<1> {
    static __device__ __forceinline__ int at(int elem, int) { return elem + (elem >> 4); }
    static constexpr int size(int L) { return L + (L >> 4); }
};

// One pass, 16 points per thread.
template <int L, int P, int SIGN, int NT, int BATCH>
struct Pass {
    using Plan = RadixPlan<L>;
    using Addr = SmemAddr<BATCH>;
    static constexpr int R = Plan::radix(P);
    static constexpr int NS = Plan::ns(P);
    static constexpr int U = 16 / R;
    static constexpr int TWOFF = Plan::tw_offset(P);
    static_assert(NT * 16 == L * BATCH, "16 points per thread");

    static __device__ __forceinline__ void load(const float2 *s, float2 *v, int tid)
    {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = tid + u * NT, b = i % BATCH, j = i / BATCH;
#pragma unroll
            for (int r = 0; r < R; ++r) v[u * R + r] = s[Addr::at(j + r * (L / R), b)];
        }
    }
    static __device__ __forceinline__ void compute(float2 *v, const float2 *__restrict__ tw, int tid)
    {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (NS > 1) {
                const int i = tid + u * NT, j = i / BATCH, k = j % NS;
                const float2 *t = tw + TWOFF + k;
#pragma unroll
                for (int r = 1; r < R; ++r) v[u * R + r] = cmul(v[u * R + r], __ldg(t + (r - 1) * NS));
            }
            Dft<R, SIGN>::run(v + u * R);
        }
    }
    static __device__ __forceinline__ void store(float2 *s, const float2 *v, int tid)
    {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = tid + u * NT, b = i % BATCH, j = i / BATCH, k = j % NS;
            const int e0 = (j / NS) * (NS * R) + k;
#pragma unroll
            for (int q = 0; q < R; ++q) s[Addr::at(e0 + q * NS, b)] = v[u * R + q];
        }
    }
    // element index (within the transform) of output q of butterfly slot u after this pass
    static __device__ __forceinline__ int out_elem(int tid, int u, int q)
    {
        const int i = tid + u * NT, j = i / BATCH, k = j % NS;
        return (j / NS) * (NS * R) + k + q * NS;
    }
    static __device__ __forceinline__ int in_elem(int tid, int u, int r)
    {
        const int i = tid + u * NT, j = i / BATCH;
        return j + r * (L / R);
    }
    static __device__ __forceinline__ int batch_of(int tid, int u) { return (tid + u * NT) % BATCH; }
};

// Passes P..npass-1.  On entry v holds the inputs of pass P (when FROM_REGS) or the data are
// in shared memory and visible (caller synchronised).  On exit v holds the outputs of the
// last pass (see Pass::out_elem of the last pass); shared memory may still be read by
// other threads: synchronise before overwriting it.
template <int L, int P, int SIGN, int NT, int BATCH, bool FROM_REGS>
__device__ __forceinline__ void fft_passes(float2 *v, float2 *s, const float2 *__restrict__ tw, int tid)
{
    using Plan = RadixPlan<L>;
    using Ps = Pass<L, P, SIGN, NT, BATCH>;
    if constexpr (!FROM_REGS) Ps::load(s, v, tid);
    Ps::compute(v, tw, tid);
    if constexpr (P + 1 < Plan::npass) {
        if constexpr (!FROM_REGS) __syncthreads();  // everyone has read this pass's inputs
        Ps::store(s, v, tid);
        __syncthreads();
        fft_passes<L, P + 1, SIGN, NT, BATCH, false>(v, s, tw, tid);
    }
}

}  // namespace cdmt
