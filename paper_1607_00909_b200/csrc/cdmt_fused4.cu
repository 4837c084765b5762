// cdmt_fused4.cu -- k_fused_sp: the fused per-DM kernel (Alg. 1 l.99-103 + time integration,
// PAPER.md:117-123), software-pipelined over the DM trials.
//
// One CTA per (subband, block, channel), both polarisations in the two lanes of packed-FP32
// registers, M = 16 * 16 * R2, 16 packed points per thread, spectrum bins and last-pass twiddles
// in tensor memory.  The point of the kernel is WHEN the chirp of Eq. 1 is formed.  If every
// trial starts with the FP64 phase polynomial and the MUFU sin/cos of its 16 bins, all warps of
// a CTA do so at the same time (they leave the same block barrier), so the FP64/XU pipes and the
// FP32 pipe take turns instead of overlapping (round-1 ncu of that form: FMA pipe 65 % busy,
// removing the chirp arithmetic or the barrier gave 17 % / 11 %).  Here the block barrier
// between pass 1 and pass 2 is split
// into arrive / wait, and the chirp of trial d+1 is computed between the two -- in the
// barrier's shadow, while the data registers are dead -- and parked in tensor memory:
//
//   trial d   X (TMEM) times H_d (TMEM), pass 0 (radix 16 over j0), 16-byte stores
//             wait B(d-1): exchange buffer drained by every thread's pass-2 loads
//             pass 1 along j1 inside the half-warp (twiddles from a 2 KB shared table), in place
//             arrive A(d)
//             H_{d+1}: per-thread degree-5 phase polynomial in fp64, reduced mod 1 and converted
//             by ONE magic-number DADD (1.5 * 2^20: the low mantissa word is the fraction in
//             units of 2^-32 cycle), I2FP, MUFU sin/cos -> TMEM
//             wait A(d)
//             pass 2 loads, arrive B(d), radix R2 along j2, detection, Stokes I, integration
#include <cstdint>

#include "cdmt_fft2.cuh"
#include "cdmt_fused_common.cuh"
#include "cdmt_internal.h"
#include "cdmt_tmem.cuh"

namespace cdmt {

template <int M>
struct SP {
    static constexpr int NT = M / 16;      // threads: 16 packed points each
    static constexpr int R2 = M / 256;     // radix of the last pass (8, 16)
    static constexpr int U2 = 16 / R2;     // last-pass butterflies per thread
    static constexpr int NWARP = NT / 32;
    static constexpr int PITCH = 17;       // float4 per d1 row: conflict-free 16-byte accesses
    static constexpr int RHO = 16 * PITCH; // float4 per j2 plane
    static constexpr int EX = R2 * RHO;    // float4 in the exchange buffer (both polarisations)
    static constexpr int TW1_PITCH = 9;    // float4 per row of the pass-1 twiddle table (8 used)
    static constexpr int COLS_SLOT = 128;  // TMEM columns per warp slot
    static constexpr int TCOLS = COLS_SLOT * ((NWARP + 3) / 4);
    static constexpr int COL_X = 0, COL_H = 64, COL_TW2 = 96;
    static constexpr size_t smem_bytes =
        sizeof(float4) * (EX + 16 * TW1_PITCH) + sizeof(double) * 6 * NT + 2 * sizeof(uint64_t) + 16;
    static constexpr int CTAS_PER_SM = 512 / TCOLS;  // tensor memory and registers (128 x 512 threads)
};

__device__ __forceinline__ unsigned sp_f2u(float x) { return __float_as_uint(x); }
__device__ __forceinline__ float sp_u2f(unsigned x) { return __uint_as_float(x); }

__device__ __forceinline__ float4 sp_c2_to_f4(const C2 &v)
{
    float4 q;
    upk(v.re, q.x, q.y);
    upk(v.im, q.z, q.w);
    return q;
}
__device__ __forceinline__ C2 sp_f4_to_c2(const float4 &q) { return C2{pk(q.x, q.y), pk(q.z, q.w)}; }

// Chirp of one DM trial along this thread's 16 bins -> TMEM columns [tH, tH + 32) as (cos, sin).
// phi(r) = dm * sum_k c_k r^k cycles in fp64; adding 1.5 * 2^20 leaves round(phi * 2^32) mod 2^32
// in the low mantissa word: the fraction of a cycle as a signed 32-bit fixed-point number.
__device__ __forceinline__ void sp_chirp_to_tmem(const double *coef, int NT, int tid, double dm, uint32_t tH)
{
    const double q0 = dm * coef[0 * NT + tid], q1 = dm * coef[1 * NT + tid], q2 = dm * coef[2 * NT + tid];
    const double q3 = dm * coef[3 * NT + tid], q4 = dm * coef[4 * NT + tid], q5 = dm * coef[5 * NT + tid];
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        unsigned r[16];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const double rr = (double)(8 * half + i);
            const double phi = fma(fma(fma(fma(fma(q5, rr, q4), rr, q3), rr, q2), rr, q1), rr, q0);
            const int frac32 = __double2loint(phi + 1572864.0);
            const float x = __int2float_rn(frac32) * 1.4629180792671596e-9f;  // 2 pi / 2^32
            r[2 * i] = sp_f2u(__cosf(x));
            r[2 * i + 1] = sp_f2u(__sinf(x));
        }
        tmem_st16(tH + 16 * half, r);
    }
}

template <int M, int LOGD>
__global__ void __launch_bounds__(M / 16, SP<M>::CTAS_PER_SM)
k_fused_sp(const FusedArgs a, const __grid_constant__ DmParams dmp)
{
    using G = SP<M>;
    constexpr int NT = G::NT, R2 = G::R2, U2 = G::U2;
    constexpr int D = 1 << LOGD;
    constexpr int LS = LOGD < 4 ? LOGD : 4;  // reduce-scatter stages (16 values per thread)
    constexpr int NKEEP = 16 >> LS;          // integrated samples per thread per DM
    extern __shared__ float4 smem4[];
    float4 *ex = smem4;
    float4 *tw1s = smem4 + G::EX;                                         // [16][TW1_PITCH]
    double *coef = reinterpret_cast<double *>(tw1s + 16 * G::TW1_PITCH);  // [6][NT]
    uint64_t *barA = reinterpret_cast<uint64_t *>(coef + 6 * NT);         // pass-1 stores done
    uint64_t *barB = barA + 1;                                            // pass-2 loads done
    uint32_t *tslot = reinterpret_cast<uint32_t *>(barB + 1);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c = blockIdx.x % a.nchan;
    const int ulocal = blockIdx.x / a.nchan;
    const int unit = a.unit0 + ulocal, b = unit / a.nsub, s = unit % a.nsub;

    if (warp == 0) tmem_alloc<G::TCOLS>(tslot);
    if (tid == 0) {
        mbar_init(barA, NT);
        mbar_init(barB, NT);
    }
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tbase = *tslot;
    const uint32_t tcol = tbase + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(G::COLS_SLOT * (warp >> 2));

    const int j1 = tid & 15, j2 = tid >> 4;  // pass-0 role; pass 1: (j2, t0 = tid & 15)
    const int rest = j1 * R2 + j2;           // input bin m = j0 M/16 + rest
    {
        // this thread's 16 bins of both polarisations -> TMEM as (re_X, re_Y, im_X, im_Y)
        const float2 *src = a.spec + ((size_t)ulocal * 2) * a.nfft + (size_t)c * M + rest;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            unsigned r[16];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int j0 = 4 * q + i;
                const float2 gx = __ldg(src + j0 * (M / 16));
                const float2 gy = __ldg(src + a.nfft + j0 * (M / 16));
                r[4 * i + 0] = sp_f2u(gx.x);
                r[4 * i + 1] = sp_f2u(gy.x);
                r[4 * i + 2] = sp_f2u(gx.y);
                r[4 * i + 3] = sp_f2u(gy.y);
            }
            tmem_st16(tcol + G::COL_X + 16 * q, r);
        }
    }
    {
        // last-pass twiddles of this thread: w2[u][r] = exp(2 pi i r beta_u / M) -> TMEM
        unsigned r[32];
#pragma unroll
        for (int u = 0; u < U2; ++u)
#pragma unroll
            for (int rr = 0; rr < R2; ++rr) {
                float sn, cs;
                sincospif((float)(2 * rr * (tid + NT * u)) * (1.0f / (float)M), &sn, &cs);
                r[2 * (u * R2 + rr)] = sp_f2u(cs);
                r[2 * (u * R2 + rr) + 1] = sp_f2u(sn);
            }
        tmem_st32(tcol + G::COL_TW2, r);
    }
    // pass-1 twiddles w1[t0][r] = exp(2 pi i r t0 / 256), two per float4, one padded row per t0
    for (int e = tid; e < 128; e += NT) {
        const int t0 = e >> 3, i = e & 7;
        float s0, c0, s1, c1;
        sincospif((float)(2 * (2 * i) * t0) * (1.0f / 256.0f), &s0, &c0);
        sincospif((float)(2 * (2 * i + 1) * t0) * (1.0f / 256.0f), &s1, &c1);
        tw1s[t0 * G::TW1_PITCH + i] = make_float4(c0, s0, c1, s1);
    }
    // Eq. 1 along this thread's bins m_r = rest + r M/16: g(f_a + bb r) = sum_k c_k r^k, Taylor in
    // bb r / (f0 + f_a) <= 1e-3 (the host checks the r^6 term)
    {
        double f0, fb0, df;
        chirp_axes(a, s, c, M, &f0, &fb0, &df);
        const double kc = 1.0 / (2.41e-10 * f0 * f0), bb = (double)(M / 16) * df;
        const double fa = fb0 + (double)rest * df;
        const double sa = f0 + fa, ee = bb / sa, pp = kc * f0 * f0 / sa;
        const double c2 = pp * ee * ee, c3 = -c2 * ee, c4 = -c3 * ee, c5 = -c4 * ee;
        coef[0 * NT + tid] = kc * fa * fa / sa;
        coef[1 * NT + tid] = kc * (fa * fa + 2.0 * fa * f0) / (sa * sa) * bb;
        coef[2 * NT + tid] = c2;
        coef[3 * NT + tid] = c3;
        coef[4 * NT + tid] = c4;
        coef[5 * NT + tid] = c5;
    }
    const int nchan_total = a.nsub * a.nchan;
    const int ochan = nchan_total - 1 - (s * a.nchan + c);
    float *out0 = a.out + (size_t)b * a.vdec * a.out_pitch + ochan;
    const int d_begin = a.dm_first + blockIdx.y * a.dm_tile;
    const int d_end = min(a.ndm, d_begin + a.dm_tile);
    float4 *const p0 = ex + j2 * G::RHO + j1 * G::PITCH;   // pass-0 stores: [t0]
    float4 *const p1 = ex + j2 * G::RHO + (tid & 15);      // pass-1 loads/stores: [d1 * PITCH]
    const float4 *const pw1 = tw1s + (tid & 15) * G::TW1_PITCH;
    if (d_begin < d_end) sp_chirp_to_tmem(coef, NT, tid, dmp.dm[d_begin - a.dm_param0], tcol + G::COL_H);
    __syncthreads();

#pragma unroll 1
    for (int d = d_begin; d < d_end; ++d) {
        const unsigned par = (unsigned)(d - d_begin) & 1u;
        C2 v[16];
        // ---- the thread's 16 bins times the chirp of this trial, both polarisations at once
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            unsigned hr[16];
            tmem_ld16(hr, tcol + G::COL_H + 16 * hh);
#pragma unroll
            for (int qq = 0; qq < 2; ++qq) {
                unsigned xr[16];
                tmem_ld16(xr, tcol + G::COL_X + 16 * (2 * hh + qq));
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int r = 8 * hh + 4 * qq + i;
                    const C2 x = C2{pk(sp_u2f(xr[4 * i]), sp_u2f(xr[4 * i + 1])),
                                    pk(sp_u2f(xr[4 * i + 2]), sp_u2f(xr[4 * i + 3]))};
                    v[r] = cmuls(x, sp_u2f(hr[2 * (4 * qq + i)]), sp_u2f(hr[2 * (4 * qq + i) + 1]));
                }
            }
        }
        // ---- pass 0 (the exchange buffer is free once every thread has loaded its pass-2 inputs
        //      of the previous trial)
        PDft<16>::run(v);
        if (d != d_begin) mbar_wait(barB, par ^ 1u);
#pragma unroll
        for (int t0 = 0; t0 < 16; ++t0) p0[t0] = sp_c2_to_f4(v[t0]);
        __syncwarp();
        // ---- pass 1: along j1, in place
        {
#pragma unroll
            for (int d1 = 0; d1 < 16; ++d1) v[d1] = sp_f4_to_c2(p1[d1 * G::PITCH]);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float4 w = pw1[i];
                if (i) v[2 * i] = cmuls(v[2 * i], w.x, w.y);
                v[2 * i + 1] = cmuls(v[2 * i + 1], w.z, w.w);
            }
            PDft<16>::run(v);
#pragma unroll
            for (int t1 = 0; t1 < 16; ++t1) p1[t1 * G::PITCH] = sp_c2_to_f4(v[t1]);
        }
        mbar_arrive(barA);
        // ---- chirp of the next trial in the barrier's shadow (the data registers are dead here)
        if (d + 1 < d_end) sp_chirp_to_tmem(coef, NT, tid, dmp.dm[d + 1 - a.dm_param0], tcol + G::COL_H);
        mbar_wait(barA, par);
        // ---- pass 2 along j2, detection, polarisation sum
        float pw[16];  // |y_X[t]|^2 + |y_Y[t]|^2, t = tid + NT n
        {
#pragma unroll
            for (int u = 0; u < U2; ++u) {
                const int beta = tid + NT * u;
                const float4 *p = ex + (beta >> 4) * G::PITCH + (beta & 15);
#pragma unroll
                for (int rr = 0; rr < R2; ++rr) v[u * R2 + rr] = sp_f4_to_c2(p[rr * G::RHO]);
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                unsigned w2[16];
                tmem_ld16(w2, tcol + G::COL_TW2 + 16 * h);
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int k = 8 * h + i;
                    if (k % R2) v[k] = cmuls(v[k], sp_u2f(w2[2 * i]), sp_u2f(w2[2 * i + 1]));
                }
            }
            mbar_arrive(barB);  // every load of this trial has been consumed
#pragma unroll
            for (int u = 0; u < U2; ++u) PDft<R2>::run(v + u * R2);
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const int n = (k / R2) + U2 * (k % R2);
                const P2 p = fma2(v[k].im, v[k].im, mul2(v[k].re, v[k].re));
                float px, py;
                upk(p, px, py);
                pw[n] = px + py;
            }
        }
        // ---- time integration over D adjacent samples = D adjacent lanes
        lane_reduce_scatter<LS>(pw, lane);
        if constexpr (LOGD > LS) pw[0] += __shfl_xor_sync(0xffffffffu, pw[0], 16);
        float *outd = out0 + (size_t)d * (size_t)a.out_stride_dm;
#pragma unroll
        for (int j = 0; j < NKEEP; ++j) {
            const int n = (lane & ((1 << LS) - 1)) + (1 << LS) * j;
            const int t0 = (tid & ~(D - 1)) + NT * n;  // first sample of the integrated group
            if ((lane & (D - 1)) < (1 << LS) && t0 >= a.hdisc && t0 < M - a.hdisc)
                outd[(size_t)((t0 - a.hdisc) >> LOGD) * a.out_pitch] = pw[j] * a.scale;
        }
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc<G::TCOLS>(tbase);
}

// ------------------------------------------------------------------------------------
// launch
// ------------------------------------------------------------------------------------
template <int M, int LOGD>
static cudaError_t launch_sp_MD(FusedArgs fa, const double *h_dm, int nunits, cudaStream_t st, long long *launches)
{
    using G = SP<M>;
    // resident CTAs x TMEM columns must stay <= 512: cap the occupancy through the shared-memory request
    size_t smem = G::smem_bytes;
    const size_t floor_bytes = (size_t)(233472 / (G::CTAS_PER_SM + 1)) - 1024 + 16;
    if (smem < floor_bytes) smem = floor_bytes;
    cudaError_t e = cudaFuncSetAttribute(k_fused_sp<M, LOGD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int ndm_total = fa.ndm;
    for (int d0 = 0; d0 < ndm_total; d0 += DM_PARAM_MAX) {
        const int cnt = ndm_total - d0 < DM_PARAM_MAX ? ndm_total - d0 : DM_PARAM_MAX;
        DmParams dmp;
        for (int i = 0; i < cnt; ++i) dmp.dm[i] = h_dm[d0 + i];
        for (int i = cnt; i < DM_PARAM_MAX; ++i) dmp.dm[i] = 0.0;
        fa.dm_first = d0;
        fa.dm_param0 = d0;
        fa.ndm = d0 + cnt;
        dim3 grid((unsigned)(nunits * fa.nchan), (unsigned)((cnt + fa.dm_tile - 1) / fa.dm_tile));
        k_fused_sp<M, LOGD><<<grid, M / 16, smem, st>>>(fa, dmp);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        ++*launches;
    }
    return cudaSuccess;
}

template <int M>
static cudaError_t launch_sp_M(int logd, const FusedArgs &fa, const double *h_dm, int nunits, cudaStream_t st,
                               long long *launches)
{
    switch (logd) {
    case 0: return launch_sp_MD<M, 0>(fa, h_dm, nunits, st, launches);
    case 1: return launch_sp_MD<M, 1>(fa, h_dm, nunits, st, launches);
    case 2: return launch_sp_MD<M, 2>(fa, h_dm, nunits, st, launches);
    case 3: return launch_sp_MD<M, 3>(fa, h_dm, nunits, st, launches);
    case 4: return launch_sp_MD<M, 4>(fa, h_dm, nunits, st, launches);
    case 5: return launch_sp_MD<M, 5>(fa, h_dm, nunits, st, launches);
    default: return cudaErrorInvalidValue;
    }
}

bool fused_sp_supported(int M, int ndec, int hdisc)
{
    if (M != 2048 && M != 4096) return false;
    if (ndec > 32 || (ndec & (ndec - 1)) != 0) return false;
    return hdisc % ndec == 0;
}

cudaError_t launch_fused_sp(int M, int logd, const FusedArgs &fa, const double *h_dm, int nunits, cudaStream_t st,
                            long long *launches)
{
    switch (M) {
    case 2048: return launch_sp_M<2048>(logd, fa, h_dm, nunits, st, launches);
    case 4096: return launch_sp_M<4096>(logd, fa, h_dm, nunits, st, launches);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace cdmt
