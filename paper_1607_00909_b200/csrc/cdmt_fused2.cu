// cdmt_fused2.cu -- k_fused_x2: the fused per-DM kernel (Alg. 1 l.99-103 + time integration,
// PAPER.md:117-123) on Blackwell's packed-FP32 pipe, with tensor memory as per-thread scratch.
//
// One CTA per (subband, block, channel) loops over a tile of DM trials.  The length-M backward
// FFT of a channel is split by decimation in time into the transforms of its even and its odd
// bins (length L = M/2 = 16 * 16 * R2); the two ride in the two lanes of f32x2 registers, so
// every butterfly and twiddle is one FADD2/FMUL2/FFMA2 for both:
//
//   y[t]     = A[t] + w_M^t B[t],   A = FFT_L(Z[2j]),  B = FFT_L(Z[2j+1]),  Z = X * chirp
//   y[t + L] = A[t] - w_M^t B[t]
//
//   pass 0   thread (j2, j1): its 16 bins X of both polarisations come from TMEM (tcgen05.ld,
//            one instruction per polarisation), times the chirp of this DM trial (Eq. 1, phase
//            from a per-thread degree-5 polynomial in fp64, reduced mod 1, MUFU sin/cos),
//            radix-16 butterfly, 16-byte stores into the exchange buffer of that polarisation
//   pass 1   the same half-warp re-reads along j1 (only __syncwarp), twiddle, radix 16, in place
//   pass 2   after the one block barrier per DM trial: radix R2 along j2, then the radix-2
//            combine above, square-law detection and the sum over the two polarisations
//   integrate  the 32 powers per thread (times t = tid + NT n [+ L]) are exchanged through a
//            per-warp shared-memory tile so that one lane sums the ndec adjacent samples
//            (PAPER.md:123 + north_star), scaled by 1/(N M) and stored time-major.
//
// Everything a thread re-reads for every DM trial lives in TMEM (its lane, 256 columns):
// X of both polarisations (128 words) and its pass-1 / pass-2 / combine twiddles; shared
// memory carries only the exchanges, so its bandwidth is spent on the transposes alone.
#include <cstdint>

#include "cdmt_fft2.cuh"
#include "cdmt_fused_common.cuh"
#include "cdmt_internal.h"
#include "cdmt_tmem.cuh"

namespace cdmt {

template <int M>
struct X2 {
    static constexpr int L = M / 2;        // length of the two half transforms
    static constexpr int NT = L / 16;      // threads: 16 packed points each
    static constexpr int R2 = L / 256;     // radix of the last pass (4, 8, 16)
    static constexpr int U2 = 16 / R2;     // last-pass butterflies per thread
    static constexpr int NWARP = NT / 32;
    static constexpr int PITCH = 17;       // float4 per d1 row: conflict-free 16-byte accesses
    static constexpr int RHO = 16 * PITCH; // float4 per j2 plane
    static constexpr int EX = R2 * RHO;    // float4 per exchange buffer (one per polarisation)
    static constexpr int IROW = 34;        // float2 per integration row: 32 lanes + 16 bytes
    static constexpr int INTEG = 16 * IROW;
    static constexpr int COLS_SLOT = 256;  // TMEM columns per warp slot
    static constexpr int TCOLS = COLS_SLOT * ((NWARP + 3) / 4);
    static constexpr int COL_X = 0, COL_TW1 = 128, COL_TW2 = 160, COL_TWF = 192;
    static constexpr size_t smem_bytes =
        sizeof(float4) * 2 * EX + sizeof(float2) * NWARP * INTEG + sizeof(double) * 12 * NT + 32;
    static constexpr int CTAS_PER_SM = 512 / TCOLS;  // bounded by tensor memory
};

__device__ __forceinline__ unsigned f2u(float x) { return __float_as_uint(x); }
__device__ __forceinline__ float u2f(unsigned x) { return __uint_as_float(x); }
__device__ __forceinline__ P2 pku(unsigned lo, unsigned hi) { return pk(u2f(lo), u2f(hi)); }
__device__ __forceinline__ P2 lo2(P2 v) { return bc(lo_of(v)); }  // (lo, lo): folds into an .F32 operand
__device__ __forceinline__ P2 hi2(P2 v) { return bc(hi_of(v)); }

__device__ __forceinline__ float4 c2_to_f4(const C2 &v)
{
    float4 q;
    upk(v.re, q.x, q.y);
    upk(v.im, q.z, q.w);
    return q;
}
__device__ __forceinline__ C2 f4_to_c2(const float4 &q) { return C2{pk(q.x, q.y), pk(q.z, q.w)}; }

// unit phasor of a phase in cycles (|phi| < 2^19, checked on the host): adding 1.5 * 2^20 leaves
// round(phi * 2^32) mod 2^32 in the low mantissa word -- the fraction of a cycle as a signed
// fixed-point number -- so one DADD reduces mod 1 and converts; I2FP, then MUFU sin/cos
__device__ __forceinline__ float2 phasor_of(double phi)
{
    const int frac32 = __double2loint(phi + 1572864.0);
    const float x = __int2float_rn(frac32) * 1.4629180792671596e-9f;  // 2 pi / 2^32
    return make_float2(__cosf(x), __sinf(x));
}

// Chirp of one DM trial on the thread's 16 x 2 bins (even bins in the low lane, odd in the high)
template <int NT>
__device__ __forceinline__ void x2_chirp(const double *coef, int tid, double dm, P2 (&Hr)[16], P2 (&Hi)[16])
{
    double pe[6], po[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        pe[k] = dm * coef[(size_t)k * NT + tid];
        po[k] = dm * coef[(size_t)(6 + k) * NT + tid];
    }
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const double rr = (double)r;
        const double phe = fma(fma(fma(fma(fma(pe[5], rr, pe[4]), rr, pe[3]), rr, pe[2]), rr, pe[1]), rr, pe[0]);
        const double pho = fma(fma(fma(fma(fma(po[5], rr, po[4]), rr, po[3]), rr, po[2]), rr, po[1]), rr, po[0]);
        const float2 he = phasor_of(phe), ho = phasor_of(pho);
        Hr[r] = pk(he.x, ho.x);
        Hi[r] = pk(he.y, ho.y);
    }
}

template <int M, int LOGD>
__global__ void __launch_bounds__(M / 32, X2<M>::CTAS_PER_SM)
k_fused_x2(const FusedArgs a, const __grid_constant__ DmParams dmp)
{
    using G = X2<M>;
    constexpr int L = G::L, NT = G::NT, R2 = G::R2, U2 = G::U2;
    constexpr int D = 1 << LOGD;
    constexpr int DG = D > 16 ? 16 : D;  // lanes summed through the shared-memory tile
    static_assert(LOGD >= 3 && LOGD <= 5, "ndec 8, 16 or 32");
    extern __shared__ float4 smem4[];
    float4 *ex0 = smem4, *ex1 = smem4 + G::EX;
    float2 *integ = reinterpret_cast<float2 *>(smem4 + 2 * G::EX);
    double *coef = reinterpret_cast<double *>(integ + G::NWARP * G::INTEG);  // [2][6][NT]
    uint64_t *bar = reinterpret_cast<uint64_t *>(coef + 12 * NT);  // pass-2 loads done (buffers free)
    uint64_t *barA = bar + 1;                                      // pass-1 stores done
    uint32_t *tslot = reinterpret_cast<uint32_t *>(barA + 1);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int bx = (int)blockIdx.x + a.cta0;
    const int c = bx % a.nchan;
    const int ulocal = bx / a.nchan;
    const int unit = a.unit0 + ulocal, b = unit / a.nsub, s = unit % a.nsub;

    if (warp == 0) tmem_alloc<G::TCOLS>(tslot);
    if (tid == 0) {
        mbar_init(bar, NT);
        mbar_init(barA, NT);
    }
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tbase = *tslot;
    const uint32_t tcol = tbase + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(G::COLS_SLOT * (warp >> 2));

    const int j1 = tid & 15, j2 = tid >> 4;  // pass-0 role; pass 1: (j2, t0 = tid & 15)
    const int rest = j1 * R2 + j2;           // half-transform input index j = j0 L/16 + rest
    {
        // this thread's bins 2j, 2j+1 of both polarisations -> TMEM as (re_e, re_o, im_e, im_o)
        const float4 *src = reinterpret_cast<const float4 *>(a.spec + ((size_t)ulocal * 2) * a.nfft + (size_t)c * M);
#pragma unroll
        for (int pol = 0; pol < 2; ++pol) {
            unsigned r[64];
#pragma unroll
            for (int j0 = 0; j0 < 16; ++j0) {
                const float4 g = __ldg(src + (size_t)pol * (a.nfft / 2) + j0 * (L / 16) + rest);
                r[4 * j0 + 0] = f2u(g.x);
                r[4 * j0 + 1] = f2u(g.z);
                r[4 * j0 + 2] = f2u(g.y);
                r[4 * j0 + 3] = f2u(g.w);
            }
            tmem_st64(tcol + G::COL_X + 64 * pol, r);
        }
    }
    {
        // pass twiddles of this thread: w1[r] = exp(2 pi i r t0 / 256), w2[u][r] = exp(2 pi i r beta_u / L)
        unsigned r[32];
#pragma unroll
        for (int rr = 0; rr < 16; ++rr) {
            float sn, cs;
            sincospif((float)(2 * rr * (tid & 15)) * (1.0f / 256.0f), &sn, &cs);
            r[2 * rr] = f2u(cs);
            r[2 * rr + 1] = f2u(sn);
        }
        tmem_st32(tcol + G::COL_TW1, r);
#pragma unroll
        for (int u = 0; u < U2; ++u)
#pragma unroll
            for (int rr = 0; rr < R2; ++rr) {
                float sn, cs;
                sincospif((float)(2 * rr * (tid + NT * u)) * (1.0f / (float)L), &sn, &cs);
                r[2 * (u * R2 + rr)] = f2u(cs);
                r[2 * (u * R2 + rr) + 1] = f2u(sn);
            }
        tmem_st32(tcol + G::COL_TW2, r);
        // combine twiddles in the order the last pass leaves its outputs: k = u R2 + t2 holds
        // t' = tid + NT n, n = u + U2 t2, as the pairs (wr, -wr), (wi, -wi) of w_M^t'
        unsigned f[64];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const int n = (k / R2) + U2 * (k % R2);
            float sn, cs;
            sincospif((float)(2 * (tid + NT * n)) * (1.0f / (float)M), &sn, &cs);
            f[4 * k + 0] = f2u(cs);
            f[4 * k + 1] = f2u(-cs);
            f[4 * k + 2] = f2u(sn);
            f[4 * k + 3] = f2u(-sn);
        }
        tmem_st64(tcol + G::COL_TWF, f);
    }
    // Eq. 1 along this thread's bins m = 2 rest + e + r M/16 (e = 0 even lane, 1 odd lane):
    // g(f_a + bb r) = sum_k c_k r^k, Taylor in bb r / (f0 + f_a) <= 1e-3 (host checks the r^6 term)
    {
        double f0, fb0, df;
        chirp_axes(a, s, c, M, &f0, &fb0, &df);
        const double kc = 1.0 / (2.41e-10 * f0 * f0), bb = (double)(M / 16) * df;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const double fa = fb0 + (double)(2 * rest + e) * df;
            const double sa = f0 + fa, ee = bb / sa, pp = kc * f0 * f0 / sa;
            const double c2 = pp * ee * ee, c3 = -c2 * ee, c4 = -c3 * ee, c5 = -c4 * ee;
            double *ce = coef + (size_t)e * 6 * NT + tid;
            ce[0 * NT] = kc * fa * fa / sa;
            ce[1 * NT] = kc * (fa * fa + 2.0 * fa * f0) / (sa * sa) * bb;
            ce[2 * NT] = c2;
            ce[3 * NT] = c3;
            ce[4 * NT] = c4;
            ce[5 * NT] = c5;
        }
    }
    const int nchan_total = a.nsub * a.nchan;
    const int ochan = nchan_total - 1 - (s * a.nchan + c);
    float *out0 = a.out + (size_t)b * a.vdec * a.out_pitch + ochan;
    const int d_begin = a.dm_first + blockIdx.y * a.dm_tile;
    const int d_end = min(a.ndm, d_begin + a.dm_tile);
    float2 *ib = integ + warp * G::INTEG;
    __syncthreads();
    // the chirp of trial d+1 is formed in the shadow of the block barrier of trial d and stays in
    // registers (the data registers are dead there); the first one is formed here
    P2 Hr[16], Hi[16];
    if (d_begin < d_end) x2_chirp<NT>(coef, tid, dmp.dm[d_begin - a.dm_param0], Hr, Hi);

#pragma unroll 1
    for (int d = d_begin; d < d_end; ++d) {
        const unsigned par = (unsigned)(d - d_begin) & 1u;
        // ---- pass 0: both polarisations (the exchange buffers are free once every thread has
        //      finished the last pass of the previous trial)
        if (d != d_begin) mbar_wait(bar, par ^ 1u);
#pragma unroll
        for (int pol = 0; pol < 2; ++pol) {
            unsigned xr[64];
            tmem_ld64(xr, tcol + G::COL_X + 64 * pol);
            C2 v[16];
#pragma unroll
            for (int r = 0; r < 16; ++r)
                v[r] = cmulp(C2{pku(xr[4 * r], xr[4 * r + 1]), pku(xr[4 * r + 2], xr[4 * r + 3])}, Hr[r], Hi[r]);
            PDft<16>::run(v);
            float4 *dst = (pol ? ex1 : ex0) + j2 * G::RHO + j1 * G::PITCH;
#pragma unroll
            for (int t0 = 0; t0 < 16; ++t0) dst[t0] = c2_to_f4(v[t0]);
        }
        __syncwarp();
        // ---- pass 1: along j1, in place
        {
            unsigned w1[32];
            tmem_ld32(w1, tcol + G::COL_TW1);
#pragma unroll
            for (int pol = 0; pol < 2; ++pol) {
                float4 *p = (pol ? ex1 : ex0) + j2 * G::RHO + (tid & 15);
                C2 v[16];
#pragma unroll
                for (int d1 = 0; d1 < 16; ++d1) v[d1] = f4_to_c2(p[d1 * G::PITCH]);
#pragma unroll
                for (int d1 = 1; d1 < 16; ++d1) v[d1] = cmuls(v[d1], u2f(w1[2 * d1]), u2f(w1[2 * d1 + 1]));
                PDft<16>::run(v);
#pragma unroll
                for (int t1 = 0; t1 < 16; ++t1) p[t1 * G::PITCH] = c2_to_f4(v[t1]);
            }
        }
        mbar_arrive(barA);
        if (d + 1 < d_end) x2_chirp<NT>(coef, tid, dmp.dm[d + 1 - a.dm_param0], Hr, Hi);
        mbar_wait(barA, par);
        // ---- pass 2 along j2, radix-2 combine, detection, polarisation sum
        P2 pw[16];  // (|y[t']|^2, |y[t' + L]|^2) summed over polarisations, order k = u R2 + t2
        {
            unsigned w2[32];
            tmem_ld32(w2, tcol + G::COL_TW2);
#pragma unroll
            for (int pol = 0; pol < 2; ++pol) {
                const float4 *ex = pol ? ex1 : ex0;
                C2 v[16];
#pragma unroll
                for (int u = 0; u < U2; ++u) {
                    const int beta = tid + NT * u;
                    const float4 *p = ex + (beta >> 4) * G::PITCH + (beta & 15);
#pragma unroll
                    for (int rr = 0; rr < R2; ++rr) v[u * R2 + rr] = f4_to_c2(p[rr * G::RHO]);
                }
#pragma unroll
                for (int u = 0; u < U2; ++u) {
#pragma unroll
                    for (int rr = 1; rr < R2; ++rr)
                        v[u * R2 + rr] = cmuls(v[u * R2 + rr], u2f(w2[2 * (u * R2 + rr)]), u2f(w2[2 * (u * R2 + rr) + 1]));
                }
                if (pol == 1) mbar_arrive(bar);  // every load of this trial has been consumed
#pragma unroll
                for (int u = 0; u < U2; ++u) PDft<R2>::run(v + u * R2);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    unsigned wf[32];
                    tmem_ld32(wf, tcol + G::COL_TWF + 32 * h);
#pragma unroll
                    for (int kk = 0; kk < 8; ++kk) {
                        const int k = 8 * h + kk;
                        const P2 Wr = pku(wf[4 * kk], wf[4 * kk + 1]), Wi = pku(wf[4 * kk + 2], wf[4 * kk + 3]);
                        const P2 re = v[k].re, im = v[k].im;  // lanes (A, B)
                        const P2 yr = fma2(hi2(im), neg2(Wi), fma2(hi2(re), Wr, lo2(re)));
                        const P2 yi = fma2(hi2(re), Wi, fma2(hi2(im), Wr, lo2(im)));
                        pw[k] = pol ? fma2(yi, yi, fma2(yr, yr, pw[k])) : fma2(yi, yi, mul2(yr, yr));
                    }
                }
            }
        }
        // ---- time integration over D adjacent samples = D adjacent lanes
        __syncwarp();  // the previous trial's reads of this warp's tile are done
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const int n = (k / R2) + U2 * (k % R2);
            float2 q;
            upk(pw[k], q.x, q.y);
            ib[n * G::IROW + lane] = q;
        }
        __syncwarp();
        float *outd = out0 + (size_t)d * (size_t)a.out_stride_dm;
        const int i = lane & (DG - 1), g0 = lane - i;
        const int tgrp = (D > 16) ? (tid & ~31) : (tid - i);  // first sample of the group, before + NT n
#pragma unroll
        for (int kk = 0; kk < 16 / DG; ++kk) {
            const int n = i + DG * kk;
            const float4 *row = reinterpret_cast<const float4 *>(ib + n * G::IROW + g0);
            P2 acc = pk(0.f, 0.f);
#pragma unroll
            for (int q = 0; q < DG / 2; ++q) {
                const float4 f = row[q];
                acc = add2(acc, add2(pk(f.x, f.y), pk(f.z, f.w)));
            }
            float s0, s1;
            upk(acc, s0, s1);
            if (D > 16) {
                s0 += __shfl_xor_sync(0xffffffffu, s0, 16);
                s1 += __shfl_xor_sync(0xffffffffu, s1, 16);
            }
            const int t0 = tgrp + NT * n;
            if (D <= 16 || lane < 16) {
                if (t0 >= a.hdisc && t0 < M - a.hdisc) outd[(size_t)((t0 - a.hdisc) >> LOGD) * a.out_pitch] = s0 * a.scale;
                const int t1 = t0 + L;
                if (t1 >= a.hdisc && t1 < M - a.hdisc) outd[(size_t)((t1 - a.hdisc) >> LOGD) * a.out_pitch] = s1 * a.scale;
            }
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
static cudaError_t launch_x2_MD(FusedArgs fa, const double *h_dm, int nunits, cudaStream_t st, long long *launches)
{
    using G = X2<M>;
    // resident CTAs x TMEM columns must stay <= 512: cap the occupancy through the shared-memory request
    size_t smem = G::smem_bytes;
    const size_t floor_bytes = (size_t)(233472 / (G::CTAS_PER_SM + 1)) - 1024 + 16;
    if (smem < floor_bytes) smem = floor_bytes;
    cudaError_t e = cudaFuncSetAttribute(k_fused_x2<M, LOGD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int ndm_total = fa.ndm;
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    for (int d0 = 0; d0 < ndm_total; d0 += DM_PARAM_MAX) {
        const int cnt = ndm_total - d0 < DM_PARAM_MAX ? ndm_total - d0 : DM_PARAM_MAX;
        DmParams dmp;
        for (int i = 0; i < cnt; ++i) dmp.dm[i] = h_dm[d0 + i];
        for (int i = cnt; i < DM_PARAM_MAX; ++i) dmp.dm[i] = 0.0;
        fa.dm_first = d0;
        fa.dm_param0 = d0;
        fa.ndm = d0 + cnt;
        // last wave of a small launch: as in k_fused_ws (cdmt_fused5.cu), the CTAs beyond the last full wave
        // run as DM tiles that fill the SMs once (c2: 2880 CTAs = 19.5 waves of 148)
        const int nctas = nunits * fa.nchan, slots = nsm * G::CTAS_PER_SM;
        const int full = nctas / slots * slots, rem = nctas - full;
        const bool split = fa.dm_tile >= cnt && rem > 0 && full > 0 && nctas / slots < 100 && 2 * rem <= slots && cnt >= 16;
        auto launch = [&](int cta0, int n, int tile) {
            FusedArgs la = fa;
            la.cta0 = cta0;
            la.dm_tile = tile;
            dim3 grid((unsigned)n, (unsigned)((cnt + tile - 1) / tile));
            k_fused_x2<M, LOGD><<<grid, M / 32, smem, st>>>(la, dmp);
            ++*launches;
            return cudaGetLastError();
        };
        if (!split) {
            e = launch(0, nctas, fa.dm_tile);
        } else {
            e = launch(0, full, fa.dm_tile);
            if (e != cudaSuccess) return e;
            int ny = slots / rem;
            if (ny > cnt / 8) ny = cnt / 8;
            e = launch(full, rem, (cnt + ny - 1) / ny);
        }
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

template <int M>
static cudaError_t launch_x2_M(int logd, const FusedArgs &fa, const double *h_dm, int nunits, cudaStream_t st,
                               long long *launches)
{
    switch (logd) {
    case 3: return launch_x2_MD<M, 3>(fa, h_dm, nunits, st, launches);
    case 4: return launch_x2_MD<M, 4>(fa, h_dm, nunits, st, launches);
    case 5: return launch_x2_MD<M, 5>(fa, h_dm, nunits, st, launches);
    default: return cudaErrorInvalidValue;
    }
}

bool fused_x2_supported(int M, int ndec, int hdisc)
{
    if (M != 2048 && M != 4096 && M != 8192) return false;
    if (ndec != 8 && ndec != 16 && ndec != 32) return false;
    return hdisc % ndec == 0;
}

cudaError_t launch_fused_x2(int M, int logd, const FusedArgs &fa, const double *h_dm, int nunits, cudaStream_t st,
                            long long *launches)
{
    switch (M) {
    case 2048: return launch_x2_M<2048>(logd, fa, h_dm, nunits, st, launches);
    case 4096: return launch_x2_M<4096>(logd, fa, h_dm, nunits, st, launches);
    case 8192: return launch_x2_M<8192>(logd, fa, h_dm, nunits, st, launches);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace cdmt
