// cdmt_fused.cu -- the fused per-DM kernels (Alg. 1 l.99-103 + time integration):
// one CTA per (subband, block, channel); the channel's spectrum of both polarisations stays
// in shared memory while the CTA loops over a tile of DM trials, so the spectrum is read from
// HBM once per DM tile and only the integrated float32 filterbank is written.
//
// Per DM trial and polarisation:  Z[m] = X[m] * exp(2 pi i DM g[m])      (Eq. 1)
//                                 y[t] = sum_m Z[m] exp(+2 pi i m t / M)
//   (the per-channel swap of halves only multiplies y[t] by (-1)^t, which detection removes)
// then |y_0|^2 + |y_1|^2, unpad, sum over ndec samples, scale 1/(N M), pack.
//
//  k_fused_fast<M, LOGD>   ndec = 2^LOGD <= 32, h % ndec == 0, M >= 512: chirp phase from a
//                          per-thread degree-5 polynomial in fp64, in-place radix-16 passes
//                          (3 barriers per transform), warp-shuffle reduce-scatter for the time
//                          integration; <= 128 registers so that two CTAs share an SM at M = 4096.
//  k_fused_generic<M>      any ndec / overlap / M >= 16: exact per-bin phase constants in
//                          registers, autosort passes, integration through shared memory.
#include <cstdint>

#include "cdmt_fft.cuh"
#include "cdmt_fused_common.cuh"
#include "cdmt_internal.h"

namespace cdmt {

// ------------------------------------------------------------------------------------
// generic kernel
// ------------------------------------------------------------------------------------
template <int M>
__global__ void __launch_bounds__(M / 16) k_fused_generic(const FusedArgs a)
{
    constexpr int NT = M / 16;
    using Plan = RadixPlan<M>;
    using First = Pass<M, 0, +1, NT, 1>;
    using Last = Pass<M, Plan::npass - 1, +1, NT, 1>;
    extern __shared__ float2 smem[];
    float2 *X = smem;           // [2][M]
    float2 *ex = smem + 2 * M;  // SmemAddr<1>::size(M)
    const int tid = threadIdx.x;
    const int c = blockIdx.x % a.nchan;
    const int ulocal = blockIdx.x / a.nchan;
    const int unit = a.unit0 + ulocal, b = unit / a.nsub, s = unit % a.nsub;
    {
        const float4 *src0 = reinterpret_cast<const float4 *>(a.spec + ((size_t)ulocal * 2) * a.nfft + (size_t)c * M);
        const float4 *src1 = reinterpret_cast<const float4 *>(a.spec + ((size_t)ulocal * 2 + 1) * a.nfft + (size_t)c * M);
        float4 *d0 = reinterpret_cast<float4 *>(X), *d1 = reinterpret_cast<float4 *>(X + M);
        for (int e = tid; e < M / 2; e += NT) {
            d0[e] = __ldg(src0 + e);
            d1[e] = __ldg(src1 + e);
        }
    }
    double g[16];  // Eq. 1 per bin: phase = DM * g, cycles
    {
        double f0, fb0, df;
        chirp_axes(a, s, c, M, &f0, &fb0, &df);
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const double f = fb0 + (double)First::in_elem(tid, 0, r) * df;
            g[r] = f * f / (2.41e-10 * f0 * f0 * (f0 + f));
        }
    }
    __syncthreads();
    const int nchan_total = a.nsub * a.nchan;
    const int ochan = nchan_total - 1 - (s * a.nchan + c);
    const int d_begin = a.dm_first + blockIdx.y * a.dm_tile;
    const int d_end = min(a.ndm, d_begin + a.dm_tile);
    for (int d = d_begin; d < d_end; ++d) {
        const double dm = a.dmlist[d];
        float2 H[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) H[r] = unit_phasor_rt(frac_cycles(dm, g[r]), a.accurate);
        float acc[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[i] = 0.f;
#pragma unroll 1
        for (int p = 0; p < 2; ++p) {
            float2 v[16];
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = cmul(X[p * M + First::in_elem(tid, 0, r)], H[r]);
            __syncthreads();  // exchange buffer free
            fft_passes<M, 0, +1, NT, 1, true>(v, ex, a.tw, tid);
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[i] = fmaf(v[i].x, v[i].x, fmaf(v[i].y, v[i].y, acc[i]));
        }
        float *outd = a.out + (size_t)d * (size_t)a.out_stride_dm + (size_t)b * a.vdec * a.out_pitch + ochan;
        float *I = reinterpret_cast<float *>(ex);
        __syncthreads();
#pragma unroll
        for (int u = 0; u < Last::U; ++u)
#pragma unroll
            for (int q = 0; q < Last::R; ++q) I[Last::out_elem(tid, u, q)] = acc[u * Last::R + q];
        __syncthreads();
        for (int qd = tid; qd < a.vdec; qd += NT) {
            float sum = 0.f;
            for (int r = 0; r < a.ndec; ++r) sum += I[a.hdisc + qd * a.ndec + r];
            outd[(size_t)qd * a.out_pitch] = sum * a.scale;
        }
    }
}

// ------------------------------------------------------------------------------------
// fast kernel: in-place passes.  Pass p transforms input digit i_p (stride M/(R_0..R_p)) into
// output digit o_p (weight T_p = R_0..R_(p-1)); a value whose digits are (d_0, d_1, rho), rho =
// the remaining digits in natural order, lives at rho*16*PITCH + d_1*PITCH + d_0:
//   pass 0: thread (rho, d_1) writes its 16 outputs d_0 = 0..15 as 8 consecutive 16-byte words
//   pass 1: thread (rho, d_0) reads/writes d_1 = 0..15 -- the same 16 threads (one half-warp)
//           that wrote them, so a __syncwarp() is all that pass 0 -> pass 1 needs
//   pass p>=2: lanes run over d_0 (consecutive addresses), block barrier before it
// The barrier that protects the buffer against the NEXT transform's pass-0 stores is split
// into an mbarrier arrive (after the last pass has read) and a wait (before pass 0 stores).
// ------------------------------------------------------------------------------------
template <int M>
struct InplacePlan {
    using Plan = RadixPlan<M>;
    static constexpr int NT = M / 16;
    static constexpr int PITCH = 18;                    // d_1 pitch in elements: 16-byte aligned, 4 banks apart
    static constexpr int RHO = 16 * PITCH;              // elements per rho
    static constexpr int size = (M / 256) * RHO;
    static constexpr int after(int p)  // product of radices after pass p
    {
        int n = 1;
        for (int q = p + 1; q < Plan::npass; ++q) n *= Plan::radix(q);
        return n;
    }
    // the bin offset (within its radix-16 column) that pass-0 thread t owns
    static __device__ __forceinline__ int rest_of_thread(int t) { return (t & 15) * (NT / 16) + (t >> 4); }
};

template <int M, int P>
struct InplacePass {
    static_assert(P >= 1, "pass 0 is written out in the kernel");
    using Plan = RadixPlan<M>;
    using IP = InplacePlan<M>;
    static constexpr int NT = IP::NT;
    static constexpr int R = Plan::radix(P);
    static constexpr int T = Plan::ns(P);     // weight of the output digit
    static constexpr int A = IP::after(P);    // stride of digit P inside rho (P >= 2)
    static constexpr int A2 = IP::after(2);
    static constexpr int U = 16 / R;
    static constexpr int TWOFF = Plan::tw_offset(P);
    static constexpr int XSTRIDE = (P == 1) ? IP::PITCH : A * IP::RHO;

    // twiddle index K of butterfly beta and the address of its element x = 0
    static __device__ __forceinline__ void decode(int beta, int *K, int *base)
    {
        if (P == 1) {  // beta = rho*16 + d0
            *K = beta & 15;
            *base = (beta >> 4) * IP::RHO + (beta & 15);
        } else {       // beta = K + T*lo, K = d0 + 16 d1 (+ 256 d2)
            const int k = beta % T, lo = beta / T;
            int rho = lo;
            if (P >= 3) rho += ((k >> 8) & 15) * A2;
            *K = k;
            *base = rho * IP::RHO + ((k >> 4) & 15) * IP::PITCH + (k & 15);
        }
    }
    static __device__ __forceinline__ void load(const float2 *ex, float2 *v, int tid)
    {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            int K, bs;
            decode(tid + u * NT, &K, &bs);
#pragma unroll
            for (int x = 0; x < R; ++x) v[u * R + x] = ex[bs + x * XSTRIDE];
        }
    }
    static __device__ __forceinline__ void store(float2 *ex, const float2 *v, int tid)
    {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            int K, bs;
            decode(tid + u * NT, &K, &bs);
#pragma unroll
            for (int x = 0; x < R; ++x) ex[bs + x * XSTRIDE] = v[u * R + x];
        }
    }
    static __device__ __forceinline__ void compute(float2 *v, const float2 *__restrict__ tw, int tid)
    {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            int K, bs;
            decode(tid + u * NT, &K, &bs);
            const float2 *t = tw + TWOFF + K;
#pragma unroll
            for (int x = 1; x < R; ++x) v[u * R + x] = cmul(v[u * R + x], __ldg(t + (x - 1) * T));
            Dft<R, +1>::run(v + u * R);
        }
    }
};

// passes 2.. : block barrier, load, butterfly, (store in place)
template <int M, int P>
__device__ __forceinline__ void inplace_tail(float2 *v, float2 *ex, const float2 *__restrict__ tw, int tid,
                                             uint64_t *bar)
{
    using Ps = InplacePass<M, P>;
    __syncthreads();  // previous pass stored
    Ps::load(ex, v, tid);
    if constexpr (P + 1 == RadixPlan<M>::npass) {
        // the multiply below depends on every load above: once it has issued, the buffer may
        // be overwritten by the next transform
        Ps::compute(v, tw, tid);
        mbar_arrive(bar);
    } else {
        Ps::compute(v, tw, tid);
        Ps::store(ex, v, tid);  // same slots this thread just read
        inplace_tail<M, P + 1>(v, ex, tw, tid, bar);
    }
}

template <int M, int LOGD>
__global__ void __launch_bounds__(M / 16, (512 / (M / 16) > 16 ? 16 : (512 / (M / 16) < 1 ? 1 : 512 / (M / 16))))
k_fused_fast(const FusedArgs a, const __grid_constant__ DmParams dmp)
{
    constexpr int NT = M / 16;
    constexpr int D = 1 << LOGD;
    constexpr int LS = LOGD < 4 ? LOGD : 4;  // reduce-scatter stages (16 values per thread)
    constexpr int NKEEP = 16 >> LS;          // integrated samples per thread per DM
    using Plan = RadixPlan<M>;
    using IP = InplacePlan<M>;
    using P1 = InplacePass<M, 1>;
    using LastP = InplacePass<M, Plan::npass - 1>;
    static_assert(Plan::npass >= 3 && NT >= 32, "fast path needs M >= 512");
    extern __shared__ float2 smem[];
    float2 *X = smem;           // [2][16][NT]: bin x NT + rest(t) at [x][t]
    float2 *ex = smem + 2 * M;  // IP::size
    double *coef = reinterpret_cast<double *>(ex + IP::size);  // [6][NT]
    uint64_t *bar = reinterpret_cast<uint64_t *>(coef + 6 * NT);
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int c = blockIdx.x % a.nchan;
    const int ulocal = blockIdx.x / a.nchan;
    const int unit = a.unit0 + ulocal, b = unit / a.nsub, s = unit % a.nsub;
    if (tid == 0) mbar_init(bar, NT);
    {
        // channel spectrum -> shared memory in the order pass 0 reads it
        const float2 *src0 = a.spec + ((size_t)ulocal * 2) * a.nfft + (size_t)c * M;
        const float2 *src1 = src0 + a.nfft;
#pragma unroll 4
        for (int m = tid; m < M; m += NT) {
            const int x = m / NT, rest = m % NT;
            const int t = (rest % (NT / 16)) * 16 + rest / (NT / 16);
            X[x * NT + t] = __ldg(src0 + m);
            X[M + x * NT + t] = __ldg(src1 + m);
        }
    }
    // Eq. 1 along this thread's bins m_r = rest + r M/16: g(f_a + b r) = sum_k ck r^k (Taylor in
    // b r / (f0 + f_a) <= 1e-3; the host checks that the r^6 term is below 1e-7 cycles).
    {
        double f0, fb0, df;
        chirp_axes(a, s, c, M, &f0, &fb0, &df);
        const double fa = fb0 + (double)IP::rest_of_thread(tid) * df, bb = (double)NT * df;
        const double kc = 1.0 / (2.41e-10 * f0 * f0);
        const double sa = f0 + fa, e = bb / sa, pp = kc * f0 * f0 / sa;
        const double c2 = pp * e * e, c3 = -c2 * e, c4 = -c3 * e, c5 = -c4 * e;
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
    // pass-0 thread (rho, d1) = (tid >> 4, tid & 15) stores at rho*RHO + d1*PITCH + 0..15
    float4 *p0_store = reinterpret_cast<float4 *>(ex + (tid >> 4) * IP::RHO + (tid & 15) * IP::PITCH);
    unsigned nfft_done = 0;  // transforms finished by this CTA: parity of the mbarrier phase
    __syncthreads();

#pragma unroll 1
    for (int d = d_begin; d < d_end; ++d) {
        const double dm = dmp.dm[d - a.dm_param0];
        // phase polynomial of this DM (scaling the coefficients keeps the evaluation inside the loop)
        const double p0 = dm * coef[0 * NT + tid], p1 = dm * coef[1 * NT + tid], p2 = dm * coef[2 * NT + tid];
        const double p3 = dm * coef[3 * NT + tid], p4 = dm * coef[4 * NT + tid], p5 = dm * coef[5 * NT + tid];
        float2 H[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const double rr = (double)r;
            const double phi = fma(fma(fma(fma(fma(p5, rr, p4), rr, p3), rr, p2), rr, p1), rr, p0);
            const double magic = 6755399441055744.0;
            const double n = (phi + magic) - magic;
            H[r] = unit_phasor<false>((float)(phi - n));
        }
        float res[NKEEP];
#pragma unroll 1
        for (int p = 0; p < 2; ++p) {
            float2 v[16];
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = cmul(X[p * M + r * NT + tid], H[r]);
            Dft<16, +1>::run(v);
            if (nfft_done) mbar_wait(bar, (nfft_done - 1) & 1);  // previous transform fully read
#pragma unroll
            for (int q = 0; q < 8; ++q)
                p0_store[q] = make_float4(v[2 * q].x, v[2 * q].y, v[2 * q + 1].x, v[2 * q + 1].y);
            __syncwarp();
            P1::load(ex, v, tid);
            P1::compute(v, a.tw, tid);
            P1::store(ex, v, tid);
            inplace_tail<M, 2>(v, ex, a.tw, tid, bar);
            ++nfft_done;
            // v[u R + x] = y[t], t = tid + NT (u + U x): reorder to n = u + U x, detect
            float pw[16];
#pragma unroll
            for (int u = 0; u < LastP::U; ++u)
#pragma unroll
                for (int x = 0; x < LastP::R; ++x) {
                    const float2 y = v[u * LastP::R + x];
                    pw[u + LastP::U * x] = fmaf(y.x, y.x, y.y * y.y);
                }
            lane_reduce_scatter<LS>(pw, lane);
            if constexpr (LOGD > LS) pw[0] += __shfl_xor_sync(0xffffffffu, pw[0], 16);
#pragma unroll
            for (int j = 0; j < NKEEP; ++j) res[j] = (p == 0) ? pw[j] : res[j] + pw[j];
        }
        float *outd = out0 + (size_t)d * (size_t)a.out_stride_dm;
#pragma unroll
        for (int j = 0; j < NKEEP; ++j) {
            const int n = (lane & ((1 << LS) - 1)) + (1 << LS) * j;
            const int t0 = (tid & ~(D - 1)) + NT * n;  // first sample of the integrated group
            if ((lane & (D - 1)) < (1 << LS) && t0 >= a.hdisc && t0 < M - a.hdisc)
                outd[(size_t)((t0 - a.hdisc) >> LOGD) * a.out_pitch] = res[j] * a.scale;
        }
    }
}

// ------------------------------------------------------------------------------------
// launch
// ------------------------------------------------------------------------------------
template <int M>
static cudaError_t launch_generic_M(const FusedArgs &fa, dim3 grid, cudaStream_t st)
{
    const size_t smem = sizeof(float2) * (2 * (size_t)M + SmemAddr<1>::size(M));
    cudaError_t e = cudaFuncSetAttribute(k_fused_generic<M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_fused_generic<M><<<grid, M / 16, smem, st>>>(fa);
    return cudaGetLastError();
}

template <int M, int LOGD>
static cudaError_t launch_fast_MD(FusedArgs fa, const double *h_dm, int nunits, cudaStream_t st, long long *launches)
{
    const size_t smem = sizeof(float2) * (2 * (size_t)M + InplacePlan<M>::size) + sizeof(double) * 6 * (M / 16) + 16;
    cudaError_t e = cudaFuncSetAttribute(k_fused_fast<M, LOGD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
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
        k_fused_fast<M, LOGD><<<grid, M / 16, smem, st>>>(fa, dmp);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        ++*launches;
    }
    return cudaSuccess;
}

template <int M>
static cudaError_t launch_fast_M(int logd, const FusedArgs &fa, const double *h_dm, int nunits, cudaStream_t st,
                                 long long *launches)
{
    switch (logd) {
    case 0: return launch_fast_MD<M, 0>(fa, h_dm, nunits, st, launches);
    case 1: return launch_fast_MD<M, 1>(fa, h_dm, nunits, st, launches);
    case 2: return launch_fast_MD<M, 2>(fa, h_dm, nunits, st, launches);
    case 3: return launch_fast_MD<M, 3>(fa, h_dm, nunits, st, launches);
    case 4: return launch_fast_MD<M, 4>(fa, h_dm, nunits, st, launches);
    case 5: return launch_fast_MD<M, 5>(fa, h_dm, nunits, st, launches);
    default: return cudaErrorInvalidValue;
    }
}

// Can the degree-5 phase polynomial be used?  Bound on the first neglected term (cycles).
static bool poly_phase_ok(const Geometry &g, const double *h_dm, const double *h_fcen)
{
    double dmax = 0.0, fmin = h_fcen[0];
    for (int d = 0; d < g.ndm; ++d) dmax = fabs(h_dm[d]) > dmax ? fabs(h_dm[d]) : dmax;
    for (int s = 0; s < g.nsub; ++s) fmin = h_fcen[s] < fmin ? h_fcen[s] : fmin;
    const double flo = fmin - 0.5 * g.bw_mhz;
    const double x = 15.0 * (g.mbin / 16) * (g.bw_mhz / g.nfft) / flo;
    const double P = dmax / (2.41e-10 * flo);
    return P * x * x * x * x * x * x < 1e-7;
}

// Upper bound on |phase| of Eq. 1 in cycles over all bins, subbands and DM trials.
static double phase_cycles_bound(const Geometry &g, const double *h_dm, const double *h_fcen)
{
    double dmax = 0.0, fmin = h_fcen[0];
    for (int d = 0; d < g.ndm; ++d) dmax = fabs(h_dm[d]) > dmax ? fabs(h_dm[d]) : dmax;
    for (int s = 0; s < g.nsub; ++s) fmin = h_fcen[s] < fmin ? h_fcen[s] : fmin;
    const double flo = fmin - 0.5 * g.bw_mhz;
    const double fmax = g.chirp_ref == 0 ? 0.5 * g.bw_mhz / g.nchan : 0.5 * g.bw_mhz;
    return dmax * fmax * fmax / (2.41e-10 * flo * flo * flo);
}

cudaError_t launch_fused(const Geometry &g, const Workspace &ws, const float2 *spec, int unit0, int nunits,
                         float *d_out, long long out_stride_dm, int out_pitch, int dm_tile, int accurate, int force_generic,
                         const double *h_dm, const double *h_fcen, double *d_segsum, int nblock_total,
                         bool *sums_done, cudaStream_t st, long long *launches)
{
    if (d_segsum && sums_done) *sums_done = false;   // set again by a kernel that takes the sums itself
    const int M = g.mbin, D = g.ndec;
    if (dm_tile <= 0 || dm_tile > g.ndm) dm_tile = g.ndm;
    dim3 grid((unsigned)(nunits * g.nchan), (unsigned)((g.ndm + dm_tile - 1) / dm_tile));
    FusedArgs fa;
    fa.spec = spec; fa.tw = ws.tw_m; fa.dmlist = ws.dm; fa.fcen = ws.fcen; fa.out = d_out;
    fa.out_stride_dm = out_stride_dm; fa.out_pitch = out_pitch > 0 ? out_pitch : g.nsub * g.nchan; fa.unit0 = unit0; fa.nsub = g.nsub; fa.nchan = g.nchan; fa.nfft = g.nfft;
    fa.hdisc = g.hdisc; fa.ndec = g.ndec; fa.vdec = g.vdec; fa.ndm = g.ndm; fa.dm_tile = dm_tile;
    fa.chirp_ref = g.chirp_ref; fa.accurate = accurate; fa.bw_mhz = g.bw_mhz;
    fa.scale = (float)(1.0 / ((double)g.nfft * (double)M));
    fa.dm_first = 0;
    fa.dm_param0 = 0;
    fa.nb_chunk = 0;
    fa.cta0 = 0;
    fa.segsum = nullptr;
    fa.nblock_total = nblock_total;
    int logd = 0;
    while ((1 << logd) < D) ++logd;
    // force_generic carries CDMT_OPT_FUSED_KERNEL: 0 auto, 1 generic, 2 scalar fast, 3 packed halves (x2),
    // 4 packed halves, warp-specialised, two blocks per CTA (ws), 5 packed pols, software-pipelined chirp (sp)
    const bool fast_ok = !accurate && M >= 512 && D <= 32 && (1 << logd) == D && (g.hdisc % D) == 0 &&
                         poly_phase_ok(g, h_dm, h_fcen);
    // x2 and sp reduce the phase mod 1 with a 2^20 magic number: |phase| must stay below 2^19 cycles
    const bool small_phase = phase_cycles_bound(g, h_dm, h_fcen) < 262144.0;
    const bool x2_ok = fast_ok && small_phase && fused_x2_supported(M, D, g.hdisc);
    const bool sp_ok = fast_ok && small_phase && fused_sp_supported(M, D, g.hdisc);
    if (force_generic == 5 && !sp_ok) return cudaErrorInvalidValue;
    const bool ws_ok = x2_ok && fused_ws_supported(M, D, g.hdisc, g.nsub, unit0, nunits);
    if (force_generic == 4 && !ws_ok) return cudaErrorInvalidValue;
    if (force_generic == 3 && !x2_ok) return cudaErrorInvalidValue;
    if (force_generic == 2 && !fast_ok) return cudaErrorInvalidValue;
    // automatic choice: x2 (measured fastest on all five configs: c3 21.8 ms per launch against 22.2 for sp),
    // then sp (covers ndec < 8)
    // automatic choice: ws needs at least one full pair of blocks (a lone block would leave the second FFT
    // group of every CTA idle: x2 is faster there)
    if (ws_ok && ((force_generic == 0 && nunits >= 2 * g.nsub) || force_generic == 4)) {
        // the warp-specialised kernel takes the block sums of l.104 itself (its chirp warps have the time);
        // in k_fused_x2 the same fp64 sums cost 7 % of the kernel (c5: 139 ms against 23 ms for the separate
        // pass over the filterbank), so every other kernel leaves them to launch_block_sums
        fa.segsum = reinterpret_cast<double2 *>(d_segsum);
        if (d_segsum && sums_done) *sums_done = true;
        return launch_fused_ws(M, logd, fa, h_dm, nunits, st, launches);
    }
    if (x2_ok && (force_generic == 0 || force_generic == 3)) return launch_fused_x2(M, logd, fa, h_dm, nunits, st, launches);
    if (sp_ok && (force_generic == 0 || force_generic == 5)) return launch_fused_sp(M, logd, fa, h_dm, nunits, st, launches);
    const bool fast = fast_ok && force_generic != 1;
    cudaError_t e = cudaErrorInvalidValue;
    if (fast) {
        switch (M) {
        case 512: e = launch_fast_M<512>(logd, fa, h_dm, nunits, st, launches); break;
        case 1024: e = launch_fast_M<1024>(logd, fa, h_dm, nunits, st, launches); break;
        case 2048: e = launch_fast_M<2048>(logd, fa, h_dm, nunits, st, launches); break;
        case 4096: e = launch_fast_M<4096>(logd, fa, h_dm, nunits, st, launches); break;
        case 8192: e = launch_fast_M<8192>(logd, fa, h_dm, nunits, st, launches); break;
        default: break;
        }
        return e;
    } else {
        switch (M) {
        case 16: e = launch_generic_M<16>(fa, grid, st); break;
        case 32: e = launch_generic_M<32>(fa, grid, st); break;
        case 64: e = launch_generic_M<64>(fa, grid, st); break;
        case 128: e = launch_generic_M<128>(fa, grid, st); break;
        case 256: e = launch_generic_M<256>(fa, grid, st); break;
        case 512: e = launch_generic_M<512>(fa, grid, st); break;
        case 1024: e = launch_generic_M<1024>(fa, grid, st); break;
        case 2048: e = launch_generic_M<2048>(fa, grid, st); break;
        case 4096: e = launch_generic_M<4096>(fa, grid, st); break;
        case 8192: e = launch_generic_M<8192>(fa, grid, st); break;
        default: break;
        }
    }
    if (e == cudaSuccess) ++*launches;
    return e;
}

}  // namespace cdmt
