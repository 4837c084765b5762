// cdmt_kernels.cu -- the sm_100a kernels of the cdmt hot path and their launchers.
//
//  k_init_tables                DM list, centre frequencies and twiddle tables into the workspace head
//  k_unpack                     Alg. 1 l.95 as a stand-alone stage
//  k_fwd_pass<L, MODE, IN>      forward FFT of length nfft = n1*n2 as two passes of a four-step
//                               decomposition; pass A reads the raw voltages (unpack fused into
//                               its loads), pass B writes the swapped-halves spectrum (l.96-97)
//  k_fused<M, ...>              l.99-103 for a tile of DM trials: chirp on the fly, length-M
//                               backward FFT, unpad, detect, Stokes I, time integration, pack
#include "cdmt_fft.cuh"
#include "cdmt_internal.h"

namespace cdmt {

// ------------------------------------------------------------------------------------
// constant tables
// ------------------------------------------------------------------------------------
constexpr int INIT_CHUNK = 1024;  // doubles carried per table in one kernel parameter block
struct DoubleChunk {
    double v[INIT_CHUNK];
};

// pass twiddles of RadixPlan<L> (runtime evaluation of the same layout); `nthreads` threads, this one is `t`
__device__ void init_pass_twiddles(float2 *tw, int L, int sign, int t, int nthreads)
{
    int log2L = 31 - __clz(L);
    int n16 = log2L / 4, rest = 1 << (log2L % 4);
    int npass = n16 + (rest > 1 ? 1 : 0);
    int off = 0, ns = 1;
    for (int p = 0; p < npass; ++p) {
        int R = p < n16 ? 16 : rest;
        if (p >= 1) {
            int cnt = (R - 1) * ns;
            for (int e = t; e < cnt; e += nthreads) {
                int r = e / ns + 1, k = e % ns;
                double s, c;
                sincospi(2.0 * (double)k * (double)r / ((double)ns * (double)R), &s, &c);
                tw[off + e] = make_float2((float)c, (float)(sign * s));
            }
            off += cnt;
        }
        ns *= R;
    }
}

// four-step twiddles: exp(-2 pi i e / N) = hi[e >> lo_bits] * lo[e & (2^lo_bits - 1)]
__device__ void init_fourstep(float2 *lo, float2 *hi, int N, int lo_bits, int t, int nthreads)
{
    int nlo = 1 << lo_bits, nhi = N >> lo_bits;
    for (int e = t; e < nlo + nhi; e += nthreads) {
        double s, c;
        if (e < nlo) {
            sincospi(-2.0 * (double)e / (double)N, &s, &c);
            lo[e] = make_float2((float)c, (float)s);
        } else {
            int a = e - nlo;
            sincospi(-2.0 * (double)a * (double)nlo / (double)N, &s, &c);
            hi[a] = make_float2((float)c, (float)s);
        }
    }
}

struct InitArgs {
    double *dm, *fcen;
    float2 *tw_n1, *tw_n2, *tw_m, *tw4_lo, *tw4_hi;
    int n1, n2, mbin, nfft, lo_bits;
    int dm0, ndm, f0, nf;   // this launch carries dm[dm0, dm0 + ndm) and fcen[f0, f0 + nf)
    int tables;             // 1: also fill the twiddle tables
};

// One launch fills the whole head of the workspace: block 0 the DM list, block 1 the centre
// frequencies (both travel in the kernel parameter block, so that the call stays capturable into
// a CUDA graph), blocks 2.. the twiddle tables by role (blockIdx % 4).
__global__ void __launch_bounds__(256)
k_init_tables(const InitArgs a, const __grid_constant__ DoubleChunk dm, const __grid_constant__ DoubleChunk fc)
{
    const int t = threadIdx.x;
    if (blockIdx.x == 0) {
        for (int i = t; i < a.ndm; i += 256) a.dm[a.dm0 + i] = dm.v[i];
        return;
    }
    if (blockIdx.x == 1) {
        for (int i = t; i < a.nf; i += 256) a.fcen[a.f0 + i] = fc.v[i];
        return;
    }
    if (!a.tables) return;
    const int role = (blockIdx.x - 2) & 3, nb = (gridDim.x - 2) >> 2;
    const int tt = ((blockIdx.x - 2) >> 2) * 256 + t, nthreads = nb * 256;
    if (role == 0) init_pass_twiddles(a.tw_n1, a.n1, -1, tt, nthreads);
    else if (role == 1) init_pass_twiddles(a.tw_n2, a.n2, -1, tt, nthreads);
    else if (role == 2) init_pass_twiddles(a.tw_m, a.mbin, +1, tt, nthreads);
    else init_fourstep(a.tw4_lo, a.tw4_hi, a.nfft, a.lo_bits, tt, nthreads);
}

// ------------------------------------------------------------------------------------
// input words -> complex float (Alg. 1 l.95 "unpack")
// ------------------------------------------------------------------------------------
// Input layouts (include/cdmt.h CDMT_IN_*): 0 interleaved float32, 1 interleaved int8, 2 planar float32,
// 3 planar int8.  Interleaved: row (s, p) = complex words; planar: rows (s, p, re) and (s, p, im) of real
// words, `stride` apart ("unpacked into two cufftComplex arrays, one for each polarization").
template <int IN>
struct InWord;
template <> struct InWord<0> { static constexpr int bytes = 8, rows = 2; };
template <> struct InWord<1> { static constexpr int bytes = 2, rows = 2; };
template <> struct InWord<2> { static constexpr int bytes = 4, rows = 4; };
template <> struct InWord<3> { static constexpr int bytes = 1, rows = 4; };

// first word of polarisation p of subband s (planar: of its real part)
template <int IN>
__device__ __forceinline__ size_t in_row0(int s, int p, long long stride)
{
    return (size_t)(InWord<IN>::rows * s + (InWord<IN>::rows / 2) * p) * (size_t)stride;
}

template <int IN>
__device__ __forceinline__ float2 load_sample(const void *base, size_t idx, long long stride);
template <>
__device__ __forceinline__ float2 load_sample<0>(const void *base, size_t idx, long long)
{
    return __ldg(reinterpret_cast<const float2 *>(base) + idx);
}
template <>
__device__ __forceinline__ float2 load_sample<1>(const void *base, size_t idx, long long)
{
    char2 q = __ldg(reinterpret_cast<const char2 *>(base) + idx);
    return make_float2((float)q.x, (float)q.y);
}
template <>
__device__ __forceinline__ float2 load_sample<2>(const void *base, size_t idx, long long stride)
{
    const float *f = reinterpret_cast<const float *>(base) + idx;
    return make_float2(__ldg(f), __ldg(f + stride));
}
template <>
__device__ __forceinline__ float2 load_sample<3>(const void *base, size_t idx, long long stride)
{
    const signed char *f = reinterpret_cast<const signed char *>(base) + idx;
    return make_float2((float)__ldg(f), (float)__ldg(f + stride));
}

__device__ __forceinline__ void unpack_int8x4(unsigned w, float (&f)[4])
{
    f[0] = (float)(signed char)(w & 0xff);
    f[1] = (float)(signed char)((w >> 8) & 0xff);
    f[2] = (float)(signed char)((w >> 16) & 0xff);
    f[3] = (float)(signed char)(w >> 24);
}

// blocks[(b nsub + s)][p][n] = in[s][p][b step + n]; 4 samples per thread
template <int IN>
__global__ void __launch_bounds__(256) k_unpack(const void *__restrict__ in, long long in_stride_pol,
                                                int nsub, int nfft, int step, float2 *__restrict__ blocks)
{
    const int row = blockIdx.x;  // (b nsub + s) * 2 + p
    const int unit = row >> 1, p = row & 1, b = unit / nsub, s = unit % nsub;
    const size_t src0 = in_row0<IN>(s, p, in_stride_pol) + (size_t)b * step;
    float2 *dst = blocks + (size_t)row * nfft;
    const int n0 = (blockIdx.y * 256 + threadIdx.x) * 4;
    if (n0 >= nfft) return;
    if (IN == 0) {
        const float4 *src = reinterpret_cast<const float4 *>(reinterpret_cast<const float2 *>(in) + src0 + n0);
        float4 a = __ldg(src), c = __ldg(src + 1);   // step and in_stride_pol are even: 16-byte aligned
        reinterpret_cast<float4 *>(dst + n0)[0] = a;
        reinterpret_cast<float4 *>(dst + n0)[1] = c;
    } else {
        float2 v[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = load_sample<IN>(in, src0 + n0 + i, in_stride_pol);
        reinterpret_cast<float4 *>(dst + n0)[0] = make_float4(v[0].x, v[0].y, v[1].x, v[1].y);
        reinterpret_cast<float4 *>(dst + n0)[1] = make_float4(v[2].x, v[2].y, v[3].x, v[3].y);
    }
}

// ------------------------------------------------------------------------------------
// forward FFT, one pass of the four-step decomposition.
//   n = n1i*n2 + n2i,  k = k1 + n1*k2
//   pass A (MODE 0): for each n2i: T[k1][n2i] = w_N^(n2i k1) * sum_n1i x[n1i n2 + n2i] w_n1^(n1i k1)
//   pass B (MODE 1): for each k1 : U[k1 + n1 k2] = sum_n2i T[k1][n2i] w_n2^(n2i k2), stored at the
//                    swapped-halves position (k + N/2) mod N
// A CTA transforms a tile of 16 transforms of length L held in shared memory as [elem][16+1].
// ------------------------------------------------------------------------------------
constexpr int FWD_BATCH = 16;

template <int L, int MODE, int IN>
__global__ void __launch_bounds__(L, (L == 256 ? ((MODE == 1 || IN == 0 || IN == 2) ? 5 : 4) : 0)) k_fwd_pass(const void *__restrict__ src_v, float2 *__restrict__ dst,
                                                const float2 *__restrict__ tw, const float2 *__restrict__ tw_lo,
                                                const float2 *__restrict__ tw_hi, int lo_bits, int nfft, int n1,
                                                int n2, int nsub, int step, long long in_stride_pol, int unit0,
                                                int vec16)
{
    constexpr int NT = L;
    using Plan = RadixPlan<L>;
    using Addr = SmemAddr<FWD_BATCH>;
    using Last = Pass<L, Plan::npass - 1, -1, NT, FWD_BATCH>;
    extern __shared__ float2 smem[];
    const int tid = threadIdx.x;
    const int tile = blockIdx.y;       // MODE 0: 16 consecutive n2i; MODE 1: 16 consecutive k1
    const int row = blockIdx.x;        // local (unit, pol)
    const int p = row & 1;
    const size_t plane = (size_t)row * nfft;

    if (MODE == 0) {
        const int unit = unit0 + (row >> 1), b = unit / nsub, s = unit % nsub;
        const size_t src0 = in_row0<IN>(s, p, in_stride_pol) + (size_t)b * step + (size_t)tile * FWD_BATCH;
        if ((IN == 1 || IN == 3) && vec16) {
            // int8, 16-byte loads along time: one row of the tile (16 samples) is 32 interleaved bytes = two
            // loads, or 16 + 16 planar bytes = one load per part.  vec16: every such address is 16-byte aligned.
            constexpr int PER_ROW = IN == 1 ? 2 : 1;
#pragma unroll 4
            for (int e = tid; e < L * PER_ROW; e += NT) {
                const int n1i = e / PER_ROW, half = e % PER_ROW;
                const signed char *q = reinterpret_cast<const signed char *>(src_v) +
                                       (src0 + (size_t)n1i * n2) * InWord<IN>::bytes + 16 * half;
                const uint4 w = __ldg(reinterpret_cast<const uint4 *>(q));
                const unsigned ww[4] = {w.x, w.y, w.z, w.w};
                if (IN == 1) {
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        float f[4];
                        unpack_int8x4(ww[k], f);
                        smem[Addr::at(n1i, 8 * half + 2 * k)] = make_float2(f[0], f[1]);
                        smem[Addr::at(n1i, 8 * half + 2 * k + 1)] = make_float2(f[2], f[3]);
                    }
                } else {
                    const uint4 wi = __ldg(reinterpret_cast<const uint4 *>(q + in_stride_pol));
                    const unsigned wwi[4] = {wi.x, wi.y, wi.z, wi.w};
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        float fr[4], fi[4];
                        unpack_int8x4(ww[k], fr);
                        unpack_int8x4(wwi[k], fi);
#pragma unroll
                        for (int j = 0; j < 4; ++j) smem[Addr::at(n1i, 4 * k + j)] = make_float2(fr[j], fi[j]);
                    }
                }
            }
        } else {
#pragma unroll 16  // all 16 loads of a thread in flight (HBM latency; measured 11.8 -> 9.6 ms per c3 step)
            for (int e = tid; e < L * FWD_BATCH; e += NT) {
                const int n1i = e / FWD_BATCH, col = e % FWD_BATCH;
                smem[Addr::at(n1i, col)] = load_sample<IN>(src_v, src0 + (size_t)n1i * n2 + col, in_stride_pol);
            }
        }
    } else {
        const float2 *src = reinterpret_cast<const float2 *>(src_v) + plane + (size_t)tile * FWD_BATCH * n2;
#pragma unroll 16
        for (int e = tid; e < L * FWD_BATCH; e += NT) {
            const int rr = e / L, n2i = e % L;
            smem[Addr::at(n2i, rr)] = __ldg(src + (size_t)rr * n2 + n2i);
        }
    }
    __syncthreads();
    float2 v[16];
    fft_passes<L, 0, -1, NT, FWD_BATCH, false>(v, smem, tw, tid);

    const int nmask = nfft - 1;
#pragma unroll
    for (int u = 0; u < Last::U; ++u) {
        const int col = Last::batch_of(tid, u);
        // MODE 0: the outputs of a butterfly are k = k0 + q NS, so their four-step twiddles w_N^(n2i k)
        // form a geometric sequence: two table look-ups (first term, ratio) and one complex multiply per
        // output instead of two look-ups per output (the gathers kept the L1 data pipe 85 % busy)
        float2 w = make_float2(1.f, 0.f), ratio = w;
        if (MODE == 0) {
            const int n2i = tile * FWD_BATCH + col;
            const int e0 = (int)(((long long)n2i * Last::out_elem(tid, u, 0)) & nmask);
            const int es = (int)(((long long)n2i * Last::NS) & nmask);
            w = cmul(__ldg(tw_hi + (e0 >> lo_bits)), __ldg(tw_lo + (e0 & ((1 << lo_bits) - 1))));
            ratio = cmul(__ldg(tw_hi + (es >> lo_bits)), __ldg(tw_lo + (es & ((1 << lo_bits) - 1))));
        }
#pragma unroll
        for (int q = 0; q < Last::R; ++q) {
            const int k = Last::out_elem(tid, u, q);
            float2 val = v[u * Last::R + q];
            if (MODE == 0) {
                const int n2i = tile * FWD_BATCH + col;
                dst[plane + (size_t)k * n2 + n2i] = cmul(val, w);
                if (q + 1 < Last::R) w = cmul(w, ratio);
            } else {
                const int k1 = tile * FWD_BATCH + col;
                const int kk = k1 + n1 * k;
                dst[plane + ((kk + (nfft >> 1)) & nmask)] = val;
            }
        }
    }
}

// ------------------------------------------------------------------------------------
// FP32 FMA rate (roofline denominator)
// ------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) k_fp32_peak(float *out, int inner)
{
    float a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = (float)(threadIdx.x + i) * 1e-3f;
    const float m = 0.9999f, c = 1e-4f;
    for (int it = 0; it < inner; ++it) {
#pragma unroll
        for (int k = 0; k < 16; ++k)
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = fmaf(a[i], m, c);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
    if (s == 12345.678f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

cudaError_t launch_fp32_peak(float *d_scratch, int nblocks, int inner, cudaStream_t st)
{
    k_fp32_peak<<<nblocks, 1024, 0, st>>>(d_scratch, inner);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------
static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

static int pass_tw_size(int L)
{
    int log2L = 0;
    while ((1 << log2L) < L) ++log2L;
    int n16 = log2L / 4, rest = 1 << (log2L % 4), npass = n16 + (rest > 1 ? 1 : 0);
    int off = 0, ns = 1;
    for (int p = 0; p < npass; ++p) {
        int R = p < n16 ? 16 : rest;
        if (p >= 1) off += (R - 1) * ns;
        ns *= R;
    }
    return off > 0 ? off : 1;
}

size_t workspace_layout(const Geometry &g, int chunk_units, char *base, Workspace *ws)
{
    size_t off = 0;
    auto take = [&](size_t bytes) {
        char *p = base ? base + off : nullptr;
        off += align256(bytes);
        return p;
    };
    Workspace w;
    w.dm = reinterpret_cast<double *>(take(sizeof(double) * (size_t)g.ndm));
    w.fcen = reinterpret_cast<double *>(take(sizeof(double) * (size_t)g.nsub));
    w.tw_n1 = reinterpret_cast<float2 *>(take(sizeof(float2) * (size_t)pass_tw_size(g.n1)));
    w.tw_n2 = reinterpret_cast<float2 *>(take(sizeof(float2) * (size_t)pass_tw_size(g.n2)));
    w.tw_m = reinterpret_cast<float2 *>(take(sizeof(float2) * (size_t)pass_tw_size(g.mbin)));
    w.tw4_lo = reinterpret_cast<float2 *>(take(sizeof(float2) * ((size_t)1 << g.lo_bits)));
    w.tw4_hi = reinterpret_cast<float2 *>(take(sizeof(float2) * ((size_t)g.nfft >> g.lo_bits)));
    const size_t plane = sizeof(float2) * 2 * (size_t)g.nfft * (size_t)chunk_units;
    w.bufA = reinterpret_cast<float2 *>(take(plane));
    w.spec = reinterpret_cast<float2 *>(take(plane));
    w.total_bytes = off;
    if (ws) *ws = w;
    return off;
}

cudaError_t launch_init_tables(const Geometry &g, const Workspace &ws, const double *h_dm,
                               const double *h_fcen, cudaStream_t st, long long *launches)
{
    InitArgs a;
    a.dm = ws.dm; a.fcen = ws.fcen; a.tw_n1 = ws.tw_n1; a.tw_n2 = ws.tw_n2; a.tw_m = ws.tw_m;
    a.tw4_lo = ws.tw4_lo; a.tw4_hi = ws.tw4_hi;
    a.n1 = g.n1; a.n2 = g.n2; a.mbin = g.mbin; a.nfft = g.nfft; a.lo_bits = g.lo_bits;
    // one launch unless a list is longer than a parameter block carries
    for (int o = 0; o < g.ndm || o < g.nsub || o == 0; o += INIT_CHUNK) {
        DoubleChunk dm, fc;
        a.dm0 = o; a.ndm = g.ndm - o < 0 ? 0 : (g.ndm - o < INIT_CHUNK ? g.ndm - o : INIT_CHUNK);
        a.f0 = o;  a.nf = g.nsub - o < 0 ? 0 : (g.nsub - o < INIT_CHUNK ? g.nsub - o : INIT_CHUNK);
        for (int i = 0; i < INIT_CHUNK; ++i) {
            dm.v[i] = i < a.ndm ? h_dm[o + i] : 0.0;
            fc.v[i] = i < a.nf ? h_fcen[o + i] : 0.0;
        }
        a.tables = o == 0;
        k_init_tables<<<a.tables ? 2 + 4 * 8 : 2, 256, 0, st>>>(a, dm, fc);
        ++*launches;
    }
    return cudaGetLastError();
}

cudaError_t launch_unpack(const Geometry &g, const void *d_in, long long in_stride_pol, int nblock,
                          float2 *d_blocks, cudaStream_t st, long long *launches)
{
    dim3 grid((unsigned)(nblock * g.nsub * 2), (unsigned)((g.nfft / 4 + 255) / 256));
    switch (g.in_dtype) {
    case 0: k_unpack<0><<<grid, 256, 0, st>>>(d_in, in_stride_pol, g.nsub, g.nfft, g.step, d_blocks); break;
    case 1: k_unpack<1><<<grid, 256, 0, st>>>(d_in, in_stride_pol, g.nsub, g.nfft, g.step, d_blocks); break;
    case 2: k_unpack<2><<<grid, 256, 0, st>>>(d_in, in_stride_pol, g.nsub, g.nfft, g.step, d_blocks); break;
    default: k_unpack<3><<<grid, 256, 0, st>>>(d_in, in_stride_pol, g.nsub, g.nfft, g.step, d_blocks); break;
    }
    ++*launches;
    return cudaGetLastError();
}

template <int L>
static cudaError_t launch_fwd_L(int mode, const Geometry &g, const Workspace &ws, const void *src, float2 *dst,
                                long long in_stride_pol, int unit0, int nunits, cudaStream_t st)
{
    const size_t smem = sizeof(float2) * SmemAddr<FWD_BATCH>::size(L);
    const float2 *tw = (mode == 0) ? ws.tw_n1 : ws.tw_n2;
    dim3 grid((unsigned)(nunits * 2), (unsigned)((mode == 0 ? g.n2 : g.n1) / FWD_BATCH));
    cudaError_t e;
#define CDMT_FWD(MODE, IN)                                                                                         \
    do {                                                                                                           \
        e = cudaFuncSetAttribute(k_fwd_pass<L, MODE, IN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
        if (e != cudaSuccess) return e;                                                                            \
        k_fwd_pass<L, MODE, IN><<<grid, L, smem, st>>>(src, dst, tw, ws.tw4_lo, ws.tw4_hi, g.lo_bits, g.nfft,      \
                                                       g.n1, g.n2, g.nsub, g.step, in_stride_pol, unit0, vec16);  \
    } while (0)
    // int8 input: 16-byte loads along time where every tile row starts on a 16-byte boundary
    const int wb = g.in_dtype == 1 ? 2 : 1;
    const int vec16 = (g.in_dtype == 1 || g.in_dtype == 3) && (reinterpret_cast<uintptr_t>(src) & 15) == 0 &&
                      ((long long)in_stride_pol * wb) % 16 == 0 && ((long long)g.step * wb) % 16 == 0 &&
                      ((long long)g.n2 * wb) % 16 == 0;
    if (mode == 0) {
        switch (g.in_dtype) {
        case 0: CDMT_FWD(0, 0); break;
        case 1: CDMT_FWD(0, 1); break;
        case 2: CDMT_FWD(0, 2); break;
        default: CDMT_FWD(0, 3); break;
        }
    } else {
        CDMT_FWD(1, 0);
    }
#undef CDMT_FWD
    return cudaGetLastError();
}

static cudaError_t launch_fwd_any(int L, int mode, const Geometry &g, const Workspace &ws, const void *src,
                                  float2 *dst, long long in_stride_pol, int unit0, int nunits, cudaStream_t st)
{
    switch (L) {
    case 16: return launch_fwd_L<16>(mode, g, ws, src, dst, in_stride_pol, unit0, nunits, st);
    case 32: return launch_fwd_L<32>(mode, g, ws, src, dst, in_stride_pol, unit0, nunits, st);
    case 64: return launch_fwd_L<64>(mode, g, ws, src, dst, in_stride_pol, unit0, nunits, st);
    case 128: return launch_fwd_L<128>(mode, g, ws, src, dst, in_stride_pol, unit0, nunits, st);
    case 256: return launch_fwd_L<256>(mode, g, ws, src, dst, in_stride_pol, unit0, nunits, st);
    case 512: return launch_fwd_L<512>(mode, g, ws, src, dst, in_stride_pol, unit0, nunits, st);
    case 1024: return launch_fwd_L<1024>(mode, g, ws, src, dst, in_stride_pol, unit0, nunits, st);
    default: return cudaErrorInvalidValue;
    }
}

bool forward_len_supported(int L) { return L >= 16 && L <= 1024 && (L & (L - 1)) == 0; }
bool fused_len_supported(int M) { return M >= 16 && M <= 8192 && (M & (M - 1)) == 0; }

cudaError_t launch_forward(const Geometry &g, const Workspace &ws, const void *d_in, long long in_stride_pol,
                           int unit0, int nunits, float2 *spec_out, cudaStream_t st, long long *launches)
{
    cudaError_t e = launch_fwd_any(g.n1, 0, g, ws, d_in, ws.bufA, in_stride_pol, unit0, nunits, st);
    if (e != cudaSuccess) return e;
    ++*launches;
    e = launch_fwd_any(g.n2, 1, g, ws, ws.bufA, spec_out, 0, unit0, nunits, st);
    if (e != cudaSuccess) return e;
    ++*launches;
    return cudaSuccess;
}

}  // namespace cdmt
