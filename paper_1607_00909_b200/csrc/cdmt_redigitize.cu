// cdmt_redigitize.cu -- Alg. 1 l.104-106: redigitisation of a batch of
// float32 filterbanks to 8 bit.  Three HBM-bound kernels, as in the paper:
//
//   k_block_sums     "compute block sums": sum I and sum I^2 over the Vd samples one data block
//                    contributed to a channel, for every (DM, block, channel); fp64 accumulators
//   k_channel_stats  "compute channel statistics": adds the block sums of a (DM, channel), mean and
//                    population standard deviation, then offset and scale (float32)
//   k_quantize       "redigitize": code = clip(rint((I - offset) / scale), 0, 255) in float32
//
// The filterbank is time-major, channel-fastest, so a warp reads 32 adjacent
// channel groups of one time sample: 512 contiguous bytes with float4 loads (nch % 4 == 0), 128
// bytes otherwise.  Algorithmic traffic: 4 B + 4 B read and 1 B written per filterbank sample.
#include <mutex>
#include <cstdint>

#include "cdmt_internal.h"

namespace cdmt {

template <int VEC>
struct VecLoad;
template <>
struct VecLoad<4> {
    static __device__ __forceinline__ void ld(const float *p, float (&v)[4])
    {
        const float4 q = __ldg(reinterpret_cast<const float4 *>(p));
        v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
    }
};
template <>
struct VecLoad<1> {
    static __device__ __forceinline__ void ld(const float *p, float (&v)[1]) { v[0] = __ldg(p); }
};

constexpr int BS_TX = 32, BS_TY = 8;  // block-sum CTA: 32 channel groups x 8 row slices

// grid (ceil(ngroups / 32), nblock, ndm); segsum[(d nblock + b) nch + c] = (sum I, sum I^2)
template <int VEC>
__global__ void __launch_bounds__(BS_TX *BS_TY)
k_block_sums(const float *__restrict__ fb, long long fb_stride_dm, int vd, int nch, double2 *__restrict__ segsum)
{
    __shared__ double sh[BS_TY][BS_TX][2 * VEC];
    const int g = blockIdx.x * BS_TX + threadIdx.x;  // channel group
    const int b = blockIdx.y, d = blockIdx.z;
    const int ngroups = nch / VEC;
    double s1[VEC], s2[VEC];
#pragma unroll
    for (int k = 0; k < VEC; ++k) s1[k] = s2[k] = 0.0;
    if (g < ngroups) {
        const float *p = fb + (size_t)d * (size_t)fb_stride_dm + ((size_t)b * vd) * nch + (size_t)g * VEC;
#pragma unroll 4
        for (int q = threadIdx.y; q < vd; q += BS_TY) {
            float v[VEC];
            VecLoad<VEC>::ld(p + (size_t)q * nch, v);
#pragma unroll
            for (int k = 0; k < VEC; ++k) {
                const double x = (double)v[k];
                s1[k] += x;
                s2[k] = fma(x, x, s2[k]);
            }
        }
    }
#pragma unroll
    for (int k = 0; k < VEC; ++k) {
        sh[threadIdx.y][threadIdx.x][2 * k] = s1[k];
        sh[threadIdx.y][threadIdx.x][2 * k + 1] = s2[k];
    }
    __syncthreads();
    if (threadIdx.y == 0 && g < ngroups) {
#pragma unroll
        for (int k = 0; k < VEC; ++k) {
            double a = 0.0, c = 0.0;
#pragma unroll
            for (int y = 0; y < BS_TY; ++y) {
                a += sh[y][threadIdx.x][2 * k];
                c += sh[y][threadIdx.x][2 * k + 1];
            }
            segsum[((size_t)d * gridDim.y + b) * nch + (size_t)g * VEC + k] = make_double2(a, c);
        }
    }
}

// one thread per (DM, channel)
__global__ void k_channel_stats(const double2 *__restrict__ segsum, int nblock, int nch, int ndm, double nsamples,
                                double qmean, double qstd, float *__restrict__ offset, float *__restrict__ scale)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)ndm * nch) return;
    const int d = (int)(i / nch), c = (int)(i % nch);
    double tot = 0.0, tot2 = 0.0;
    for (int b = 0; b < nblock; ++b) {
        const double2 s = segsum[((size_t)d * nblock + b) * nch + c];
        tot += s.x;
        tot2 += s.y;
    }
    // explicit roundings: no fused multiply-add in the statistics
    const double mu = __ddiv_rn(tot, nsamples);
    double var = __dsub_rn(__ddiv_rn(tot2, nsamples), __dmul_rn(mu, mu));
    if (var < 0.0) var = 0.0;
    const double sd = sqrt(var);
    const double sc = sd > 0.0 ? __ddiv_rn(sd, qstd) : 1.0;
    scale[i] = (float)sc;
    offset[i] = (float)__dsub_rn(mu, __dmul_rn(qmean, sc));
}

__device__ __forceinline__ unsigned quantize_one(float x, float off, float sc)
{
    const float q = rintf(__fdiv_rn(__fsub_rn(x, off), sc));  // round half to even
    return (unsigned)fminf(fmaxf(q, 0.0f), 255.0f);           // NaN -> 0
}

constexpr int QZ_ROWS = 16;  // time samples per thread

// grid (ceil(ngroups / 128), ceil(nt / QZ_ROWS), ndm), 128 threads
template <int VEC>
__global__ void __launch_bounds__(128)
k_quantize(const float *__restrict__ fb, long long fb_stride_dm, int nt, int nch, const float *__restrict__ offset,
           const float *__restrict__ scale, unsigned char *__restrict__ codes, long long codes_stride_dm)
{
    const int g = blockIdx.x * 128 + threadIdx.x;
    if (g >= nch / VEC) return;
    const int d = blockIdx.z;
    const int t0 = blockIdx.y * QZ_ROWS;
    float off[VEC], sc[VEC];
    VecLoad<VEC>::ld(offset + (size_t)d * nch + (size_t)g * VEC, off);
    VecLoad<VEC>::ld(scale + (size_t)d * nch + (size_t)g * VEC, sc);
    const float *p = fb + (size_t)d * (size_t)fb_stride_dm + (size_t)g * VEC;
    unsigned char *o = codes + (size_t)d * (size_t)codes_stride_dm + (size_t)g * VEC;
#pragma unroll 4
    for (int r = 0; r < QZ_ROWS; ++r) {
        const int t = t0 + r;
        if (t >= nt) break;
        float v[VEC];
        VecLoad<VEC>::ld(p + (size_t)t * nch, v);
        if (VEC == 4) {
            const unsigned w = quantize_one(v[0], off[0], sc[0]) | (quantize_one(v[1 % VEC], off[1 % VEC], sc[1 % VEC]) << 8) |
                               (quantize_one(v[2 % VEC], off[2 % VEC], sc[2 % VEC]) << 16) |
                               (quantize_one(v[3 % VEC], off[3 % VEC], sc[3 % VEC]) << 24);
            *reinterpret_cast<unsigned *>(o + (size_t)t * nch) = w;
        } else {
            o[(size_t)t * nch] = (unsigned char)quantize_one(v[0], off[0], sc[0]);
        }
    }
}

size_t redigitize_workspace_bytes(const Geometry &g, long long nblock)
{
    return sizeof(double2) * (size_t)g.ndm * (size_t)nblock * (size_t)g.nsub * g.nchan;
}

// float4 / 32-bit paths need 16-byte (4-byte) aligned rows
static bool fb_vec4(int nch, const float *d_fb, long long fb_stride_dm)
{
    return nch % 4 == 0 && fb_stride_dm % 4 == 0 && (reinterpret_cast<uintptr_t>(d_fb) & 15) == 0;
}

// l.104 as a stand-alone pass over the filterbank (the packed fused kernels take the sums themselves)
cudaError_t launch_block_sums(const Geometry &g, const float *d_fb, long long fb_stride_dm, long long nblock,
                              double *d_segsum, cudaStream_t st, long long *launches)
{
    const int nch = g.nsub * g.nchan, vd = g.vdec;
    double2 *segsum = reinterpret_cast<double2 *>(d_segsum);
    const bool vec4 = fb_vec4(nch, d_fb, fb_stride_dm);
    const int ngroups = vec4 ? nch / 4 : nch;
    dim3 grid((unsigned)((ngroups + BS_TX - 1) / BS_TX), (unsigned)nblock, (unsigned)g.ndm), block(BS_TX, BS_TY);
    if (vec4)
        k_block_sums<4><<<grid, block, 0, st>>>(d_fb, fb_stride_dm, vd, nch, segsum);
    else
        k_block_sums<1><<<grid, block, 0, st>>>(d_fb, fb_stride_dm, vd, nch, segsum);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) ++*launches;
    return e;
}

// l.105-106 from given block sums
cudaError_t launch_stats_quantize(const Geometry &g, const float *d_fb, long long fb_stride_dm, long long nblock,
                                  double qmean, double qstd, const double *d_segsum, unsigned char *d_codes,
                                  long long codes_stride_dm, float *d_offset, float *d_scale, cudaStream_t st,
                                  long long *launches)
{
    const int nch = g.nsub * g.nchan, vd = g.vdec;
    const long long nt = nblock * vd;
    const double2 *segsum = reinterpret_cast<const double2 *>(d_segsum);
    const bool vec4 = fb_vec4(nch, d_fb, fb_stride_dm) && codes_stride_dm % 4 == 0 &&
                      (reinterpret_cast<uintptr_t>(d_codes) & 3) == 0 &&
                      (reinterpret_cast<uintptr_t>(d_offset) & 15) == 0 && (reinterpret_cast<uintptr_t>(d_scale) & 15) == 0;
    const int ngroups = vec4 ? nch / 4 : nch;
    {
        const long long n = (long long)g.ndm * nch;
        k_channel_stats<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(segsum, (int)nblock, nch, g.ndm, (double)nt, qmean,
                                                                      qstd, d_offset, d_scale);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        ++*launches;
    }
    {
        dim3 grid((unsigned)((ngroups + 127) / 128), (unsigned)((nt + QZ_ROWS - 1) / QZ_ROWS), (unsigned)g.ndm);
        if (vec4)
            k_quantize<4><<<grid, 128, 0, st>>>(d_fb, fb_stride_dm, (int)nt, nch, d_offset, d_scale, d_codes, codes_stride_dm);
        else
            k_quantize<1><<<grid, 128, 0, st>>>(d_fb, fb_stride_dm, (int)nt, nch, d_offset, d_scale, d_codes, codes_stride_dm);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        ++*launches;
    }
    return cudaSuccess;
}

cudaError_t launch_redigitize(const Geometry &g, const float *d_fb, long long fb_stride_dm, long long nblock,
                              double qmean, double qstd, unsigned char *d_codes, long long codes_stride_dm,
                              float *d_offset, float *d_scale, void *d_workspace, cudaStream_t st, long long *launches)
{
    double *segsum = reinterpret_cast<double *>(d_workspace);
    cudaError_t e = launch_block_sums(g, d_fb, fb_stride_dm, nblock, segsum, st, launches);
    if (e != cudaSuccess) return e;
    return launch_stats_quantize(g, d_fb, fb_stride_dm, nblock, qmean, qstd, segsum, d_codes, codes_stride_dm, d_offset,
                                 d_scale, st, launches);
}

// ------------------------------------------------------------------------------------------------
// cdmt_redigitize_static: the same three kernels with the block sums in memory the LIBRARY holds, for
// callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc).  The scratch is a file-scope device array of a fixed, modest size: every GPU that
// loads the library keeps these 4 MiB until the process exits.
//
//  * In host code `g_redig_scratch` is only a stand-in for the symbol, NOT a device address: the device
//    address is looked up with cudaGetSymbolAddress, once per device, with that device current, and it
//    is that pointer the kernels are given.
//  * All calls on a device share the array.  It keeps the last call's contents, but nothing has to start
//    at zero: k_block_sums overwrites every (DM, block, channel) entry that k_channel_stats of the same
//    call reads.  Calls that overlap on the GPU (two streams, two plans, two host threads) race on it:
//    the caller must order them (one stream, or events).
//  * No cudaMalloc, cudaFree, cudaMallocHost or other allocating routine is called.
// ------------------------------------------------------------------------------------------------
constexpr size_t REDIG_STATIC_BYTES = (size_t)4 << 20;                       // 262144 (DM, block, channel) entries
static __device__ __align__(256) unsigned char g_redig_scratch[REDIG_STATIC_BYTES];

constexpr int REDIG_MAX_DEVICES = 64;
static void *g_redig_scratch_addr[REDIG_MAX_DEVICES];   // device address of the array, per device ordinal
static std::mutex g_redig_scratch_mutex;

size_t redigitize_static_max_bytes() { return REDIG_STATIC_BYTES; }

// device address of this device's copy of the scratch array (looked up on first use, then remembered)
static cudaError_t redig_scratch_on_current_device(void **ptr)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= REDIG_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_redig_scratch_mutex);
    if (!g_redig_scratch_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_redig_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_redig_scratch_addr[dev] = p;
    }
    *ptr = g_redig_scratch_addr[dev];
    return cudaSuccess;
}

// The caller (cdmt_api.cu) has checked redigitize_workspace_bytes(g, nblock) <= redigitize_static_max_bytes().
cudaError_t launch_redigitize_static(const Geometry &g, const float *d_fb, long long fb_stride_dm, long long nblock,
                                     double qmean, double qstd, unsigned char *d_codes, long long codes_stride_dm,
                                     float *d_offset, float *d_scale, cudaStream_t st, long long *launches)
{
    if (redigitize_workspace_bytes(g, nblock) > REDIG_STATIC_BYTES) return cudaErrorInvalidValue;
    void *scratch = nullptr;
    cudaError_t e = redig_scratch_on_current_device(&scratch);
    if (e != cudaSuccess) return e;
    return launch_redigitize(g, d_fb, fb_stride_dm, nblock, qmean, qstd, d_codes, codes_stride_dm, d_offset, d_scale,
                             scratch, st, launches);
}

}  // namespace cdmt
