// cdmt_fused_common.cuh -- argument blocks and small device helpers shared by the fused per-DM
// kernels (cdmt_fused.cu: scalar kernels; cdmt_fused2.cu: packed-FP32 + TMEM kernel).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cdmt {

template <bool ACCURATE>
__device__ __forceinline__ float2 unit_phasor(float frac_cycles)
{
    float s, c;
    if (ACCURATE) {
        sincospif(2.0f * frac_cycles, &s, &c);
    } else {
        const float x = frac_cycles * 6.283185307179586f;
        s = __sinf(x);
        c = __cosf(x);
    }
    return make_float2(c, s);
}

__device__ __forceinline__ float2 unit_phasor_rt(float frac_cycles, int accurate)
{
    return accurate ? unit_phasor<true>(frac_cycles) : unit_phasor<false>(frac_cycles);
}

// fractional part in [-0.5, 0.5] of dm * g, exact to fp64 rounding
__device__ __forceinline__ float frac_cycles(double dm, double g)
{
    const double magic = 6755399441055744.0;  // 1.5 * 2^52: adding it rounds to the nearest integer
    const double n = fma(dm, g, magic) - magic;
    return (float)fma(dm, g, -n);
}

constexpr int DM_PARAM_MAX = 1024;  // DM trials carried in the kernel parameter block (constant bank)

struct DmParams {
    double dm[DM_PARAM_MAX];
};

struct FusedArgs {
    const float2 *spec;      // [units][2][nfft] swapped-halves spectra of this chunk
    const float2 *tw;        // pass twiddles of the length-M backward transform
    const double *dmlist;
    const double *fcen;
    float *out;
    long long out_stride_dm;
    int out_pitch;           // elements between consecutive time samples of `out` (>= nsub * nchan)
    int unit0, nsub, nchan, nfft, hdisc, ndec, vdec, ndm, dm_tile, chirp_ref, accurate;
    int dm_first, dm_param0;  // DM range [dm_first, ndm) of this launch; dmp.dm[0] is trial dm_param0
    int nb_chunk;             // k_fused_ws: whole blocks in this chunk (units = nb_chunk * nsub)
    int cta0;                 // k_fused_ws: blockIdx.x of this launch starts at CTA cta0 of the chunk
    double2 *segsum;          // block sums [ndm][nblock_total][nsub nchan] of (I, I^2) (Alg. 1 l.104), or null
    int nblock_total;         // blocks of this execute (second dimension of segsum)
    double bw_mhz;
    float scale;
};

// frequency set-up shared by both kernels: nu_0 of Eq. 1 and the offset of bin m (MHz)
__device__ __forceinline__ void chirp_axes(const FusedArgs &a, int s, int c, int M, double *f0, double *f_bin0,
                                           double *df)
{
    const double fc = a.fcen[s];
    *df = a.bw_mhz / (double)a.nfft;
    if (a.chirp_ref == 0) {
        *f0 = fc + ((double)c + 0.5 - 0.5 * (double)a.nchan) * a.bw_mhz / (double)a.nchan;
        *f_bin0 = -(double)(M / 2) * *df;
    } else {
        *f0 = fc;
        *f_bin0 = (double)(c * M - a.nfft / 2) * *df;
    }
}

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(
                     (unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}" ::"r"((unsigned)__cvta_generic_to_shared(bar)),
        "r"(parity)
        : "memory");
}

// reduce-scatter over 2^LOGD adjacent lanes: in[n], n < 16, becomes out[j] = sum over the lane
// group of slot n = (lane & (D-1)) + D j
template <int LOGD, int S = 0>
__device__ __forceinline__ void lane_reduce_scatter(float *a, int lane)
{
    if constexpr (S < LOGD) {
        constexpr int cnt = 16 >> S;  // values held before this stage
        const bool up = (lane >> S) & 1;
#pragma unroll
        for (int j = 0; j < cnt / 2; ++j) {
            const float lo = a[2 * j], hi = a[2 * j + 1];
            const float send = up ? lo : hi;
            const float keep = up ? hi : lo;
            a[j] = keep + __shfl_xor_sync(0xffffffffu, send, 1 << S);
        }
        lane_reduce_scatter<LOGD, S + 1>(a, lane);
    }
}

// Block sums of Alg. 1 l.104 inside a packed fused kernel: every thread adds the float32 values it has
// just stored (sum and sum of squares, fp64), the warp reduces them by shuffles and lane 0 leaves the
// warp's pair in shared memory; one thread adds the warps' pairs later (see the kernels).
__device__ __forceinline__ void warp_sum_pair(double &a, double &q)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, off);
        q += __shfl_xor_sync(0xffffffffu, q, off);
    }
}

// cdmt_fused2.cu
bool fused_x2_supported(int M, int ndec, int hdisc);
cudaError_t launch_fused_x2(int M, int logd, const FusedArgs &fa, const double *h_dm, int nunits, cudaStream_t st,
                            long long *launches);
// cdmt_fused5.cu
bool fused_ws_supported(int M, int ndec, int hdisc, int nsub, int unit0, int nunits);
cudaError_t launch_fused_ws(int M, int logd, const FusedArgs &fa, const double *h_dm, int nunits, cudaStream_t st,
                            long long *launches);

// cdmt_fused4.cu
bool fused_sp_supported(int M, int ndec, int hdisc);
cudaError_t launch_fused_sp(int M, int logd, const FusedArgs &fa, const double *h_dm, int nunits, cudaStream_t st,
                            long long *launches);

}  // namespace cdmt
