// cdmt_internal.h -- host-side description of one execute, shared by the API and the launchers.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include <vector>

namespace cdmt {

struct Geometry {
    int nsub, nfft, noverlap, nchan, ndec, ndm, in_dtype, chirp_ref;
    double bw_mhz;
    // derived
    int step, mbin, hdisc, vdec;  // N-O, M, h, Vd
    int n1, n2;                   // four-step split nfft = n1 * n2 (n1 >= n2)
    int tw_hi_bits;               // w_N^e = hi[e >> lo_bits] * lo[e & mask]
    int lo_bits;
};

// input layouts (CDMT_IN_*): bytes of one word of a row and rows per subband
// 0 interleaved float32 (8, 2), 1 interleaved int8 (2, 2), 2 planar float32 (4, 4), 3 planar int8 (1, 4)
inline int in_word_bytes(int in_dtype) { return in_dtype == 0 ? 8 : in_dtype == 1 ? 2 : in_dtype == 2 ? 4 : 1; }
inline int in_rows_per_sub(int in_dtype) { return in_dtype >= 2 ? 4 : 2; }

// Device pointers into the workspace (all 256-byte aligned).
struct Workspace {
    double *dm;         // [ndm]
    double *fcen;       // [nsub]
    float2 *tw_n1;      // pass twiddles of the length-n1 forward transform
    float2 *tw_n2;      // ... length-n2
    float2 *tw_m;       // pass twiddles of the length-M backward transform
    float2 *tw4_lo;     // four-step twiddle tables
    float2 *tw4_hi;
    float2 *bufA;       // [chunk_units][2][nfft] after pass A
    float2 *spec;       // [chunk_units][2][nfft] shifted spectra Xs
    size_t total_bytes;
};

size_t workspace_layout(const Geometry &g, int chunk_units, char *base, Workspace *ws);

// Launchers: return cudaError_t of the launch; *launches is incremented per kernel launched.
cudaError_t launch_init_tables(const Geometry &g, const Workspace &ws, const double *h_dm,
                               const double *h_fcen, cudaStream_t st, long long *launches);
cudaError_t launch_forward(const Geometry &g, const Workspace &ws, const void *d_in,
                           long long in_stride_pol, int unit0, int nunits, float2 *spec_out,
                           cudaStream_t st, long long *launches);
// d_segsum (may be null): block sums [ndm][nblock_total][nch] x (sum I, sum I^2); *sums_done is cleared if the
// kernel chosen cannot take them (the caller then runs launch_block_sums over the finished filterbank)
cudaError_t launch_fused(const Geometry &g, const Workspace &ws, const float2 *spec, int unit0,
                         int nunits, float *d_out, long long out_stride_dm, int out_pitch, int dm_tile,
                         int accurate, int force_generic, const double *h_dm, const double *h_fcen,
                         double *d_segsum, int nblock_total, bool *sums_done,
                         cudaStream_t st, long long *launches);
cudaError_t launch_unpack(const Geometry &g, const void *d_in, long long in_stride_pol,
                          int nblock, float2 *d_blocks, cudaStream_t st, long long *launches);
cudaError_t launch_fp32_peak(float *d_scratch, int nblocks, int inner, cudaStream_t st);

// cdmt_redigitize.cu: Alg. 1 l.104-106
size_t redigitize_workspace_bytes(const Geometry &g, long long nblock);
cudaError_t launch_redigitize(const Geometry &g, const float *d_fb, long long fb_stride_dm, long long nblock,
                              double qmean, double qstd, unsigned char *d_codes, long long codes_stride_dm,
                              float *d_offset, float *d_scale, void *d_workspace, cudaStream_t st,
                              long long *launches);

// the same with the block sums in a file-scope device array of redigitize_static_max_bytes() bytes (no allocation)
size_t redigitize_static_max_bytes();
cudaError_t launch_redigitize_static(const Geometry &g, const float *d_fb, long long fb_stride_dm, long long nblock,
                                     double qmean, double qstd, unsigned char *d_codes, long long codes_stride_dm,
                                     float *d_offset, float *d_scale, cudaStream_t st, long long *launches);

cudaError_t launch_block_sums(const Geometry &g, const float *d_fb, long long fb_stride_dm, long long nblock,
                              double *d_segsum, cudaStream_t st, long long *launches);
cudaError_t launch_stats_quantize(const Geometry &g, const float *d_fb, long long fb_stride_dm, long long nblock,
                                  double qmean, double qstd, const double *d_segsum, unsigned char *d_codes,
                                  long long codes_stride_dm, float *d_offset, float *d_scale, cudaStream_t st,
                                  long long *launches);

// cdmt_incoherent.cu: incoherent dedispersion of the filterbanks over fine DM offsets
struct IncoherentTables {            // host side, owned by the plan (must outlive the async upload)
    int nfine = 0, nch = 0;
    int smin = 0, range = 0;         // extremes of the shift table: range = smax - smin
    std::vector<int> shifts;         // [nfine][nch] samples, channel order of the filterbank (descending)
    std::vector<uint2> entries;      // [ngroups][nch]: x = first trial's shift - smin, y = 2-bit increments
    std::vector<uint4> segs;         // per group: channel ranges [x, y) that share the first shift and the pattern;
                                     // z = first shift - smin | spread << 24 | closes-its-run << 28, w = 2-bit increments
    std::vector<int> seg_off;        // [ngroups + 1]: first segment of a group
    std::vector<int2> groups;        // [ngroups]: (first trial, number of trials <= 8)
    void *pinned = nullptr;          // page-locked copy of segs + seg_off + groups (made by the first dedisperse)
};
// Fills the tables; returns false if ddm is not ascending.
bool incoherent_plan(const Geometry &g, const double *h_fcen, int nfine, const double *ddm, IncoherentTables *T);
size_t incoherent_workspace_bytes(const IncoherentTables &T);
// false if the shift range or the number of trial groups is beyond what the kernel can be launched with
bool incoherent_config(const IncoherentTables &T, int *cc, int *tw, int *gpc, int *tt, size_t *smem);
void incoherent_release(IncoherentTables *T);
cudaError_t launch_incoherent(const Geometry &g, IncoherentTables &T, const float *d_fb, long long fb_stride_dm,
                              long long nt_in, float *d_ts, long long ts_stride_dm, long long ts_pitch,
                              void *d_workspace, cudaStream_t st, long long *launches);
cudaError_t launch_carry_rows(float *d_fb, long long fb_stride_dm, long long nt_in, int nrows, int nch, int ndm,
                              cudaStream_t st, long long *launches);

bool forward_len_supported(int L);
bool fused_len_supported(int M);

}  // namespace cdmt
