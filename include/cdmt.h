/*
 * cdmt.h -- C ABI of the B200-native coherent-dedispersion hot path
 * (Bassa, Pleunis & Hessels, arXiv:1607.00909, "cdmt"; line numbers below are PAPER.md).
 *
 * What the library computes (Fig. 2; Algorithm 1), for every
 * subband s < nsub, overlap-save block b < nblock, channel c < nchan and DM trial d < ndm:
 *
 *   step = nfft - noverlap, M = nfft/nchan, h = noverlap/(2 nchan), Vd = (M - 2h)/ndec
 *   u_p[n]  = in[s][p][b step + n],                 n < nfft, p < 2       (l.95)
 *   U_p[k]  = sum_n u_p[n] exp(-2 pi i k n / nfft)                         (l.96)
 *   Xs_p[j] = U_p[(j + nfft/2) mod nfft]            bins in increasing frequency   (l.97)
 *   Z_p[m]  = Xs_p[c M + m] exp(+2 pi i dm[d] f^2 / (2.41e-10 f0^2 (f0 + f)))   (l.99; Eq. 1)
 *             f0, f in MHz: CDMT_REF_CHANNEL f0 = centre of channel c, f = (m - M/2) bw/nfft
 *                           CDMT_REF_SUBBAND f0 = fcen[s], f = (c M + m - nfft/2) bw/nfft
 *   y_p[t]  = sum_m Z_p[m] exp(+2 pi i (m - M/2) t / M),  t < M            (l.101-102)
 *   I[t]    = (|y_0[t]|^2 + |y_1[t]|^2) / (nfft M)                         (l.103)
 *   out[d][b Vd + q][nsub nchan - 1 - (s nchan + c)] = sum_{r<ndec} I[h + q ndec + r]
 *
 * i.e. one float32 filterbank per DM, time-major, channel-fastest, DECREASING frequency
 * (PAPER.md:123).  Blocks are "valid only": nblock = floor((nsamp - nfft)/step) + 1, the first
 * output sample starts at input sample noverlap/2, trailing samples that do not fill a block
 * are ignored.
 *
 * Conventions
 *  - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  The caller owns all of
 *    them; the library never allocates device memory.  A plan owns host state, plus -- created
 *    lazily, destroyed with the plan -- the CUDA events of CDMT_OPT_PROFILE and the two copy
 *    streams and ordering events of the host-buffer path.
 *  - Every entry point returns a CDMT_* status and never aborts or throws.  All arguments
 *    are validated on the host before anything is launched.
 *  - cdmt_execute and the stage calls are asynchronous on `cuda_stream` (a cudaStream_t
 *    passed as void*; NULL = the legacy default stream) and do no host synchronisation.
 *    They are stateless between calls; one call may be in flight per (plan, workspace).
 */
#ifndef CDMT_H
#define CDMT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cdmt_plan cdmt_plan; /* opaque */

enum {
    CDMT_OK = 0,
    CDMT_ERR_ARG = 1,       /* null / misaligned pointer, non-finite or non-positive value */
    CDMT_ERR_SIZE = 2,      /* sizes violate a divisibility / range rule listed below */
    CDMT_ERR_WORKSPACE = 3, /* workspace_bytes smaller than cdmt_plan_query reports */
    CDMT_ERR_CUDA = 4,      /* a CUDA call or launch failed (sticky error cleared) */
    CDMT_ERR_ALLOC = 5      /* host allocation failed */
};

/* Input layouts.  Interleaved: a row holds complex words (re, im), rows (s, p) = (subband, polarisation).
 * Planar ("two cufftComplex arrays, one for each polarization" upstream of the unpack step;
 * telescope back ends write the four real streams Xre, Xim, Yre, Yim separately): a row holds real
 * words, rows (s, p, part) with part 0 = re, 1 = im.  Row r of subband s starts at element
 * (rows_per_subband s + r) * in_stride_pol of its word type; in_stride_pol counts words of a row. */
enum { CDMT_IN_CF32 = 0, CDMT_IN_CI8 = 1, CDMT_IN_PF32 = 2, CDMT_IN_PI8 = 3 };
enum { CDMT_REF_CHANNEL = 0, CDMT_REF_SUBBAND = 1 }; /* nu_0 of Eq. 1 */

/* Tuning knobs for cdmt_plan_set_option (defaults chosen by the library). */
enum {
    CDMT_OPT_CHUNK_UNITS = 0, /* (subband, block) units whose spectra are resident at once (0 = about 4 GiB of
                                 spectra, a whole and even number of blocks; the workspace holds twice that) */
    CDMT_OPT_DM_TILE = 1,     /* DM trials looped inside one CTA of the fused kernel (0 = all) */
    CDMT_OPT_ACCURATE_SINCOS = 2, /* 1: sincospif instead of the fast approximation */
    CDMT_OPT_PROFILE = 3,     /* 1: record CUDA events round each kernel class (cdmt_profile_read) */
    CDMT_OPT_FUSED_KERNEL = 4, /* fused per-DM kernel: 0 = best applicable (default), 1 = general kernel (any ndec /
                                  overlap), 2 = scalar fast kernel, 3 = packed-FP32 + tensor-memory kernel with the
                                  even/odd half transforms in the register lanes (k_fused_x2), 4 = the same
                                  arithmetic warp-specialised: two blocks per CTA share a chirp that dedicated
                                  warps form and hand over through tensor memory (k_fused_ws; nfft/nchan = 4096),
                                  5 = packed kernel with the two polarisations in the lanes, chirp of the next
                                  trial formed in the shadow of the block barrier (k_fused_sp); 2 to 5 make
                                  cdmt_execute fail with CDMT_ERR_CUDA where they do not apply */
    CDMT_OPT_FORCE_GENERIC = 4, /* older name of the same key (value 1) */
    CDMT_OPT_HOST_GROUP_BLOCKS = 5, /* cdmt_execute_host: blocks staged per group (0 = about 1 GiB of output, an even number) */
    CDMT_OPT_KEEP_TABLES = 6  /* 1: the caller promises that nothing but this plan's executes writes to
                                 d_workspace between calls that pass the same workspace pointer; the DM list,
                                 centre frequencies and twiddle tables at its head are then written by the
                                 first such execute only (default 0: every execute rewrites them with one
                                 extra small launch).  Setting the option (to either value) forgets the
                                 remembered workspace. */
};

enum { CDMT_OUT_F32 = 0, CDMT_OUT_U8 = 1 };           /* host path: float32 filterbanks / redigitised to 8 bit */

/*
 * Create a plan ("user-defined choices" n_c, N_bin, n_d and the DM list).
 *   nsub      number of subbands (>= 1)
 *   fcen_mhz  HOST [nsub] subband centre frequencies in MHz, ascending; copied
 *   bw_mhz    subband bandwidth = complex sample rate, MHz (> 0; fcen - bw/2 > 0)
 *   nfft      N_bin, power of two, 256 <= nfft <= 2^20
 *   noverlap  n_d n_c in INPUT samples: 0 <= noverlap < nfft, noverlap % (2 nchan) == 0
 *   nchan     n_c, power of two, 16 <= nfft/nchan <= 8192
 *   ndec      time-integration factor >= 1, (nfft - noverlap) % (nchan ndec) == 0
 *   ndm, dm   HOST [ndm] DM trials in pc cm^-3 (any sign: -DM applies the conjugate chirp); copied
 *   in_dtype  CDMT_IN_*; chirp_ref CDMT_REF_*
 * Errors: CDMT_ERR_ARG, CDMT_ERR_SIZE, CDMT_ERR_ALLOC.  *plan is NULL on error.
 * Pure host code: works without a GPU.
 */
int cdmt_plan_create(cdmt_plan **plan, int nsub, const double *fcen_mhz, double bw_mhz,
                     int nfft, int noverlap, int nchan, int ndec, int ndm, const double *dm,
                     int in_dtype, int chirp_ref);

int cdmt_plan_destroy(cdmt_plan *plan);

/* Set a CDMT_OPT_* knob; CDMT_ERR_ARG for an unknown key or out-of-range value. */
int cdmt_plan_set_option(cdmt_plan *plan, int key, long long value);

/*
 * Sizes for an input of `nsamp` samples per polarisation per subband (host arithmetic only;
 * PAPER.md:81, 123).  Any output pointer may be NULL.
 *   nblock          blocks processed
 *   nsamp_consumed  (nblock-1) step + nfft: samples actually read
 *   nout_per_chan   nblock * Vd output time samples per channel per DM
 *   out_bytes       ndm * nout_per_chan * nsub*nchan * 4 (dense DM planes)
 *   workspace_bytes bytes cdmt_execute needs in d_workspace
 * Errors: CDMT_ERR_ARG (null plan), CDMT_ERR_SIZE (nsamp < nfft).
 */
int cdmt_plan_query(const cdmt_plan *plan, long long nsamp, int *nblock,
                    long long *nsamp_consumed, long long *nout_per_chan, size_t *out_bytes,
                    size_t *workspace_bytes);

/*
 * Run the whole hot path on device-resident input.
 *   d_in           DEVICE, [nsub][2 pols][..] complex words (interleaved layouts) or
 *                  [nsub][2 pols][re, im][..] real words (planar layouts) of the plan's in_dtype, time
 *                  fastest; consecutive rows are in_stride_pol words apart.  Aligned to one word
 *                  (8 / 2 / 4 / 1 bytes for CF32 / CI8 / PF32 / PI8); the int8 layouts are read with
 *                  16-byte loads when the pointer, the row stride, the block step and the pass
 *                  length are multiples of 16 bytes, else word by word.
 *   nsamp          samples per row to process (>= nfft)
 *   in_stride_pol  distance between consecutive rows, in words of a row (>= nsamp)
 *   d_out          DEVICE float32, DM plane d starts at d * out_stride_dm elements; inside a
 *                  plane [nblock*Vd][nsub*nchan].  Every element of every plane is written.
 *   out_stride_dm  elements between DM planes (>= nblock*Vd*nsub*nchan)
 *   d_workspace    DEVICE scratch, 256-byte aligned, >= workspace_bytes from cdmt_plan_query
 *   cuda_stream    cudaStream_t
 * To stream a long observation call repeatedly, advancing d_in by nblock*step samples (the
 * last noverlap samples are re-supplied).
 * Errors: CDMT_ERR_ARG, CDMT_ERR_SIZE, CDMT_ERR_WORKSPACE, CDMT_ERR_CUDA.
 */
int cdmt_execute(cdmt_plan *plan, const void *d_in, long long nsamp, long long in_stride_pol,
                 float *d_out, long long out_stride_dm, void *d_workspace,
                 size_t workspace_bytes, void *cuda_stream);

/*
 * cdmt_execute that also returns the "block sums" of Alg. 1 l.104:
 *   d_segsum   DEVICE fp64 [ndm][nblock][nsub*nchan][2] = (sum I, sum I^2) over the Vd float32
 *              samples that block b gave channel j (output order) at trial d; dense;
 *              cdmt_redigitize_workspace_bytes() bytes, 16-byte aligned.
 * The warp-specialised fused kernel (nfft/nchan = 4096, ndec 8, 16 or 32) takes the sums from the
 * values it is about to store -- each CTA owns whole segments, and its chirp warps have the time --
 * so the filterbank is not read back for them; for every other shape the sums come from a separate
 * pass over d_out (on this hardware cheaper than fp64 sums inside an ALU-bound kernel).  Feed them
 * to cdmt_redigitize_sums.  Same errors as cdmt_execute.
 */
int cdmt_execute_sums(cdmt_plan *plan, const void *d_in, long long nsamp, long long in_stride_pol,
                      float *d_out, long long out_stride_dm, double *d_segsum, void *d_workspace,
                      size_t workspace_bytes, void *cuda_stream);

/*
 * The same path with HOST buffers (read block, copy to device, ...,
 * redigitize, copy to host).  The observation is staged through device scratch in groups of
 * blocks, input and output double-buffered (the transfers, not the kernels, are the
 * paper's bottleneck).  Kernels run on `cuda_stream`; the host-to-device copy of the next group
 * and the device-to-host copy of the previous one run meanwhile on two streams the plan creates on
 * first use (ordered after the work already queued on `cuda_stream`).
 *
 * cdmt_execute_host_async only queues work: it returns at once, and `cuda_stream` is made to wait
 * for both copy streams at the end, so the results are complete when the work queued on
 * `cuda_stream` is (synchronise it, or record an event on it).  The host buffers and d_scratch
 * must stay untouched until then.
 *   h_in        HOST, layout of d_in (cdmt_execute); pinned memory for full copy speed
 *   out_kind    CDMT_OUT_F32: h_out is float32 [ndm][nblock*Vd][nsub*nchan] (dense planes), the
 *               output of cdmt_execute; h_offset / h_scale / qmean / qstd are ignored.
 *               CDMT_OUT_U8 (Alg. 1 l.104-108): h_out is uint8 with the same shape, redigitised
 *               group by group -- the batch whose statistics are taken is the
 *               group of blocks staged together -- with the mapping of cdmt_redigitize;
 *               h_offset / h_scale are float32 [ngroups][ndm][nsub*nchan].
 *   d_scratch   DEVICE, 256-byte aligned, >= scratch_bytes of cdmt_host_layout for this out_kind
 * cdmt_host_layout (host arithmetic; any output pointer may be NULL): device scratch needed, the
 * number of groups and blocks per group (the last group may be shorter), and the bytes one call
 * copies host-to-device (each group re-sends the noverlap samples it shares with the previous
 * one) and device-to-host.
 * cdmt_execute_host = cdmt_execute_host_async(CDMT_OUT_F32) followed by a wait on all three
 * streams; cdmt_host_scratch_bytes / cdmt_host_traffic_bytes = cdmt_host_layout(CDMT_OUT_F32).
 * Errors: CDMT_ERR_ARG, CDMT_ERR_SIZE, CDMT_ERR_WORKSPACE (scratch too small), CDMT_ERR_CUDA.
 */
int cdmt_execute_host_async(cdmt_plan *plan, const void *h_in, long long nsamp, long long in_stride_pol,
                            int out_kind, void *h_out, float *h_offset, float *h_scale, double qmean,
                            double qstd, void *d_scratch, size_t scratch_bytes, void *cuda_stream);
int cdmt_host_layout(const cdmt_plan *plan, long long nsamp, int out_kind, size_t *scratch_bytes,
                     int *ngroups, int *group_blocks, size_t *h2d_bytes, size_t *d2h_bytes);
int cdmt_execute_host(cdmt_plan *plan, const void *h_in, long long nsamp,
                      long long in_stride_pol, float *h_out, void *d_scratch,
                      size_t scratch_bytes, void *cuda_stream);
int cdmt_host_scratch_bytes(const cdmt_plan *plan, long long nsamp, size_t *scratch_bytes);
int cdmt_host_traffic_bytes(const cdmt_plan *plan, long long nsamp, size_t *h2d_bytes, size_t *d2h_bytes);

/*
 * Stage entry points (used by the per-kernel parity tests; same validation rules).
 *
 * cdmt_unpack: Alg. 1 l.95 "unpack, segment and pad": writes the overlapped
 * blocks as float32 complex, d_blocks[(b nsub + s)][p][nfft].
 *
 * cdmt_forward_spectrum: l.95-97: unpack + forward FFT + swap halves; d_spec[(b nsub + s)][p][nfft]
 * holds Xs_p[j] (float32 complex, increasing frequency).  Needs the same workspace as cdmt_execute.
 */
int cdmt_unpack(cdmt_plan *plan, const void *d_in, long long nsamp, long long in_stride_pol,
                void *d_blocks, void *cuda_stream);
int cdmt_forward_spectrum(cdmt_plan *plan, const void *d_in, long long nsamp,
                          long long in_stride_pol, void *d_spec, void *d_workspace,
                          size_t workspace_bytes, void *cuda_stream);

/*
 * Redigitisation of one batch of filterbanks to 8 bit: Alg. 1 l.104-106 "compute block sums",
 * "compute channel statistics", "redigitize".
 *   d_fb          DEVICE float32, the output of cdmt_execute for `nblock` blocks: DM plane d at
 *                 d * fb_stride_dm elements, [nblock*Vd][nsub*nchan] inside a plane.  Read only.
 *   nblock        blocks in the batch (>= 1); statistics are taken per DM trial and per channel
 *                 over the nblock*Vd samples of the batch
 *   qmean, qstd   mean and standard deviation the codes of a channel shall have (qstd > 0).  The
 *                 paper does not print its mapping; this library uses
 *                     scale = std / qstd (1 if std == 0),  offset = mean - qmean * scale,
 *                     code  = clip(rint((I - offset) / scale), 0, 255)
 *                 with mean and population std from the per-block sums of I and I^2 (fp64), offset
 *                 and scale rounded to float32, and the decision taken in float32 (IEEE subtract
 *                 and divide, round half to even).
 *   d_codes       DEVICE uint8, plane d at d * codes_stride_dm bytes, same [time][channel] order
 *   d_offset, d_scale   DEVICE float32 [ndm][nsub*nchan] (dense), written
 *   d_workspace   DEVICE scratch, 256-byte aligned, >= cdmt_redigitize_workspace_bytes():
 *                 the block sums [ndm][nblock][nsub*nchan] x (sum I, sum I^2) in fp64
 *   cuda_stream   cudaStream_t; three kernels are queued, nothing is synchronised
 * Errors: CDMT_ERR_ARG (null / misaligned pointer, qstd <= 0), CDMT_ERR_SIZE (nblock < 1, stride
 * shorter than a plane), CDMT_ERR_WORKSPACE, CDMT_ERR_CUDA.
 */
int cdmt_redigitize(cdmt_plan *plan, const float *d_fb, long long fb_stride_dm, long long nblock,
                    double qmean, double qstd, unsigned char *d_codes, long long codes_stride_dm,
                    float *d_offset, float *d_scale, void *d_workspace, size_t workspace_bytes,
                    void *cuda_stream);
int cdmt_redigitize_workspace_bytes(const cdmt_plan *plan, long long nblock, size_t *workspace_bytes);
/*
 * cdmt_redigitize for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): same arguments, results and kernels, but no
 * workspace -- the block sums go to a fixed scratch array inside the library (a file-scope device array
 * of cdmt_redigitize_static_max_bytes() = 4 MiB, which every GPU that loads the library holds until
 * the process exits).  The call allocates nothing (no cudaMalloc / cudaFree / pinned memory).
 *   Limit: ndm * nblock * nsub*nchan * 16 bytes <= 4 MiB, i.e. at most 262144 (DM, block, channel)
 *   triples per call; a larger batch returns CDMT_ERR_WORKSPACE ("workspace too small") before anything
 *   is launched -- split it into groups of blocks, or use cdmt_redigitize with your own workspace.
 *   Sharing: all calls on a device use the one array.  Nothing in it needs to start at zero (the first
 *   kernel overwrites every entry the second reads), but two calls that overlap on the GPU -- other
 *   streams, other plans, other host threads -- race on it: order them on one stream or with events.
 *   The array's device address is looked up once per device, with the caller's current device.
 * Errors: as cdmt_redigitize, without the workspace-pointer checks.
 */
int cdmt_redigitize_static(cdmt_plan *plan, const float *d_fb, long long fb_stride_dm, long long nblock,
                           double qmean, double qstd, unsigned char *d_codes, long long codes_stride_dm,
                           float *d_offset, float *d_scale, void *cuda_stream);
int cdmt_redigitize_static_max_bytes(size_t *max_bytes);
/* Alg. 1 l.105-106 only, from block sums already taken (cdmt_execute_sums): reads the filterbank once
 * (4 bytes read, 1 byte written per sample).  d_segsum as in cdmt_execute_sums; two kernels. */
int cdmt_redigitize_sums(cdmt_plan *plan, const float *d_fb, long long fb_stride_dm, long long nblock,
                         double qmean, double qstd, const double *d_segsum, unsigned char *d_codes,
                         long long codes_stride_dm, float *d_offset, float *d_scale, void *cuda_stream);

/*
 * Incoherent dedispersion of the coherently dedispersed filterbanks over a grid of fine DM offsets:
 * the second stage of the semi-coherent search ("each of the coherently
 * dedispersed filterbanks was then incoherently dedispersed at steps of 0.002 pc cm^-3 ranging
 * from -0.5 to 0.5 pc cm^-3 around the coherently dedispersed DM ... brute force dedispersion").
 * With f_j the centre of filterbank channel j (descending order, f_0 the highest) and tsamp =
 * nchan * ndec / bw the filterbank sample time,
 *     shift[k][j] = rint(ddm[k] * (f_j^-2 - f_0^-2) / 2.41e-4 / tsamp)          (Eq. 2; fp64, half to even)
 *     ts[d][k][t] = sum_j fb[d][t + shift[k][j] - shift_min][j],  t < nt_out = nt_in - shift_range
 * (valid-only: output sample t is time t - shift_min of the highest channel).  The same offsets are
 * applied to every coherent DM plane d.
 *   nfine, ddm     HOST [nfine] DM offsets in pc cm^-3, strictly ascending; copied
 *   d_fb           DEVICE float32, plane d at d * fb_stride_dm elements, [nt_in][nsub*nchan] inside
 *   d_ts           DEVICE float32, plane d at d * ts_stride_dm elements, row k at k * ts_pitch,
 *                  nt_out samples per row (ts_pitch >= nt_out, ts_stride_dm >= nfine * ts_pitch)
 *   d_workspace    DEVICE scratch, 256-byte aligned, >= workspace_bytes from cdmt_incoherent_query
 * cdmt_incoherent_query: host arithmetic only; any output pointer may be NULL.  ngroups = number
 * of trial groups the kernel works in (<= 8 trials each; fewer where the shifts of consecutive
 * trials differ by more than the kernel's register window allows).
 * cdmt_incoherent_shifts: copies the shift table [nfine][nsub*nchan] to HOST memory.
 * Sums are accumulated in float32; the terms of a trial are those of the definition above, added in
 * another order (channels that share their shifts over a group of trials are summed once), so results
 * are exact on integer-valued data and equal to the definition to float32 rounding otherwise.  The plan
 * caches the shift and group tables of the last ddm list it was given (these calls therefore take a
 * non-const plan and, like every other call, must not run concurrently on one plan) and, from the first
 * cdmt_incoherent_dedisperse on, a page-locked copy of them: the call queues one asynchronous copy
 * from that memory and one kernel on `cuda_stream`, nothing else (capturable into a CUDA graph).
 * Limits (CDMT_ERR_SIZE from all three calls): shift_range <= about 14000 samples (four channels of
 * 256 + shift_range samples must fit shared memory), at most 16 x 65535 trial groups.
 *
 * Streaming over block groups (40 000 trials over a 20-minute observation are never
 * resident): keep per DM plane a window of shift_range + nt_group rows; let cdmt_execute write each
 * group's rows behind the first shift_range rows (pass d_out + shift_range * nsub*nchan and the
 * window's plane stride); dedisperse the window (the first group without the empty head: nt_in =
 * nt_group, giving nt_group - shift_range samples; every later one with nt_in = shift_range +
 * nt_group, giving nt_group samples that continue the series); then cdmt_incoherent_carry moves the
 * last shift_range rows of every plane to its front (needs nt_in >= 2 shift_range).  The
 * concatenated outputs are bit for bit those of one call on the whole span.
 * Errors: CDMT_ERR_ARG (null / misaligned pointer, non-finite or non-ascending ddm), CDMT_ERR_SIZE
 * (nt_in <= shift_range, short strides, limits above), CDMT_ERR_WORKSPACE, CDMT_ERR_ALLOC, CDMT_ERR_CUDA.
 */
int cdmt_incoherent_query(cdmt_plan *plan, int nfine, const double *ddm, long long nt_in,
                          int *shift_min, int *shift_range, long long *nt_out, int *ngroups,
                          size_t *workspace_bytes);
int cdmt_incoherent_shifts(cdmt_plan *plan, int nfine, const double *ddm, int *h_shifts);
int cdmt_incoherent_dedisperse(cdmt_plan *plan, const float *d_fb, long long fb_stride_dm,
                               long long nt_in, int nfine, const double *ddm, float *d_ts,
                               long long ts_stride_dm, long long ts_pitch, void *d_workspace,
                               size_t workspace_bytes, void *cuda_stream);
int cdmt_incoherent_carry(cdmt_plan *plan, float *d_fb, long long fb_stride_dm, long long nt_in,
                          int shift_range, void *cuda_stream);
/* Additions per call of cdmt_incoherent_dedisperse over all DM planes (host arithmetic): those of the
 * brute-force definition (one per plane, trial, channel and output sample) and those the kernel
 * performs (one per plane, trial group, channel, DISTINCT shift and sample, plus the hand-over of the
 * run sums to the trials). */
int cdmt_incoherent_work(cdmt_plan *plan, int nfine, const double *ddm, long long nt_in,
                         double *adds_definition, double *adds_performed);

/* Eq. 2: dispersion sweep across [fcen - bw/2, fcen + bw/2] in seconds. */
double cdmt_sweep_seconds(double fcen_mhz, double bw_mhz, double dm);
/* smallest legal noverlap (input samples, rounded up to a multiple of 2 nchan)
 * that covers the sweep of the lowest channel (REF_CHANNEL) or lowest subband (REF_SUBBAND)
 * at the largest |DM| of the plan. */
long long cdmt_min_overlap(const cdmt_plan *plan);

/* Sizes from the dispersion sweep ("n_d n_c >= r t_d ... for the channel with the lowest
 * frequency"; PAPER.md:175 names the single N_bin / n_d for all subbands as an
 * inefficiency): for the given subbands (call it per subband, or per group of subbands that share a
 * plan) returns the smallest noverlap (input samples; a multiple of 2 nchan ndec, so that each discarded edge is a
 * whole number of integrated samples)
 * that covers the sweep of the lowest channel (REF_CHANNEL) or subband (REF_SUBBAND) at DM
 * dm_max_abs, and the smallest power-of-two nfft this library supports whose kept fraction
 * (nfft - noverlap) / nfft is at least min_efficiency (0 < min_efficiency < 1).  Host arithmetic only.
 * Errors: CDMT_ERR_ARG, CDMT_ERR_SIZE (no supported nfft reaches the efficiency). */
int cdmt_suggest_sizes(int nsub, const double *fcen_mhz, double bw_mhz, int nchan, int ndec,
                       double dm_max_abs, int chirp_ref, double min_efficiency, int *nfft,
                       int *noverlap);

/*
 * Per-group sizes inside the library (PAPER.md:79 fixes one N_bin and n_d for all subbands; PAPER.md:175
 * names that as the program's inefficiency next to digifil, which "optimizes the choice for FFT size and
 * data overlap ... depending on the DM and observing frequency").  A multiplan cuts the subbands (ascending
 * fcen_mhz) into at most max_groups contiguous groups.  nfft is chosen as the paper chooses it -- by
 * cdmt_suggest_sizes(min_efficiency) for the lowest subband at the largest |DM| -- and kept for every
 * group (the same kernels run everywhere); a group takes the overlap Eq. 2 asks for at ITS lowest
 * subband, and the cuts are those that keep most of the input (minimum of sum_g nsub_g noverlap_g over
 * all contiguous partitions).  cdmt_multiplan_execute runs the groups one after the other (one workspace) into ONE filterbank
 * d_out[ndm][nout_alloc][nsub*nchan] (descending frequency, plane stride out_stride_dm >= nout_alloc *
 * nsub*nchan).  Common time grid: group g starts reading at input sample first_sample_g = max_h(noverlap_h/2)
 * - noverlap_g/2, so row 0 of every group is the output sample that starts at input sample
 * max_h(noverlap_h/2); group g fills rows [0, nout_g) of its columns, nout_g = nblock_g * Vd_g with its own
 * block length; nout_valid = min_g nout_g rows are complete in every column, rows beyond nout_g of a group's
 * columns are left untouched.  Results of group g are those of a plan made of its subbands and sizes, run on
 * the input from first_sample_g on (same kernels, same bits).
 * cdmt_multiplan_query / _group: host arithmetic; any output pointer may be NULL; kept_fraction = the
 * subband-weighted (nfft - noverlap) / nfft.  Same alignment rules and errors as cdmt_execute.
 */
typedef struct cdmt_multiplan cdmt_multiplan; /* opaque */
int cdmt_multiplan_create(cdmt_multiplan **mplan, int nsub, const double *fcen_mhz, double bw_mhz, int nchan,
                          int ndec, int ndm, const double *dm, int in_dtype, int chirp_ref,
                          double min_efficiency, int max_groups);
int cdmt_multiplan_destroy(cdmt_multiplan *mplan);
int cdmt_multiplan_query(const cdmt_multiplan *mplan, long long nsamp, int *ngroups, long long *nout_valid,
                         long long *nout_alloc, size_t *out_bytes, size_t *workspace_bytes,
                         double *kept_fraction);
int cdmt_multiplan_group(const cdmt_multiplan *mplan, int group, long long nsamp, int *first_subband, int *nsub,
                         int *nfft, int *noverlap, long long *first_sample, long long *nout);
int cdmt_multiplan_execute(cdmt_multiplan *mplan, const void *d_in, long long nsamp, long long in_stride_pol,
                           float *d_out, long long out_stride_dm, void *d_workspace, size_t workspace_bytes,
                           void *cuda_stream);
long long cdmt_multiplan_last_launch_count(const cdmt_multiplan *mplan);

/* Measure the FP32 FMA rate of the device the stream belongs to (the "alu" roofline
 * denominator): runs `iters` dependent-chain FMA launches and returns
 * TFLOP/s in *tflops.  d_scratch: >= 4 bytes * 148 * 1024. */
int cdmt_measure_fp32_peak(void *d_scratch, size_t scratch_bytes, int iters, double *tflops,
                           void *cuda_stream);

/* With CDMT_OPT_PROFILE = 1 every execute records CUDA events on its stream round (kind 0) the
 * two forward-FFT passes of a chunk and (kind 1) each fused per-DM kernel launch.  This call
 * waits for the recorded events, returns the summed durations in milliseconds and the number of
 * spans of each kind since the previous read, and resets the record.  Nothing is recorded while
 * the stream is being captured into a CUDA graph; a record that is never read is discarded once it
 * holds 8192 spans. */
int cdmt_profile_read(cdmt_plan *plan, double *ms_forward, double *ms_fused,
                      long long *n_forward, long long *n_fused);

/* Number of kernel launches cdmt_execute issued on its last call with this plan. */
long long cdmt_last_launch_count(const cdmt_plan *plan);

const char *cdmt_strerror(int status);
const char *cdmt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CDMT_H */
