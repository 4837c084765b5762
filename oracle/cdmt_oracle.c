/*
 * cdmt_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, double-precision CPU restatement of the hot path of cdmt
 * (Bassa, Pleunis & Hessels, arXiv:1607.00909): coherent dedispersion of
 * dual-polarisation complex-voltage subbands to many DM trials, written step by
 * step in the order of the paper's Algorithm 1 and Fig. 2
 * (PAPER.md:51).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or constant with the CUDA library under paper_1607_00909_b200/csrc/.
 *
 * Readings of the paper adopted here are the Q1..Q17 rows of DESIGN.md
 * ("Readings of the paper"); each function cites the passage it follows.
 *
 * Pins (tests/test_oracle_pins.py): P1 brute-force DFT, P2 DM=0 equals direct
 * time-domain channelisation, P3 impulse closed form, P4 tone closed form /
 * descending channel order, P5 Parseval, P6 H(DM)H(-DM)=1 and circular identity,
 * P7 group delay = Eq. 2 and the paper's printed 3.3 ms / 5.7 ms, P8 subband- vs
 * channel-referenced chirp identity, P9 dispersed impulse recovered only at the
 * matching DM.  Not pinned (no data in this container): anything that needs the
 * paper's LOFAR recordings -- "parity unpinned" for real-sky behaviour only.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o liboracle_cdmt.so cdmt_oracle.c -lm
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#define ORACLE_IN_CF32 0
#define ORACLE_IN_CI8 1
#define ORACLE_REF_CHANNEL 0
#define ORACLE_REF_SUBBAND 1

/* k_DM^-1 = 2.41e-4 s MHz^2.  With f, f0 in MHz the phase of Eq. 1 in
 * cycles is DM f^2 / (2.41e-4 * 1e-6 * f0^2 (f0+f)): the 1e-6 turns the remaining MHz
 * into Hz (reading Q1). */
static const double KDM_INV_S_MHZ2 = 2.41e-4;

typedef struct {
    int nsub;
    const double *fcen_mhz; /* [nsub] subband centre frequencies, ascending */
    double bw_mhz;          /* subband bandwidth = complex sample rate */
    int nfft;               /* N_bin */
    int noverlap;           /* n_d * n_c, in input samples (reading Q7) */
    int nchan;              /* n_c */
    int ndec;               /* time-integration factor (north_star; not in Alg. 1) */
    int ndm;
    const double *dm;       /* [ndm] */
    int in_dtype;           /* ORACLE_IN_* : interleaved (re,im) float32 or int8 */
    int chirp_ref;          /* ORACLE_REF_* : nu_0 = channel centre or subband centre (Q3) */
} oracle_params;

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* The library primitive: an FFT.  Iterative radix-2 Cooley-Tukey, double.   */
/* out[k] = sum_n in[n] exp(sign * 2 pi i k n / n), unnormalised.            */
/* Pinned by P1 against an O(n^2) DFT.                                        */
/* ------------------------------------------------------------------------- */
int oracle_fft(int n, int sign, const cplx *in, cplx *out)
{
    if (n < 1 || (n & (n - 1)) != 0) return 1;
    int logn = 0;
    while ((1 << logn) < n) logn++;
    for (int i = 0; i < n; i++) {
        int r = 0;
        for (int b = 0; b < logn; b++)
            if (i & (1 << b)) r |= 1 << (logn - 1 - b);
        out[r] = in[i];
    }
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)(n / 2 + 1));
    if (!w) return 2;
    for (int k = 0; k < n / 2; k++) {
        double a = 2.0 * M_PI * (double)k / (double)n;
        w[k] = cos(a) + I * (sign * sin(a));
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len / 2, tstep = n / len;
        for (int base = 0; base < n; base += len)
            for (int k = 0; k < half; k++) {
                cplx a = out[base + k];
                cplx b = out[base + k + half] * w[k * tstep];
                out[base + k] = a + b;
                out[base + k + half] = a - b;
            }
    }
    free(w);
    return 0;
}

/* Eq. 1: phase of H(nu + nu0) in cycles, nu = f_off, nu0 = f0 (MHz). */
double oracle_chirp_phase_cycles(double dm, double f0_mhz, double f_off_mhz)
{
    return dm * f_off_mhz * f_off_mhz /
           (KDM_INV_S_MHZ2 * 1e-6 * f0_mhz * f0_mhz * (f0_mhz + f_off_mhz));
}

/* Eq. 2: t_d = k_DM (nu_min^-2 - nu_max^-2) DM, seconds. */
double oracle_sweep_seconds(double fcen_mhz, double bw_mhz, double dm)
{
    double lo = fcen_mhz - 0.5 * bw_mhz, hi = fcen_mhz + 0.5 * bw_mhz;
    return (1.0 / KDM_INV_S_MHZ2) * (1.0 / (lo * lo) - 1.0 / (hi * hi)) * dm;
}

/* Block bookkeeping (readings Q7, Q8). */
int oracle_sizes(const oracle_params *p, long nsamp, int *nblock, int *mbin, int *hdisc, int *vdec)
{
    if (p->nfft <= 0 || p->nchan <= 0 || p->ndec <= 0 || p->nfft % p->nchan) return 1;
    if (p->noverlap < 0 || p->noverlap >= p->nfft || p->noverlap % (2 * p->nchan)) return 1;
    int step = p->nfft - p->noverlap;
    if (step % (p->nchan * p->ndec)) return 1;
    if (nsamp < p->nfft) return 1;
    *nblock = (int)((nsamp - p->nfft) / step) + 1;
    *mbin = p->nfft / p->nchan;
    *hdisc = p->noverlap / (2 * p->nchan);
    *vdec = (*mbin - 2 * *hdisc) / p->ndec;
    return 0;
}

/* "unpack" (Alg. 1 l.95): one input word -> a complex number (Q14). */
static cplx unpack_sample(const void *x, int in_dtype, long idx)
{
    if (in_dtype == ORACLE_IN_CI8) {
        const int8_t *q = (const int8_t *)x;
        return (double)q[2 * idx] + I * (double)q[2 * idx + 1];
    }
    const float *q = (const float *)x;
    return (double)q[2 * idx] + I * (double)q[2 * idx + 1];
}

/* Stages 1-3 of Fig. 2 for one polarisation of one block, plus Alg. 1 l.97:
 *  - segment of N_bin samples starting at `first` (caller applies the overlap),
 *  - forward FFT, kernel exp(-2 pi i k n / N),
 *  - swap halves so that bins increase in frequency:
 *    Xs[j] = U[(j + N/2) mod N]; bin j is (j - N/2) bw/N from the subband centre (Q4, Q5).
 * `xpol` points at sample 0 of this polarisation. */
int oracle_block_spectrum(const void *xpol, int in_dtype, long first, int nfft, cplx *Xs)
{
    cplx *u = (cplx *)malloc(sizeof(cplx) * (size_t)nfft);
    cplx *U = (cplx *)malloc(sizeof(cplx) * (size_t)nfft);
    if (!u || !U) { free(u); free(U); return 2; }
    for (int n = 0; n < nfft; n++) u[n] = unpack_sample(xpol, in_dtype, first + n);
    int rc = oracle_fft(nfft, -1, u, U);
    for (int j = 0; j < nfft; j++) Xs[j] = U[(j + nfft / 2) % nfft];
    free(u);
    free(U);
    return rc;
}

/* The transfer function of one channel at one DM (Alg. 1 l.89-91, Eq. 1):
 * H[m], m < M, for channel c of a subband centred at fcen.
 *   REF_CHANNEL: nu0 = centre of channel c, nu = (m - M/2) bw/N          (Q3 default, Q4)
 *   REF_SUBBAND: nu0 = fcen,               nu = (c M + m - N/2) bw/N     (Q3 alternative)
 * Multiplying by H (exponent +, as printed) removes the dispersion (Q2). */
void oracle_transfer_function(const oracle_params *p, double fcen, int c, double dm, cplx *H)
{
    int N = p->nfft, C = p->nchan, M = N / C;
    for (int m = 0; m < M; m++) {
        double f0, f;
        if (p->chirp_ref == ORACLE_REF_CHANNEL) {
            f0 = fcen + ((double)c + 0.5 - 0.5 * (double)C) * p->bw_mhz / (double)C;
            f = (double)(m - M / 2) * p->bw_mhz / (double)N;
        } else {
            f0 = fcen;
            f = (double)(c * M + m - N / 2) * p->bw_mhz / (double)N;
        }
        double phi = oracle_chirp_phase_cycles(dm, f0, f);
        H[m] = cexp(2.0 * M_PI * I * phi);
    }
}

/* Everything Alg. 1 does with one (subband, block) unit, for all DMs.
 *   xblock : the unit's N_bin input samples of both pols, [2][N] in p->in_dtype
 *   out    : [ndm][Vd][C] doubles, channel index ASCENDING in frequency here;
 *            the descending pack of PAPER.md:123 is done by the callers below.
 * Steps per DM (Alg. 1 l.98-103; Fig. 2 stages 4-6):
 *   multiply by the transfer functions of the C consecutive channels
 *   swap halves per channel
 *   backward FFT of length M, kernel exp(+2 pi i k t / M)
 *   unpad: drop h = noverlap/(2C) samples at each edge
 *   detect and add the polarisations: |y0|^2 + |y1|^2 (Q11), scaled 1/(N M) (Q6)
 *   integrate ndec consecutive kept samples (plain sum, Q9)
 */
int oracle_unit(const oracle_params *p, int s, const void *xblock, double *out)
{
    int N = p->nfft, C = p->nchan, M = N / C, D = p->ndec;
    int h = p->noverlap / (2 * C), V = M - 2 * h, Vd = V / D;
    size_t esz = (p->in_dtype == ORACLE_IN_CI8) ? 2 : 8;
    cplx *Xs[2];
    cplx *H = (cplx *)malloc(sizeof(cplx) * (size_t)M);
    cplx *Z = (cplx *)malloc(sizeof(cplx) * (size_t)M);
    cplx *Zsw = (cplx *)malloc(sizeof(cplx) * (size_t)M);
    cplx *y[2];
    double *Ipow = (double *)malloc(sizeof(double) * (size_t)M);
    for (int q = 0; q < 2; q++) {
        Xs[q] = (cplx *)malloc(sizeof(cplx) * (size_t)N);
        y[q] = (cplx *)malloc(sizeof(cplx) * (size_t)M);
    }
    int rc = 0;
    for (int q = 0; q < 2; q++)
        rc |= oracle_block_spectrum((const char *)xblock + (size_t)q * N * esz, p->in_dtype, 0, N, Xs[q]);
    for (int d = 0; d < p->ndm && !rc; d++) {
        for (int c = 0; c < C; c++) {
            oracle_transfer_function(p, p->fcen_mhz[s], c, p->dm[d], H);
            for (int q = 0; q < 2; q++) {
                for (int m = 0; m < M; m++) Z[m] = Xs[q][c * M + m] * H[m];
                for (int k = 0; k < M; k++) Zsw[k] = Z[(k + M / 2) % M];
                rc |= oracle_fft(M, +1, Zsw, y[q]);
            }
            for (int t = 0; t < M; t++) {
                double a0 = creal(y[0][t]), b0 = cimag(y[0][t]);
                double a1 = creal(y[1][t]), b1 = cimag(y[1][t]);
                Ipow[t] = (a0 * a0 + b0 * b0 + a1 * a1 + b1 * b1) / ((double)N * (double)M);
            }
            for (int qd = 0; qd < Vd; qd++) {
                double acc = 0.0;
                for (int r = 0; r < D; r++) acc += Ipow[h + qd * D + r];
                out[((size_t)d * Vd + qd) * C + c] = acc;
            }
        }
    }
    for (int q = 0; q < 2; q++) { free(Xs[q]); free(y[q]); }
    free(H); free(Z); free(Zsw); free(Ipow);
    return rc;
}

/* A batch of independent units (used for sampled parity at full size and for timing).
 *   unit_s[u]  : subband index of unit u (selects fcen)
 *   xblocks    : [nunits][2][N] input words
 *   out        : [nunits][ndm][Vd][C] doubles, channels ascending
 */
int oracle_units(const oracle_params *p, int nunits, const int *unit_s, const void *xblocks, double *out)
{
    int N = p->nfft, C = p->nchan, M = N / C;
    int h = p->noverlap / (2 * C), Vd = (M - 2 * h) / p->ndec;
    size_t esz = (p->in_dtype == ORACLE_IN_CI8) ? 2 : 8;
    size_t in_unit = (size_t)2 * N * esz, out_unit = (size_t)p->ndm * Vd * C;
    int rc = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(| : rc)
    for (int u = 0; u < nunits; u++)
        rc |= oracle_unit(p, unit_s[u], (const char *)xblocks + (size_t)u * in_unit, out + (size_t)u * out_unit);
    return rc;
}

/* The whole path on a whole input.
 *   x   : [nsub][2][nsamp] input words, time fastest (Q14)
 *   out : [ndm][nblock*Vd][nsub*C] float32 and/or out64 (same layout, double); either may be NULL.
 * Block b is input samples [b step, b step + N) (valid-only blocking, Q8); its kept output
 * samples are tau = b Vd + q.  Channel (s, c) is stored at S C - 1 - (s C + c): decreasing
 * frequency (Q10).
 */
int oracle_run(const oracle_params *p, const void *x, long nsamp, float *out, double *out64)
{
    int B, M, h, Vd;
    if (oracle_sizes(p, nsamp, &B, &M, &h, &Vd)) return 1;
    int N = p->nfft, C = p->nchan, S = p->nsub, step = N - p->noverlap;
    size_t esz = (p->in_dtype == ORACLE_IN_CI8) ? 2 : 8;
    size_t ntime = (size_t)B * Vd, nch = (size_t)S * C;
    int rc = 0;
#pragma omp parallel for collapse(2) schedule(dynamic, 1) reduction(| : rc)
    for (int s = 0; s < S; s++)
        for (int b = 0; b < B; b++) {
            char *blk = (char *)malloc((size_t)2 * N * esz);
            double *o = (double *)malloc(sizeof(double) * (size_t)p->ndm * Vd * C);
            for (int q = 0; q < 2; q++)
                memcpy(blk + (size_t)q * N * esz,
                       (const char *)x + (((size_t)s * 2 + q) * (size_t)nsamp + (size_t)b * step) * esz,
                       (size_t)N * esz);
            rc |= oracle_unit(p, s, blk, o);
            for (int d = 0; d < p->ndm; d++)
                for (int qd = 0; qd < Vd; qd++)
                    for (int c = 0; c < C; c++) {
                        double v = o[((size_t)d * Vd + qd) * C + c];
                        size_t idx = ((size_t)d * ntime + (size_t)b * Vd + qd) * nch + (nch - 1 - ((size_t)s * C + c));
                        if (out) out[idx] = (float)v;
                        if (out64) out64[idx] = v;
                    }
            free(blk);
            free(o);
        }
    return rc;
}

/* Intermediate for per-kernel tests: dedispersed, channelised complex time series of one
 * channel of one pol of one block BEFORE unpad/detect: y[t], t < M (Fig. 2 stage 5). */
int oracle_channel_timeseries(const oracle_params *p, int s, int c, double dm, const void *xpol_block, cplx *y)
{
    int N = p->nfft, M = N / p->nchan;
    cplx *Xs = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    cplx *H = (cplx *)malloc(sizeof(cplx) * (size_t)M);
    cplx *Z = (cplx *)malloc(sizeof(cplx) * (size_t)M);
    cplx *Zsw = (cplx *)malloc(sizeof(cplx) * (size_t)M);
    int rc = oracle_block_spectrum(xpol_block, p->in_dtype, 0, N, Xs);
    oracle_transfer_function(p, p->fcen_mhz[s], c, dm, H);
    for (int m = 0; m < M; m++) Z[m] = Xs[c * M + m] * H[m];
    for (int k = 0; k < M; k++) Zsw[k] = Z[(k + M / 2) % M];
    rc |= oracle_fft(M, +1, Zsw, y);
    free(Xs); free(H); free(Z); free(Zsw);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Redigitisation to 8 bit: Algorithm 1 l.104-106 ("compute block sums", "compute channel
 * statistics", "redigitize").  Same four steps, same
 * order, statistics in double.
 *
 *   fb      [ndm][nblock*vd][nch] float32 filterbank of ONE batch of nblock data blocks
 *           (what oracle_run returns); statistics are per DM trial and per channel over the
 *           nblock*vd samples of the batch ("the floating point timeseries of each
 *           channel of N_FFT (M_bin - n_d) samples"; reading Q19)
 *   segsum  [ndm][nblock][nch][2]: sum of I and of I^2 over the vd samples that block b gave to
 *           the channel ("sums of intensity and intensity squared for segments of M samples";
 *           reading Q20: one segment = one data block's samples)
 *   mean, std [ndm][nch]: mean = sum I / n,  std = sqrt(max(0, sum I^2 / n - mean^2)),
 *           n = nblock*vd ("average and standard deviation of each channel" from the segment
 *           sums; population form, reading Q21)
 *   offset, scale [ndm][nch] float32 and codes [ndm][nblock*vd][nch] uint8: the paper says only
 *           that offset and scale follow from mean and std; reading Q22:
 *               scale  = std / qstd          (1 if std == 0)
 *               offset = mean - qmean * scale
 *               code   = clip(rint((I - offset) / scale), 0, 255)
 *           so that a channel's codes have mean qmean and standard deviation qstd.  offset and
 *           scale are rounded to float32 once; the decision (subtract, divide, round half to
 *           even, clip) is taken in float32, the precision of the paper's data path
 *           (cufftComplex / float), one correctly rounded operation at a time.
 * Any of segsum, mean, std, offset, scale, codes may be NULL.
 */
int oracle_redigitize(const float *fb, long ndm, long nblock, long vd, long nch, double qmean, double qstd,
                      double *segsum, double *mean, double *std, float *offset, float *scale, uint8_t *codes)
{
    if (!fb || ndm < 1 || nblock < 1 || vd < 1 || nch < 1 || !(qstd > 0.0)) return 1;
    const long nt = nblock * vd;
    for (long d = 0; d < ndm; d++) {
        const float *f = fb + (size_t)d * nt * nch;
        for (long c = 0; c < nch; c++) {
            /* compute block sums (l.104) */
            double tot = 0.0, tot2 = 0.0;
            for (long b = 0; b < nblock; b++) {
                double s1 = 0.0, s2 = 0.0;
                for (long q = 0; q < vd; q++) {
                    const double v = (double)f[(size_t)(b * vd + q) * nch + c];
                    s1 += v;
                    s2 += v * v;
                }
                if (segsum) {
                    segsum[(((size_t)d * nblock + b) * nch + c) * 2 + 0] = s1;
                    segsum[(((size_t)d * nblock + b) * nch + c) * 2 + 1] = s2;
                }
                /* compute channel statistics (l.105): the segment sums are added up */
                tot += s1;
                tot2 += s2;
            }
            const double mu = tot / (double)nt;
            double var = tot2 / (double)nt - mu * mu;
            if (var < 0.0) var = 0.0;
            const double sd = sqrt(var);
            if (mean) mean[(size_t)d * nch + c] = mu;
            if (std) std[(size_t)d * nch + c] = sd;
            /* redigitize (l.106) */
            const double sc64 = sd > 0.0 ? sd / qstd : 1.0;
            const float sc = (float)sc64;
            const float off = (float)(mu - qmean * sc64);
            if (scale) scale[(size_t)d * nch + c] = sc;
            if (offset) offset[(size_t)d * nch + c] = off;
            if (codes)
                for (long t = 0; t < nt; t++) {
                    volatile float diff = f[(size_t)t * nch + c] - off; /* float32 subtraction */
                    volatile float quot = diff / sc;                    /* float32 division */
                    float r = nearbyintf(quot);                         /* round half to even */
                    if (!(r >= 0.0f)) r = 0.0f;
                    if (r > 255.0f) r = 255.0f;
                    codes[((size_t)d * nt + t) * nch + c] = (uint8_t)r;
                }
        }
    }
    return 0;
}

/* The decision of l.106 alone, with offset and scale GIVEN (float32, [ndm][nch]): used to
 * check a quantiser bit for bit on the offsets and scales it reports itself. */
int oracle_quantize(const float *fb, long ndm, long nt, long nch, const float *offset, const float *scale,
                    uint8_t *codes)
{
    if (!fb || !offset || !scale || !codes) return 1;
    for (long d = 0; d < ndm; d++)
        for (long t = 0; t < nt; t++)
            for (long c = 0; c < nch; c++) {
                volatile float diff = fb[((size_t)d * nt + t) * nch + c] - offset[(size_t)d * nch + c];
                volatile float quot = diff / scale[(size_t)d * nch + c];
                float r = nearbyintf(quot);
                if (!(r >= 0.0f)) r = 0.0f;
                if (r > 255.0f) r = 255.0f;
                codes[((size_t)d * nt + t) * nch + c] = (uint8_t)r;
            }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Incoherent dedispersion of ONE coherently dedispersed filterbank over a grid of fine DM
 * offsets: the second stage of the semi-coherent search of PAPER.md:35 and PAPER.md:141
 * ("each of the coherently dedispersed filterbanks was then incoherently dedispersed at steps
 * of 0.002 pc cm^-3 ranging from -0.5 to 0.5 pc cm^-3 around the coherently dedispersed DM ...
 * brute force dedispersion algorithm").  The paper uses a third-party library and prints no
 * formula beyond Eq. 2; the brute-force definition is written out here (readings Q23-Q26):
 *
 *   channel j of the filterbank (DESCENDING frequency) has centre frequency f_j;
 *   the residual delay of channel j at DM offset ddm relative to the highest channel f_0 is
 *       tau_j = ddm (f_j^-2 - f_0^-2) / 2.41e-4   seconds   (Eq. 2 between two frequencies, MHz)
 *   shift[k][j] = rint(tau_j(ddm_k) / tsamp)       samples (round half to even, fp64)
 *   smin, smax  = extremes of shift over all k, j (smin <= 0 <= smax: shift[k][0] = 0)
 *   ts[k][t]    = sum_j fb[t + shift[k][j] - smin][j],   t < nt - (smax - smin)
 *
 * so output sample t is time t - smin of the highest channel, and only samples for which
 * every channel is inside the filterbank are produced (valid-only, as reading Q8).
 * The sum over channels is taken in double, in channel order, and rounded to float32 last.
 *
 *   fb      [nt][nch] float32       fch [nch] channel centre frequencies, MHz
 *   ddm     [nfine]                 tsamp: filterbank sample time, seconds
 *   shifts  [nfine][nch] int32 (may be NULL), ts [nfine][nt - (smax-smin)] float32 (may be NULL)
 * Returns smax - smin in *range and smin in *smin_out (either may be NULL); nonzero on error.
 */
int oracle_incoherent(const float *fb, long nt, long nch, const double *fch, double tsamp, long nfine,
                      const double *ddm, int *shifts, float *ts, long *range, long *smin_out)
{
    if (nt < 1 || nch < 1 || nfine < 1 || !fch || !ddm || !(tsamp > 0.0)) return 1;
    int *sh = shifts ? shifts : (int *)malloc(sizeof(int) * (size_t)nfine * nch);
    if (!sh) return 2;
    long smin = 0, smax = 0;
    for (long k = 0; k < nfine; k++)
        for (long j = 0; j < nch; j++) {
            const double tau = ddm[k] * (1.0 / (fch[j] * fch[j]) - 1.0 / (fch[0] * fch[0])) / KDM_INV_S_MHZ2;
            const long s = (long)nearbyint(tau / tsamp);
            sh[k * nch + j] = (int)s;
            if (s < smin) smin = s;
            if (s > smax) smax = s;
        }
    if (range) *range = smax - smin;
    if (smin_out) *smin_out = smin;
    int rc = 0;
    const long nout = nt - (smax - smin);
    if (ts) {
        if (!fb || nout < 1) rc = 3;
        else
            for (long k = 0; k < nfine; k++)
                for (long t = 0; t < nout; t++) {
                    double acc = 0.0;
                    for (long j = 0; j < nch; j++) acc += (double)fb[(size_t)(t + sh[k * nch + j] - smin) * nch + j];
                    ts[(size_t)k * nout + t] = (float)acc;
                }
    }
    if (!shifts) free(sh);
    return rc;
}
