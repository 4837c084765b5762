// cdmt_api.cu -- the C ABI declared in include/cdmt.h: plan bookkeeping (host only) and the
// launch sequences.  No arithmetic of the method lives here except the Eq. 2 helper.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/cdmt.h"
#include "cdmt_internal.h"

using namespace cdmt;

struct cdmt_plan {
    Geometry g;
    std::vector<double> fcen, dm;
    long long chunk_units;   // 0 = automatic
    int dm_tile;             // 0 = all
    int accurate;
    int profile;             // record CUDA events around each kernel class
    long long host_group;    // CDMT_OPT_HOST_GROUP_BLOCKS: blocks per staged group of the host path (0 = automatic)
    int force_generic;       // CDMT_OPT_FUSED_KERNEL: 0 auto, 1 generic, 2 scalar fast, 3 packed halves, 4 packed pols, 5 pipelined
    int keep_tables;         // CDMT_OPT_KEEP_TABLES: the caller leaves the workspace head alone between calls
    const void *tables_ws;   // workspace whose head holds this plan's tables (keep_tables only)
    long long tables_cu;     // ... laid out for this many chunk units
    long long last_launches;
    std::vector<cudaEvent_t> ev_pool;   // created lazily, reused
    size_t ev_used;
    struct Span { size_t e0, e1; int kind; };   // kind 0: forward FFT passes, 1: fused per-DM kernel
    std::vector<Span> spans;
    // host-buffer path (cdmt_execute_host): copy streams and the events that order the double buffers
    IncoherentTables ic;     // incoherent-dedispersion tables of the last fine-DM list used
    std::vector<double> ic_ddm;
    cudaStream_t s_in, s_out;
    cudaEvent_t ev_start, ev_h2d[2], ev_comp[2], ev_d2h[2], ev_join[2];
    bool host_ready;
};

// Lazily create the copy streams and ordering events of the host-buffer path.
static bool plan_host_pipeline(cdmt_plan *p)
{
    if (p->host_ready) return true;
    bool ok = cudaStreamCreateWithFlags(&p->s_in, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&p->s_out, cudaStreamNonBlocking) == cudaSuccess &&
              cudaEventCreateWithFlags(&p->ev_start, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < 2 && ok; ++i)
        ok = cudaEventCreateWithFlags(&p->ev_h2d[i], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&p->ev_comp[i], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&p->ev_d2h[i], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&p->ev_join[i], cudaEventDisableTiming) == cudaSuccess;
    p->host_ready = ok;
    return ok;
}

static cudaEvent_t plan_event(cdmt_plan *p, size_t *idx)
{
    if (p->ev_used == p->ev_pool.size()) {
        cudaEvent_t e = nullptr;
        if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
        p->ev_pool.push_back(e);
    }
    *idx = p->ev_used;
    return p->ev_pool[p->ev_used++];
}

constexpr size_t PROFILE_MAX_SPANS = 8192;  // unread profile spans kept per plan

static bool is_pow2(long long x) { return x > 0 && (x & (x - 1)) == 0; }

static int ilog2(long long x)
{
    int n = 0;
    while ((1LL << n) < x) ++n;
    return n;
}

extern "C" const char *cdmt_strerror(int status)
{
    switch (status) {
    case CDMT_OK: return "ok";
    case CDMT_ERR_ARG: return "invalid argument (null or misaligned pointer, or bad value)";
    case CDMT_ERR_SIZE: return "sizes violate a divisibility or range rule";
    case CDMT_ERR_WORKSPACE: return "workspace too small";
    case CDMT_ERR_CUDA: return "CUDA call or kernel launch failed";
    case CDMT_ERR_ALLOC: return "host allocation failed";
    default: return "unknown status";
    }
}

extern "C" const char *cdmt_version(void) { return "cdmt-b200 0.1 (sm_100a)"; }

// Eq. 2.
extern "C" double cdmt_sweep_seconds(double fcen_mhz, double bw_mhz, double dm)
{
    const double lo = fcen_mhz - 0.5 * bw_mhz, hi = fcen_mhz + 0.5 * bw_mhz;
    return (1.0 / 2.41e-4) * (1.0 / (lo * lo) - 1.0 / (hi * hi)) * dm;
}

extern "C" int cdmt_plan_create(cdmt_plan **plan, int nsub, const double *fcen_mhz, double bw_mhz, int nfft,
                                int noverlap, int nchan, int ndec, int ndm, const double *dm, int in_dtype,
                                int chirp_ref)
{
    if (!plan) return CDMT_ERR_ARG;
    *plan = nullptr;
    if (!fcen_mhz || !dm || nsub < 1 || ndm < 1) return CDMT_ERR_ARG;
    if (!(bw_mhz > 0.0) || !std::isfinite(bw_mhz)) return CDMT_ERR_ARG;
    if (in_dtype < CDMT_IN_CF32 || in_dtype > CDMT_IN_PI8) return CDMT_ERR_ARG;
    if (chirp_ref != CDMT_REF_CHANNEL && chirp_ref != CDMT_REF_SUBBAND) return CDMT_ERR_ARG;
    for (int s = 0; s < nsub; ++s)
        if (!std::isfinite(fcen_mhz[s]) || !(fcen_mhz[s] - 0.5 * bw_mhz > 0.0)) return CDMT_ERR_ARG;
    for (int d = 0; d < ndm; ++d)
        if (!std::isfinite(dm[d])) return CDMT_ERR_ARG;
    if (!is_pow2(nfft) || nfft < 256 || nfft > (1 << 20)) return CDMT_ERR_SIZE;
    if (!is_pow2(nchan) || nchan > nfft) return CDMT_ERR_SIZE;
    const int M = nfft / nchan;
    if (!fused_len_supported(M)) return CDMT_ERR_SIZE;
    if (ndec < 1) return CDMT_ERR_SIZE;
    if (noverlap < 0 || noverlap >= nfft || noverlap % (2 * nchan) != 0) return CDMT_ERR_SIZE;
    if ((nfft - noverlap) % (nchan * ndec) != 0) return CDMT_ERR_SIZE;

    cdmt_plan *p = new (std::nothrow) cdmt_plan();
    if (!p) return CDMT_ERR_ALLOC;
    try {
        p->fcen.assign(fcen_mhz, fcen_mhz + nsub);
        p->dm.assign(dm, dm + ndm);
    } catch (...) {
        delete p;
        return CDMT_ERR_ALLOC;
    }
    Geometry &g = p->g;
    g.nsub = nsub; g.nfft = nfft; g.noverlap = noverlap; g.nchan = nchan; g.ndec = ndec; g.ndm = ndm;
    g.in_dtype = in_dtype; g.chirp_ref = chirp_ref; g.bw_mhz = bw_mhz;
    g.step = nfft - noverlap;
    g.mbin = M;
    g.hdisc = noverlap / (2 * nchan);
    g.vdec = (M - 2 * g.hdisc) / ndec;
    const int lg = ilog2(nfft);
    g.n1 = 1 << ((lg + 1) / 2);
    g.n2 = nfft / g.n1;
    g.lo_bits = (lg + 1) / 2;
    g.tw_hi_bits = lg - g.lo_bits;
    if (!forward_len_supported(g.n1) || !forward_len_supported(g.n2)) {
        delete p;
        return CDMT_ERR_SIZE;
    }
    p->chunk_units = 0;
    p->dm_tile = 0;
    p->accurate = 0;
    p->profile = 0;
    p->force_generic = 0;
    p->ev_used = 0;
    p->last_launches = 0;
    p->host_ready = false;
    p->host_group = 0;
    p->keep_tables = 0;
    p->tables_ws = nullptr;
    p->tables_cu = 0;
    p->s_in = p->s_out = nullptr;
    *plan = p;
    return CDMT_OK;
}

extern "C" int cdmt_plan_destroy(cdmt_plan *plan)
{
    if (!plan) return CDMT_ERR_ARG;
    for (cudaEvent_t e : plan->ev_pool) cudaEventDestroy(e);
    incoherent_release(&plan->ic);
    if (plan->host_ready) {
        cudaStreamDestroy(plan->s_in);
        cudaStreamDestroy(plan->s_out);
        cudaEventDestroy(plan->ev_start);
        for (int i = 0; i < 2; ++i) {
            cudaEventDestroy(plan->ev_h2d[i]);
            cudaEventDestroy(plan->ev_comp[i]);
            cudaEventDestroy(plan->ev_d2h[i]);
            cudaEventDestroy(plan->ev_join[i]);
        }
    }
    delete plan;
    return CDMT_OK;
}

extern "C" int cdmt_plan_set_option(cdmt_plan *plan, int key, long long value)
{
    if (!plan) return CDMT_ERR_ARG;
    switch (key) {
    case CDMT_OPT_CHUNK_UNITS:
        if (value < 0 || value > (1 << 30)) return CDMT_ERR_ARG;
        plan->chunk_units = value;
        return CDMT_OK;
    case CDMT_OPT_DM_TILE:
        if (value < 0 || value > (1 << 30)) return CDMT_ERR_ARG;
        plan->dm_tile = (int)value;
        return CDMT_OK;
    case CDMT_OPT_ACCURATE_SINCOS:
        if (value != 0 && value != 1) return CDMT_ERR_ARG;
        plan->accurate = (int)value;
        return CDMT_OK;
    case CDMT_OPT_PROFILE:
        if (value != 0 && value != 1) return CDMT_ERR_ARG;
        plan->profile = (int)value;
        return CDMT_OK;
    case CDMT_OPT_FUSED_KERNEL:
        if (value < 0 || value > 5) return CDMT_ERR_ARG;
        plan->force_generic = (int)value;
        return CDMT_OK;
    case CDMT_OPT_HOST_GROUP_BLOCKS:
        if (value < 0 || value > (1LL << 30)) return CDMT_ERR_ARG;
        plan->host_group = value;
        return CDMT_OK;
    case CDMT_OPT_KEEP_TABLES:
        if (value != 0 && value != 1) return CDMT_ERR_ARG;
        plan->keep_tables = (int)value;
        plan->tables_ws = nullptr;
        return CDMT_OK;
    default: return CDMT_ERR_ARG;
    }
}

static long long nblock_for(const Geometry &g, long long nsamp)
{
    return nsamp < g.nfft ? 0 : (nsamp - g.nfft) / g.step + 1;
}

// units resident at once: by default about 4 GiB of spectra (and as much again for the pass-A buffer).
// The fused kernel runs one CTA per SM for ~0.4 ms, so a launch of n CTAs loses the unfilled part of
// its last wave: 4608 CTAs (c3 at 1 GiB) are 31.1 waves on 148 SMs = 2.7 % idle, 32256 are 217.9 = 0.03 %.
static long long chunk_units_for(const cdmt_plan *p, long long nunits)
{
    long long c = p->chunk_units;
    if (c <= 0) {
        const long long per_unit = 2LL * p->g.nfft * (long long)sizeof(float2);
        c = (4LL << 30) / per_unit;
        if (c < 1) c = 1;
    }
    // grid.x of the fused kernel = chunk * nchan must stay below 2^31
    const long long cap = ((1LL << 31) - 1) / p->g.nchan / 2;
    if (c > cap) c = cap;
    if (c > nunits) c = nunits;
    // whole blocks -- and an even number of them -- let the warp-specialised kernel pair the blocks of a
    // (subband, channel); a caller's explicit CDMT_OPT_CHUNK_UNITS is taken as it is
    if (p->chunk_units <= 0) {
        const long long S = p->g.nsub;
        if (c >= 2 * S) c -= c % (2 * S);
        else if (c >= S) c -= c % S;
    }
    return c < 1 ? 1 : c;
}

extern "C" int cdmt_plan_query(const cdmt_plan *plan, long long nsamp, int *nblock, long long *nsamp_consumed,
                               long long *nout_per_chan, size_t *out_bytes, size_t *workspace_bytes)
{
    if (!plan) return CDMT_ERR_ARG;
    const Geometry &g = plan->g;
    const long long nb = nblock_for(g, nsamp);
    if (nb < 1 || nb > (1LL << 30)) return CDMT_ERR_SIZE;
    if (nblock) *nblock = (int)nb;
    if (nsamp_consumed) *nsamp_consumed = (nb - 1) * g.step + g.nfft;
    if (nout_per_chan) *nout_per_chan = nb * g.vdec;
    if (out_bytes) *out_bytes = (size_t)g.ndm * (size_t)(nb * g.vdec) * (size_t)g.nsub * g.nchan * sizeof(float);
    if (workspace_bytes) {
        const long long cu = chunk_units_for(plan, nb * g.nsub);
        *workspace_bytes = workspace_layout(g, (int)cu, nullptr, nullptr);
    }
    return CDMT_OK;
}

static int check_cuda(cudaError_t e)
{
    if (e == cudaSuccess) return CDMT_OK;
    cudaGetLastError();  // clear the sticky state
    return CDMT_ERR_CUDA;
}

static int validate_input(const cdmt_plan *plan, const void *d_in, long long nsamp, long long in_stride_pol,
                          long long *nb, bool align16 = false)
{
    if (!plan || !d_in) return CDMT_ERR_ARG;
    const Geometry &g = plan->g;
    // one complex word: the forward pass reads 8-byte (float32) or 2-byte (int8) words and takes wider
    // loads only where the address allows; cdmt_unpack's float4 path wants 16 bytes (align16)
    const uintptr_t word = g.in_dtype == CDMT_IN_CF32 ? (align16 ? 16 : 8) : (uintptr_t)in_word_bytes(g.in_dtype);
    if ((reinterpret_cast<uintptr_t>(d_in) & (word - 1)) != 0) return CDMT_ERR_ARG;
    if (nsamp < g.nfft) return CDMT_ERR_SIZE;
    if (in_stride_pol < nsamp) return CDMT_ERR_SIZE;
    if (align16 && g.in_dtype == CDMT_IN_CF32 && (in_stride_pol & 1)) return CDMT_ERR_SIZE;
    *nb = nblock_for(g, nsamp);
    if (*nb < 1 || *nb * g.nsub > (1LL << 30)) return CDMT_ERR_SIZE;
    return CDMT_OK;
}

static int run_chunks(cdmt_plan *plan, const void *d_in, long long in_stride_pol, long long nb, float *d_out,
                      long long out_stride_dm, float2 *d_spec_out, void *d_workspace, size_t workspace_bytes,
                      cudaStream_t st, double *d_segsum = nullptr, int out_pitch = 0)
{
    const Geometry &g = plan->g;
    const long long nunits = nb * g.nsub;
    const long long cu = chunk_units_for(plan, nunits);
    Workspace ws;
    const size_t need = workspace_layout(g, (int)cu, reinterpret_cast<char *>(d_workspace), &ws);
    if (workspace_bytes < need) return CDMT_ERR_WORKSPACE;
    plan->last_launches = 0;
    int rc = CDMT_OK;
    if (!(plan->keep_tables && plan->tables_ws == d_workspace && plan->tables_cu == cu)) {
        rc = check_cuda(launch_init_tables(g, ws, plan->dm.data(), plan->fcen.data(), st, &plan->last_launches));
        if (rc) return rc;
        plan->tables_ws = plan->keep_tables ? d_workspace : nullptr;
        plan->tables_cu = cu;
    }
    // no event timing inside a stream capture (the events could not be read back), and an unread
    // record is overwritten rather than grown without bound
    bool profile = plan->profile != 0;
    if (profile) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) profile = false;
        cudaGetLastError();
        if (plan->spans.size() > PROFILE_MAX_SPANS) {
            plan->spans.clear();
            plan->ev_used = 0;
        }
    }
    auto mark = [&](size_t *idx) -> bool {
        if (!profile) return true;
        cudaEvent_t e = plan_event(plan, idx);
        return e && cudaEventRecord(e, st) == cudaSuccess;
    };
    bool sums_done = true;   // cleared by a fused launch that cannot take the block sums itself
    for (long long u0 = 0; u0 < nunits; u0 += cu) {
        const int n = (int)((nunits - u0 < cu) ? nunits - u0 : cu);
        float2 *spec = d_spec_out ? d_spec_out + (size_t)u0 * 2 * g.nfft : ws.spec;
        size_t a = 0, b = 0, c = 0;
        if (!mark(&a)) return check_cuda(cudaErrorUnknown);
        rc = check_cuda(launch_forward(g, ws, d_in, in_stride_pol, (int)u0, n, spec, st, &plan->last_launches));
        if (rc) return rc;
        if (!mark(&b)) return check_cuda(cudaErrorUnknown);
        if (profile) plan->spans.push_back({a, b, 0});
        if (d_out) {
            bool chunk_sums = true;
            rc = check_cuda(launch_fused(g, ws, spec, (int)u0, n, d_out, out_stride_dm, out_pitch, plan->dm_tile,
                                         plan->accurate, plan->force_generic, plan->dm.data(),
                                         plan->fcen.data(), d_segsum, (int)nb, &chunk_sums, st,
                                         &plan->last_launches));
            if (rc) return rc;
            sums_done = sums_done && chunk_sums;
            if (!mark(&c)) return check_cuda(cudaErrorUnknown);
            if (profile) plan->spans.push_back({b, c, 1});
        }
    }
    if (d_out && d_segsum && !sums_done)
        return check_cuda(launch_block_sums(g, d_out, out_stride_dm, nb, d_segsum, st, &plan->last_launches));
    return CDMT_OK;
}

// Sum of the event-timed kernel durations recorded since the last read (CDMT_OPT_PROFILE = 1).
// Synchronises on the recorded events.
extern "C" int cdmt_profile_read(cdmt_plan *plan, double *ms_forward, double *ms_fused, long long *n_forward,
                                 long long *n_fused)
{
    if (!plan) return CDMT_ERR_ARG;
    double t[2] = {0.0, 0.0};
    long long n[2] = {0, 0};
    int rc = CDMT_OK;
    for (const cdmt_plan::Span &sp : plan->spans) {
        float ms = 0.f;
        if (cudaEventSynchronize(plan->ev_pool[sp.e1]) != cudaSuccess ||
            cudaEventElapsedTime(&ms, plan->ev_pool[sp.e0], plan->ev_pool[sp.e1]) != cudaSuccess) {
            rc = check_cuda(cudaErrorUnknown);
            break;
        }
        t[sp.kind] += ms;
        n[sp.kind] += 1;
    }
    plan->spans.clear();
    plan->ev_used = 0;
    if (ms_forward) *ms_forward = t[0];
    if (ms_fused) *ms_fused = t[1];
    if (n_forward) *n_forward = n[0];
    if (n_fused) *n_fused = n[1];
    return rc;
}

extern "C" int cdmt_execute(cdmt_plan *plan, const void *d_in, long long nsamp, long long in_stride_pol,
                            float *d_out, long long out_stride_dm, void *d_workspace, size_t workspace_bytes,
                            void *cuda_stream)
{
    long long nb = 0;
    int rc = validate_input(plan, d_in, nsamp, in_stride_pol, &nb);
    if (rc) return rc;
    if (!d_out || !d_workspace) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_workspace) & 255) != 0) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_out) & 3) != 0) return CDMT_ERR_ARG;
    const Geometry &g = plan->g;
    if (out_stride_dm < nb * g.vdec * (long long)g.nsub * g.nchan) return CDMT_ERR_SIZE;
    return run_chunks(plan, d_in, in_stride_pol, nb, d_out, out_stride_dm, nullptr, d_workspace, workspace_bytes,
                      static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int cdmt_execute_sums(cdmt_plan *plan, const void *d_in, long long nsamp, long long in_stride_pol,
                                 float *d_out, long long out_stride_dm, double *d_segsum, void *d_workspace,
                                 size_t workspace_bytes, void *cuda_stream)
{
    long long nb = 0;
    int rc = validate_input(plan, d_in, nsamp, in_stride_pol, &nb);
    if (rc) return rc;
    if (!d_out || !d_workspace || !d_segsum) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_workspace) & 255) != 0) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_out) & 3) != 0 || (reinterpret_cast<uintptr_t>(d_segsum) & 15) != 0)
        return CDMT_ERR_ARG;
    const Geometry &g = plan->g;
    if (out_stride_dm < nb * g.vdec * (long long)g.nsub * g.nchan) return CDMT_ERR_SIZE;
    if (nb > 65535 || g.ndm > 65535) return CDMT_ERR_SIZE;   // grid limits of the stand-alone block-sum pass
    return run_chunks(plan, d_in, in_stride_pol, nb, d_out, out_stride_dm, nullptr, d_workspace, workspace_bytes,
                      static_cast<cudaStream_t>(cuda_stream), d_segsum);
}

extern "C" int cdmt_forward_spectrum(cdmt_plan *plan, const void *d_in, long long nsamp, long long in_stride_pol,
                                     void *d_spec, void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    long long nb = 0;
    int rc = validate_input(plan, d_in, nsamp, in_stride_pol, &nb);
    if (rc) return rc;
    if (!d_spec || !d_workspace) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_workspace) & 255) != 0) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_spec) & 15) != 0) return CDMT_ERR_ARG;
    return run_chunks(plan, d_in, in_stride_pol, nb, nullptr, 0, reinterpret_cast<float2 *>(d_spec), d_workspace,
                      workspace_bytes, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int cdmt_unpack(cdmt_plan *plan, const void *d_in, long long nsamp, long long in_stride_pol,
                           void *d_blocks, void *cuda_stream)
{
    long long nb = 0;
    int rc = validate_input(plan, d_in, nsamp, in_stride_pol, &nb, true);
    if (rc) return rc;
    if (!d_blocks || (reinterpret_cast<uintptr_t>(d_blocks) & 15) != 0) return CDMT_ERR_ARG;
    plan->last_launches = 0;
    return check_cuda(launch_unpack(plan->g, d_in, in_stride_pol, (int)nb, reinterpret_cast<float2 *>(d_blocks),
                                    static_cast<cudaStream_t>(cuda_stream), &plan->last_launches));
}

// ---- host-buffer path --------------------------------------------------------------------
// the observation is streamed through the GPU in groups of
// blocks, and the paper's measured bottleneck is this traffic, not the kernels.  Input and
// output staging buffers are doubled: the host-to-device copy of group i+1 and the
// device-to-host copy of group i-1 run on their own streams while group i computes.

// blocks per staged group: keep the staged output near 1 GiB, and the number of blocks even (the
// warp-specialised fused kernel works on pairs of blocks)
static long long host_group_blocks(const cdmt_plan *plan, long long nb)
{
    const Geometry &g = plan->g;
    const long long per_block = (long long)g.ndm * g.vdec * g.nsub * g.nchan * (long long)sizeof(float);
    long long gb = (1LL << 30) / (per_block > 0 ? per_block : 1);
    if (gb < 2) gb = 2;
    gb -= gb & 1;
    if (plan->host_group > 0) gb = plan->host_group;
    if (gb < 1) gb = 1;
    if (gb > nb) gb = nb;
    return gb;
}

struct HostLayout {
    size_t in_off[2], in_bytes, ws_off, ws_bytes, out_off[2], out_bytes, total;
    // CDMT_OUT_U8 only: one float32 filterbank buffer, block sums, doubled code and offset/scale buffers
    size_t sums_off, sums_bytes, codes_off[2], codes_bytes, osc_off[2], osc_bytes;
    long long gb, in_rowlen, ngroup;
};

static int host_layout(const cdmt_plan *plan, long long nsamp, int out_kind, HostLayout *L)
{
    const Geometry &g = plan->g;
    const long long nb = nblock_for(g, nsamp);
    if (nb < 1) return CDMT_ERR_SIZE;
    if (out_kind != CDMT_OUT_F32 && out_kind != CDMT_OUT_U8) return CDMT_ERR_ARG;
    const long long esz = in_word_bytes(g.in_dtype), rps = in_rows_per_sub(g.in_dtype);
    L->gb = host_group_blocks(plan, nb);
    L->ngroup = (nb + L->gb - 1) / L->gb;
    long long rowlen = (L->gb - 1) * g.step + g.nfft;
    rowlen = (rowlen + 15) & ~15LL;  // keep rows 16-byte aligned for every word size
    L->in_rowlen = rowlen;
    auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
    const int nbuf = L->gb < nb ? 2 : 1;  // a single group needs no second buffer
    L->in_bytes = al((size_t)rowlen * esz * rps * g.nsub);
    L->in_off[0] = 0;
    L->in_off[1] = nbuf == 2 ? L->in_bytes : 0;
    L->ws_off = L->in_bytes * nbuf;
    const long long cu = chunk_units_for(plan, L->gb * g.nsub);
    L->ws_bytes = al(workspace_layout(g, (int)cu, nullptr, nullptr));
    const size_t samples = (size_t)g.ndm * L->gb * g.vdec * g.nsub * g.nchan;
    L->out_bytes = al(samples * sizeof(float));
    L->out_off[0] = L->ws_off + L->ws_bytes;
    if (out_kind == CDMT_OUT_F32) {
        L->out_off[1] = nbuf == 2 ? L->out_off[0] + L->out_bytes : L->out_off[0];
        L->total = L->out_off[0] + L->out_bytes * nbuf;
        L->sums_off = L->sums_bytes = L->codes_bytes = L->osc_bytes = 0;
        L->codes_off[0] = L->codes_off[1] = L->osc_off[0] = L->osc_off[1] = 0;
        return CDMT_OK;
    }
    if (L->gb > 65535 || g.ndm > 65535 || L->gb * g.vdec > 65535LL * 16) return CDMT_ERR_SIZE;
    L->out_off[1] = L->out_off[0];
    L->sums_off = L->out_off[0] + L->out_bytes;
    L->sums_bytes = al(redigitize_workspace_bytes(g, L->gb));
    L->codes_bytes = al(samples);
    L->codes_off[0] = L->sums_off + L->sums_bytes;
    L->codes_off[1] = nbuf == 2 ? L->codes_off[0] + L->codes_bytes : L->codes_off[0];
    L->osc_bytes = al((size_t)2 * g.ndm * g.nsub * g.nchan * sizeof(float));
    L->osc_off[0] = L->codes_off[0] + L->codes_bytes * nbuf;
    L->osc_off[1] = nbuf == 2 ? L->osc_off[0] + L->osc_bytes : L->osc_off[0];
    L->total = L->osc_off[0] + L->osc_bytes * nbuf;
    return CDMT_OK;
}

extern "C" int cdmt_host_layout(const cdmt_plan *plan, long long nsamp, int out_kind, size_t *scratch_bytes,
                                int *ngroups, int *group_blocks, size_t *h2d_bytes, size_t *d2h_bytes)
{
    if (!plan) return CDMT_ERR_ARG;
    HostLayout L;
    int rc = host_layout(plan, nsamp, out_kind, &L);
    if (rc) return rc;
    const Geometry &g = plan->g;
    const long long nb = nblock_for(g, nsamp);
    const size_t esz = (size_t)in_word_bytes(g.in_dtype), rps = (size_t)in_rows_per_sub(g.in_dtype);
    size_t in = 0;
    for (long long b0 = 0; b0 < nb; b0 += L.gb) {
        const long long nbg = (nb - b0 < L.gb) ? nb - b0 : L.gb;
        in += (size_t)((nbg - 1) * g.step + g.nfft) * esz * rps * g.nsub;
    }
    const size_t samples = (size_t)g.ndm * (size_t)(nb * g.vdec) * (size_t)g.nsub * g.nchan;
    if (scratch_bytes) *scratch_bytes = L.total;
    if (ngroups) *ngroups = (int)L.ngroup;
    if (group_blocks) *group_blocks = (int)L.gb;
    if (h2d_bytes) *h2d_bytes = in;
    if (d2h_bytes)
        *d2h_bytes = out_kind == CDMT_OUT_F32
                         ? samples * sizeof(float)
                         : samples + (size_t)L.ngroup * 2 * g.ndm * g.nsub * g.nchan * sizeof(float);
    return CDMT_OK;
}

extern "C" int cdmt_host_scratch_bytes(const cdmt_plan *plan, long long nsamp, size_t *scratch_bytes)
{
    if (!scratch_bytes) return CDMT_ERR_ARG;
    return cdmt_host_layout(plan, nsamp, CDMT_OUT_F32, scratch_bytes, nullptr, nullptr, nullptr, nullptr);
}

extern "C" int cdmt_host_traffic_bytes(const cdmt_plan *plan, long long nsamp, size_t *h2d_bytes, size_t *d2h_bytes)
{
    return cdmt_host_layout(plan, nsamp, CDMT_OUT_F32, nullptr, nullptr, nullptr, h2d_bytes, d2h_bytes);
}

// `height` rows of `width` bytes between pitched buffers.  cudaMemcpy2DAsync rejects pitches above
// cudaDeviceProp::memPitch (2^31 - 1 bytes), which a long observation exceeds: then one copy per row.
static cudaError_t copy_rows_async(void *dst, size_t dpitch, const void *src, size_t spitch, size_t width,
                                   size_t height, cudaMemcpyKind kind, cudaStream_t st)
{
    const size_t lim = 0x7fffffffu;
    if (dpitch <= lim && spitch <= lim) return cudaMemcpy2DAsync(dst, dpitch, src, spitch, width, height, kind, st);
    for (size_t r = 0; r < height; ++r) {
        cudaError_t e = cudaMemcpyAsync(static_cast<char *>(dst) + r * dpitch, static_cast<const char *>(src) + r * spitch,
                                        width, kind, st);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

extern "C" int cdmt_execute_host_async(cdmt_plan *plan, const void *h_in, long long nsamp, long long in_stride_pol,
                                       int out_kind, void *h_out, float *h_offset, float *h_scale, double qmean,
                                       double qstd, void *d_scratch, size_t scratch_bytes, void *cuda_stream)
{
    if (!plan || !h_in || !h_out || !d_scratch) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_scratch) & 255) != 0) return CDMT_ERR_ARG;
    const bool u8 = out_kind == CDMT_OUT_U8;
    if (u8 && (!h_offset || !h_scale || !(qstd > 0.0) || !std::isfinite(qstd) || !std::isfinite(qmean)))
        return CDMT_ERR_ARG;
    const Geometry &g = plan->g;
    if (nsamp < g.nfft || in_stride_pol < nsamp) return CDMT_ERR_SIZE;
    HostLayout L;
    int rc = host_layout(plan, nsamp, out_kind, &L);
    if (rc) return rc;
    if (scratch_bytes < L.total) return CDMT_ERR_WORKSPACE;
    if (!plan_host_pipeline(plan)) return check_cuda(cudaErrorUnknown);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const long long nb = nblock_for(g, nsamp);
    const long long esz = in_word_bytes(g.in_dtype), rps = in_rows_per_sub(g.in_dtype);
    char *base = reinterpret_cast<char *>(d_scratch);
    const size_t nchtot = (size_t)g.nsub * g.nchan;
    const size_t plane_host = (size_t)nb * g.vdec * nchtot;
    const size_t osz = u8 ? 1 : sizeof(float);
    const long long ngroup = L.ngroup;
    long long launches = 0;
    // the scratch workspace is ours for the whole call: its tables are written by the first group only
    const int keep_saved = plan->keep_tables;
    const void *ws_saved = plan->tables_ws;
    plan->keep_tables = 1;
    plan->tables_ws = nullptr;

    // the copy streams start after whatever the caller queued on `st` before this call
    rc = check_cuda(cudaEventRecord(plan->ev_start, st));
    if (!rc) rc = check_cuda(cudaStreamWaitEvent(plan->s_in, plan->ev_start, 0));
    if (!rc) rc = check_cuda(cudaStreamWaitEvent(plan->s_out, plan->ev_start, 0));

    auto h2d = [&](long long i) -> int {
        const int k = (int)(i & 1);
        const long long b0 = i * L.gb;
        const long long nbg = (nb - b0 < L.gb) ? nb - b0 : L.gb;
        const long long len = (nbg - 1) * g.step + g.nfft;
        // buffer k was last read by the kernels of group i-2
        if (i >= 2) {
            int r = check_cuda(cudaStreamWaitEvent(plan->s_in, plan->ev_comp[k], 0));
            if (r) return r;
        }
        int r = check_cuda(copy_rows_async(base + L.in_off[k], (size_t)L.in_rowlen * esz,
                                           reinterpret_cast<const char *>(h_in) + (size_t)b0 * g.step * esz,
                                           (size_t)in_stride_pol * esz, (size_t)len * esz, (size_t)rps * g.nsub,
                                           cudaMemcpyHostToDevice, plan->s_in));
        if (r) return r;
        return check_cuda(cudaEventRecord(plan->ev_h2d[k], plan->s_in));
    };

    if (!rc) rc = h2d(0);
    for (long long i = 0; i < ngroup && !rc; ++i) {
        const int k = (int)(i & 1);
        const long long b0 = i * L.gb;
        const long long nbg = (nb - b0 < L.gb) ? nb - b0 : L.gb;
        const size_t plane_dev = (size_t)nbg * g.vdec * nchtot;
        float *d_out = reinterpret_cast<float *>(base + L.out_off[k]);
        // compute of group i: needs its input, and the buffer the copy of group i-2 read from
        rc = check_cuda(cudaStreamWaitEvent(st, plan->ev_h2d[k], 0));
        if (!rc && i >= 2) rc = check_cuda(cudaStreamWaitEvent(st, plan->ev_d2h[k], 0));
        if (rc) break;
        double *d_sums = u8 ? reinterpret_cast<double *>(base + L.sums_off) : nullptr;
        rc = run_chunks(plan, base + L.in_off[k], L.in_rowlen, nbg, d_out, (long long)plane_dev, nullptr,
                        base + L.ws_off, L.ws_bytes, st, d_sums);
        if (rc) break;
        launches += plan->last_launches;
        unsigned char *d_codes = reinterpret_cast<unsigned char *>(base + L.codes_off[k]);
        float *d_off = reinterpret_cast<float *>(base + L.osc_off[k]), *d_sc = d_off + (size_t)g.ndm * nchtot;
        if (u8) {
            // Alg. 1 l.105-106 on the batch just computed (its block sums came with the filterbank)
            rc = check_cuda(launch_stats_quantize(g, d_out, (long long)plane_dev, nbg, qmean, qstd, d_sums, d_codes,
                                                  (long long)plane_dev, d_off, d_sc, st, &launches));
            if (rc) break;
        }
        rc = check_cuda(cudaEventRecord(plan->ev_comp[k], st));
        if (rc) break;
        // the next group's input travels while this group computes
        if (i + 1 < ngroup) {
            rc = h2d(i + 1);
            if (rc) break;
        }
        rc = check_cuda(cudaStreamWaitEvent(plan->s_out, plan->ev_comp[k], 0));
        if (!rc)
            rc = check_cuda(copy_rows_async(static_cast<char *>(h_out) + (size_t)b0 * g.vdec * nchtot * osz, plane_host * osz,
                                            u8 ? static_cast<const void *>(d_codes) : static_cast<const void *>(d_out),
                                            plane_dev * osz, plane_dev * osz, (size_t)g.ndm, cudaMemcpyDeviceToHost,
                                            plan->s_out));
        if (!rc && u8) {
            const size_t n = (size_t)g.ndm * nchtot;
            rc = check_cuda(cudaMemcpyAsync(h_offset + (size_t)i * n, d_off, n * sizeof(float), cudaMemcpyDeviceToHost,
                                            plan->s_out));
            if (!rc)
                rc = check_cuda(cudaMemcpyAsync(h_scale + (size_t)i * n, d_sc, n * sizeof(float), cudaMemcpyDeviceToHost,
                                                plan->s_out));
        }
        if (!rc) rc = check_cuda(cudaEventRecord(plan->ev_d2h[k], plan->s_out));
    }
    plan->last_launches = launches;
    plan->keep_tables = keep_saved;
    plan->tables_ws = ws_saved;
    // join: whatever was queued on the copy streams completes before later work on `st` (also on error,
    // so that draining `st` is enough before the buffers are reused or freed)
    int rj = check_cuda(cudaEventRecord(plan->ev_join[0], plan->s_in));
    if (!rj) rj = check_cuda(cudaStreamWaitEvent(st, plan->ev_join[0], 0));
    if (!rj) rj = check_cuda(cudaEventRecord(plan->ev_join[1], plan->s_out));
    if (!rj) rj = check_cuda(cudaStreamWaitEvent(st, plan->ev_join[1], 0));
    return rc ? rc : rj;
}

extern "C" int cdmt_execute_host(cdmt_plan *plan, const void *h_in, long long nsamp, long long in_stride_pol,
                                 float *h_out, void *d_scratch, size_t scratch_bytes, void *cuda_stream)
{
    const int rc = cdmt_execute_host_async(plan, h_in, nsamp, in_stride_pol, CDMT_OUT_F32, h_out, nullptr, nullptr, 0.0,
                                           1.0, d_scratch, scratch_bytes, cuda_stream);
    if (rc == CDMT_ERR_ARG || rc == CDMT_ERR_SIZE || rc == CDMT_ERR_WORKSPACE) return rc;   // nothing was queued
    // drain whatever happened, so that the scratch can be reused or freed
    const int r1 = plan->host_ready ? check_cuda(cudaStreamSynchronize(plan->s_in)) : CDMT_OK;
    const int r2 = check_cuda(cudaStreamSynchronize(static_cast<cudaStream_t>(cuda_stream)));
    const int r3 = plan->host_ready ? check_cuda(cudaStreamSynchronize(plan->s_out)) : CDMT_OK;
    if (rc) return rc;
    return r1 ? r1 : (r2 ? r2 : r3);
}

// ---- redigitisation (Alg. 1 l.104-106) ---------------------------------------------------
extern "C" int cdmt_redigitize_workspace_bytes(const cdmt_plan *plan, long long nblock, size_t *workspace_bytes)
{
    if (!plan || !workspace_bytes) return CDMT_ERR_ARG;
    if (nblock < 1 || nblock > 65535) return CDMT_ERR_SIZE;
    *workspace_bytes = redigitize_workspace_bytes(plan->g, nblock);
    return CDMT_OK;
}

extern "C" int cdmt_redigitize(cdmt_plan *plan, const float *d_fb, long long fb_stride_dm, long long nblock,
                               double qmean, double qstd, unsigned char *d_codes, long long codes_stride_dm,
                               float *d_offset, float *d_scale, void *d_workspace, size_t workspace_bytes,
                               void *cuda_stream)
{
    if (!plan || !d_fb || !d_codes || !d_offset || !d_scale || !d_workspace) return CDMT_ERR_ARG;
    if (!(qstd > 0.0) || !std::isfinite(qstd) || !std::isfinite(qmean)) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_fb) & 3) != 0 || (reinterpret_cast<uintptr_t>(d_offset) & 3) != 0 ||
        (reinterpret_cast<uintptr_t>(d_scale) & 3) != 0 || (reinterpret_cast<uintptr_t>(d_workspace) & 255) != 0)
        return CDMT_ERR_ARG;
    const Geometry &g = plan->g;
    if (nblock < 1 || nblock > 65535 || g.ndm > 65535) return CDMT_ERR_SIZE;
    const long long plane = nblock * g.vdec * (long long)g.nsub * g.nchan;
    if (fb_stride_dm < plane || codes_stride_dm < plane) return CDMT_ERR_SIZE;
    if (nblock * g.vdec > 65535LL * 16) return CDMT_ERR_SIZE;
    if (workspace_bytes < redigitize_workspace_bytes(g, nblock)) return CDMT_ERR_WORKSPACE;
    plan->last_launches = 0;
    return check_cuda(launch_redigitize(g, d_fb, fb_stride_dm, nblock, qmean, qstd, d_codes, codes_stride_dm, d_offset,
                                        d_scale, d_workspace, static_cast<cudaStream_t>(cuda_stream),
                                        &plan->last_launches));
}

// cdmt_redigitize without a caller-supplied workspace and without any allocation: the block sums live in a
// file-scope device array of the library (cdmt_redigitize.cu) of cdmt_redigitize_static_max_bytes() bytes.
extern "C" int cdmt_redigitize_static_max_bytes(size_t *max_bytes)
{
    if (!max_bytes) return CDMT_ERR_ARG;
    *max_bytes = redigitize_static_max_bytes();
    return CDMT_OK;
}

extern "C" int cdmt_redigitize_static(cdmt_plan *plan, const float *d_fb, long long fb_stride_dm, long long nblock,
                                      double qmean, double qstd, unsigned char *d_codes, long long codes_stride_dm,
                                      float *d_offset, float *d_scale, void *cuda_stream)
{
    if (!plan || !d_fb || !d_codes || !d_offset || !d_scale) return CDMT_ERR_ARG;
    if (!(qstd > 0.0) || !std::isfinite(qstd) || !std::isfinite(qmean)) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_fb) & 3) != 0 || (reinterpret_cast<uintptr_t>(d_offset) & 3) != 0 ||
        (reinterpret_cast<uintptr_t>(d_scale) & 3) != 0)
        return CDMT_ERR_ARG;
    const Geometry &g = plan->g;
    if (nblock < 1 || nblock > 65535 || g.ndm > 65535) return CDMT_ERR_SIZE;
    const long long plane = nblock * g.vdec * (long long)g.nsub * g.nchan;
    if (fb_stride_dm < plane || codes_stride_dm < plane) return CDMT_ERR_SIZE;
    if (nblock * g.vdec > 65535LL * 16) return CDMT_ERR_SIZE;
    // the block sums of this batch must fit the library's fixed scratch: ndm * nblock * nsub*nchan * 16 bytes
    if (redigitize_workspace_bytes(g, nblock) > redigitize_static_max_bytes()) return CDMT_ERR_WORKSPACE;
    plan->last_launches = 0;
    return check_cuda(launch_redigitize_static(g, d_fb, fb_stride_dm, nblock, qmean, qstd, d_codes, codes_stride_dm,
                                               d_offset, d_scale, static_cast<cudaStream_t>(cuda_stream),
                                               &plan->last_launches));
}

extern "C" int cdmt_redigitize_sums(cdmt_plan *plan, const float *d_fb, long long fb_stride_dm, long long nblock,
                                    double qmean, double qstd, const double *d_segsum, unsigned char *d_codes,
                                    long long codes_stride_dm, float *d_offset, float *d_scale, void *cuda_stream)
{
    if (!plan || !d_fb || !d_codes || !d_offset || !d_scale || !d_segsum) return CDMT_ERR_ARG;
    if (!(qstd > 0.0) || !std::isfinite(qstd) || !std::isfinite(qmean)) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_fb) & 3) != 0 || (reinterpret_cast<uintptr_t>(d_offset) & 3) != 0 ||
        (reinterpret_cast<uintptr_t>(d_scale) & 3) != 0 || (reinterpret_cast<uintptr_t>(d_segsum) & 15) != 0)
        return CDMT_ERR_ARG;
    const Geometry &g = plan->g;
    if (nblock < 1 || nblock > 65535 || g.ndm > 65535) return CDMT_ERR_SIZE;
    const long long plane = nblock * g.vdec * (long long)g.nsub * g.nchan;
    if (fb_stride_dm < plane || codes_stride_dm < plane) return CDMT_ERR_SIZE;
    if (nblock * g.vdec > 65535LL * 16) return CDMT_ERR_SIZE;
    plan->last_launches = 0;
    return check_cuda(launch_stats_quantize(g, d_fb, fb_stride_dm, nblock, qmean, qstd, d_segsum, d_codes,
                                            codes_stride_dm, d_offset, d_scale, static_cast<cudaStream_t>(cuda_stream),
                                            &plan->last_launches));
}

// ---- incoherent dedispersion over fine DM offsets ----------------------------
static int plan_incoherent(cdmt_plan *plan, int nfine, const double *ddm)
{
    if (!plan || !ddm) return CDMT_ERR_ARG;
    if (nfine < 1 || nfine > (1 << 20)) return CDMT_ERR_SIZE;
    for (int k = 0; k < nfine; ++k)
        if (!std::isfinite(ddm[k])) return CDMT_ERR_ARG;
    if ((int)plan->ic_ddm.size() == nfine && std::memcmp(plan->ic_ddm.data(), ddm, sizeof(double) * nfine) == 0)
        return CDMT_OK;
    try {
        plan->ic_ddm.clear();
        if (!incoherent_plan(plan->g, plan->fcen.data(), nfine, ddm, &plan->ic)) return CDMT_ERR_ARG;
        // shift range beyond the shared-memory tile, or more trial groups than a grid dimension holds
        if (!incoherent_config(plan->ic, nullptr, nullptr, nullptr, nullptr, nullptr)) return CDMT_ERR_SIZE;
        plan->ic_ddm.assign(ddm, ddm + nfine);
    } catch (...) {
        plan->ic_ddm.clear();
        return CDMT_ERR_ALLOC;
    }
    return CDMT_OK;
}

extern "C" int cdmt_incoherent_query(cdmt_plan *plan, int nfine, const double *ddm, long long nt_in, int *shift_min,
                                     int *shift_range, long long *nt_out, int *ngroups, size_t *workspace_bytes)
{
    int rc = plan_incoherent(plan, nfine, ddm);
    if (rc) return rc;
    if (shift_min) *shift_min = plan->ic.smin;
    if (shift_range) *shift_range = plan->ic.range;
    if (nt_out) *nt_out = nt_in - plan->ic.range;
    if (ngroups) *ngroups = (int)plan->ic.groups.size();
    if (workspace_bytes) *workspace_bytes = incoherent_workspace_bytes(plan->ic);
    return CDMT_OK;
}

extern "C" int cdmt_incoherent_shifts(cdmt_plan *plan, int nfine, const double *ddm, int *h_shifts)
{
    if (!h_shifts) return CDMT_ERR_ARG;
    int rc = plan_incoherent(plan, nfine, ddm);
    if (rc) return rc;
    std::memcpy(h_shifts, plan->ic.shifts.data(), sizeof(int) * plan->ic.shifts.size());
    return CDMT_OK;
}

extern "C" int cdmt_incoherent_dedisperse(cdmt_plan *plan, const float *d_fb, long long fb_stride_dm, long long nt_in,
                                          int nfine, const double *ddm, float *d_ts, long long ts_stride_dm,
                                          long long ts_pitch, void *d_workspace, size_t workspace_bytes,
                                          void *cuda_stream)
{
    if (!plan || !d_fb || !d_ts || !d_workspace) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_fb) & 3) != 0 || (reinterpret_cast<uintptr_t>(d_ts) & 3) != 0 ||
        (reinterpret_cast<uintptr_t>(d_workspace) & 255) != 0)
        return CDMT_ERR_ARG;
    int rc = plan_incoherent(plan, nfine, ddm);
    if (rc) return rc;
    const Geometry &g = plan->g;
    const long long nch = (long long)g.nsub * g.nchan;
    const long long nt_out = nt_in - plan->ic.range;
    if (nt_in < 1 || nt_in > (1LL << 30) || nt_out < 1) return CDMT_ERR_SIZE;
    if (fb_stride_dm < nt_in * nch || ts_pitch < nt_out || ts_stride_dm < (long long)nfine * ts_pitch) return CDMT_ERR_SIZE;
    if (g.ndm > 65535) return CDMT_ERR_SIZE;
    if (workspace_bytes < incoherent_workspace_bytes(plan->ic)) return CDMT_ERR_WORKSPACE;
    plan->last_launches = 0;
    return check_cuda(launch_incoherent(g, plan->ic, d_fb, fb_stride_dm, nt_in, d_ts, ts_stride_dm, ts_pitch,
                                        d_workspace, static_cast<cudaStream_t>(cuda_stream), &plan->last_launches));
}

extern "C" int cdmt_incoherent_work(cdmt_plan *plan, int nfine, const double *ddm, long long nt_in,
                                    double *adds_definition, double *adds_performed)
{
    int rc = plan_incoherent(plan, nfine, ddm);
    if (rc) return rc;
    const IncoherentTables &T = plan->ic;
    const double nt_out = (double)(nt_in - T.range);
    if (nt_out < 1.0) return CDMT_ERR_SIZE;
    double steps = 0.0, run_ends = 0.0;
    for (const uint2 &e : T.entries) {
        steps += 1.0 + (double)((e.x >> 24) & 7u);
        if (e.x & (1u << 28)) run_ends += 1.0;
    }
    if (adds_definition) *adds_definition = (double)plan->g.ndm * nfine * T.nch * nt_out;
    if (adds_performed) *adds_performed = (double)plan->g.ndm * nt_out * (steps + 8.0 * run_ends);
    return CDMT_OK;
}

// Streaming the incoherent stage over block groups (the filterbanks of a 20-minute
// observation are never resident at once): the last `shift_range` rows of every plane become the first.
extern "C" int cdmt_incoherent_carry(cdmt_plan *plan, float *d_fb, long long fb_stride_dm, long long nt_in,
                                     int shift_range, void *cuda_stream)
{
    if (!plan || !d_fb || (reinterpret_cast<uintptr_t>(d_fb) & 3) != 0) return CDMT_ERR_ARG;
    const Geometry &g = plan->g;
    const long long nch = (long long)g.nsub * g.nchan;
    if (shift_range < 0 || nt_in < 2LL * shift_range || fb_stride_dm < nt_in * nch) return CDMT_ERR_SIZE;
    if (g.ndm > 65535) return CDMT_ERR_SIZE;
    plan->last_launches = 0;
    return check_cuda(launch_carry_rows(d_fb, fb_stride_dm, nt_in, shift_range, (int)nch, g.ndm,
                                        static_cast<cudaStream_t>(cuda_stream), &plan->last_launches));
}

// n_d n_c >= r t_d for the lowest-frequency channel (or subband) at the largest |DM|.
extern "C" long long cdmt_min_overlap(const cdmt_plan *plan)
{
    if (!plan) return -1;
    const Geometry &g = plan->g;
    double dmax = 0.0;
    for (double d : plan->dm) dmax = std::fabs(d) > dmax ? std::fabs(d) : dmax;
    double fmin = plan->fcen[0];
    for (double f : plan->fcen) fmin = f < fmin ? f : fmin;
    double td;
    if (g.chirp_ref == CDMT_REF_CHANNEL) {
        const double cw = g.bw_mhz / g.nchan;
        td = cdmt_sweep_seconds(fmin - 0.5 * g.bw_mhz + 0.5 * cw, cw, dmax);
    } else {
        td = cdmt_sweep_seconds(fmin, g.bw_mhz, dmax);
    }
    const long long samples = (long long)std::ceil(td * g.bw_mhz * 1e6);
    const long long q = 2LL * g.nchan;
    return (samples + q - 1) / q * q;
}

// N_bin and n_d follow from the dispersion sweep (Eq. 2) of the lowest channel
// at the largest DM; the paper fixes one pair for all subbands and names that as an inefficiency.
extern "C" int cdmt_suggest_sizes(int nsub, const double *fcen_mhz, double bw_mhz, int nchan, int ndec,
                                  double dm_max_abs, int chirp_ref, double min_efficiency, int *nfft, int *noverlap)
{
    if (!fcen_mhz || !nfft || !noverlap || nsub < 1) return CDMT_ERR_ARG;
    if (!(bw_mhz > 0.0) || !std::isfinite(bw_mhz) || !std::isfinite(dm_max_abs) || dm_max_abs < 0.0) return CDMT_ERR_ARG;
    if (!(min_efficiency > 0.0) || !(min_efficiency < 1.0)) return CDMT_ERR_ARG;
    if (chirp_ref != CDMT_REF_CHANNEL && chirp_ref != CDMT_REF_SUBBAND) return CDMT_ERR_ARG;
    if (!is_pow2(nchan) || ndec < 1) return CDMT_ERR_SIZE;
    double fmin = fcen_mhz[0];
    for (int s = 0; s < nsub; ++s) {
        if (!std::isfinite(fcen_mhz[s]) || !(fcen_mhz[s] - 0.5 * bw_mhz > 0.0)) return CDMT_ERR_ARG;
        fmin = fcen_mhz[s] < fmin ? fcen_mhz[s] : fmin;
    }
    double td;
    if (chirp_ref == CDMT_REF_CHANNEL) {
        const double cw = bw_mhz / nchan;
        td = cdmt_sweep_seconds(fmin - 0.5 * bw_mhz + 0.5 * cw, cw, dm_max_abs);
    } else {
        td = cdmt_sweep_seconds(fmin, bw_mhz, dm_max_abs);
    }
    const long long sweep = (long long)std::ceil(td * bw_mhz * 1e6);   // input samples (r t_d)
    // noverlap: a multiple of 2 nchan ndec -- half per edge, and each half a whole number of INTEGRATED
    // samples (what the packed fused kernels need; it also satisfies the plan's two divisibility rules)
    const long long unit = 2LL * nchan * ndec, r = (long long)nchan * ndec;
    const long long ov = (sweep + unit - 1) / unit * unit;
    // nfft: smallest power of two whose kept fraction reaches min_efficiency and that the kernels support
    for (long long n = 256; n <= (1LL << 20); n <<= 1) {
        if (n % nchan || !fused_len_supported((int)(n / nchan))) continue;
        if (n % r) continue;
        if (ov >= n) continue;
        if ((double)(n - ov) < min_efficiency * (double)n) continue;
        const int lg = ilog2(n);
        if (!forward_len_supported(1 << ((lg + 1) / 2)) || !forward_len_supported((int)(n >> ((lg + 1) / 2)))) continue;
        *nfft = (int)n;
        *noverlap = (int)ov;
        return CDMT_OK;
    }
    return CDMT_ERR_SIZE;
}

// ---- per-group sizes inside the library (N4) ------------------------------------------------
// PAPER.md:79 fixes one (N_bin, n_d) for all subbands, "chosen for the lowest observing frequency of the
// input data and highest DM", and names that as the program's own inefficiency next to
// digifil.  A multiplan cuts the subbands into contiguous groups, sizes each from Eq. 2 (cdmt_suggest_sizes)
// and runs them one after the other into ONE filterbank: every group starts reading its input at the sample
// that puts its first output sample at the same time as the others', so the rows line up.
struct cdmt_multiplan {
    std::vector<cdmt_plan *> plans;      // one per group, ascending frequency
    std::vector<int> sub0, nsubg;        // subband range of each group
    int nsub, nchan, ndec, ndm, in_dtype;
    long long last_launches;
};

struct MultiSizes {
    std::vector<long long> delta, nblock, rows;   // first input sample, blocks and output rows of each group
    long long rows_valid, rows_alloc;
    size_t workspace;
    double kept;                                  // kept fraction of the input, subband-weighted
};

static int multi_sizes(const cdmt_multiplan *mp, long long nsamp, MultiSizes *z)
{
    const size_t ng = mp->plans.size();
    long long tstart = 0;
    for (const cdmt_plan *p : mp->plans) tstart = std::max<long long>(tstart, p->g.noverlap / 2);
    z->delta.resize(ng); z->nblock.resize(ng); z->rows.resize(ng);
    z->rows_valid = -1; z->rows_alloc = 0; z->workspace = 0; z->kept = 0.0;
    for (size_t i = 0; i < ng; ++i) {
        const cdmt_plan *p = mp->plans[i];
        const Geometry &g = p->g;
        z->delta[i] = tstart - g.noverlap / 2;
        const long long nb = nblock_for(g, nsamp - z->delta[i]);
        if (nb < 1 || nb * g.nsub > (1LL << 30)) return CDMT_ERR_SIZE;
        z->nblock[i] = nb;
        z->rows[i] = nb * g.vdec;
        z->rows_valid = z->rows_valid < 0 ? z->rows[i] : std::min(z->rows_valid, z->rows[i]);
        z->rows_alloc = std::max(z->rows_alloc, z->rows[i]);
        const long long cu = chunk_units_for(p, nb * g.nsub);
        z->workspace = std::max(z->workspace, workspace_layout(g, (int)cu, nullptr, nullptr));
        z->kept += (double)g.nsub * (double)g.step / (double)g.nfft;
    }
    z->kept /= (double)mp->nsub;
    return CDMT_OK;
}

extern "C" int cdmt_multiplan_destroy(cdmt_multiplan *mp)
{
    if (!mp) return CDMT_ERR_ARG;
    for (cdmt_plan *p : mp->plans) cdmt_plan_destroy(p);
    delete mp;
    return CDMT_OK;
}

extern "C" int cdmt_multiplan_create(cdmt_multiplan **mplan, int nsub, const double *fcen_mhz, double bw_mhz, int nchan,
                                     int ndec, int ndm, const double *dm, int in_dtype, int chirp_ref,
                                     double min_efficiency, int max_groups)
{
    if (!mplan) return CDMT_ERR_ARG;
    *mplan = nullptr;
    if (!fcen_mhz || !dm || nsub < 1 || ndm < 1 || max_groups < 1) return CDMT_ERR_ARG;
    for (int s = 1; s < nsub; ++s)
        if (!(fcen_mhz[s] > fcen_mhz[s - 1])) return CDMT_ERR_ARG;   // groups are contiguous in frequency
    double dmax = 0.0;
    for (int d = 0; d < ndm; ++d) {
        if (!std::isfinite(dm[d])) return CDMT_ERR_ARG;
        dmax = std::max(dmax, std::fabs(dm[d]));
    }
    try {
        // nfft as the paper chooses it: from the lowest subband at the largest DM.  Every group
        // keeps that nfft (the same kernels run everywhere) and takes the overlap Eq. 2 asks for at ITS lowest
        // subband; the cuts are the ones that keep most of the input: minimise sum_g n_g noverlap_g over all
        // partitions into at most max_groups contiguous groups (dynamic programme over the subbands).
        int nfft0 = 0, nov0 = 0;
        int rc0 = cdmt_suggest_sizes(nsub, fcen_mhz, bw_mhz, nchan, ndec, dmax, chirp_ref, min_efficiency, &nfft0, &nov0);
        if (rc0) return rc0;
        std::vector<int> nov((size_t)nsub);
        for (int s = 0; s < nsub; ++s) {
            int nf = 0;
            rc0 = cdmt_suggest_sizes(1, fcen_mhz + s, bw_mhz, nchan, ndec, dmax, chirp_ref, 1e-6, &nf, &nov[s]);
            if (rc0) return rc0;
        }
        struct Grp { int s0, n, nfft, nov; };
        std::vector<Grp> grp;
        const int G = std::min(max_groups, nsub);
        if (nsub > 8192) {
            // very wide bands: even cuts (the programme above is quadratic in nsub)
            for (int g = 0; g < G; ++g) {
                const int a = (int)((long long)nsub * g / G), b = (int)((long long)nsub * (g + 1) / G);
                grp.push_back({a, b - a, nfft0, nov[a]});
            }
        } else {
            const double INF = 1e300;
            std::vector<std::vector<double>> cost((size_t)G + 1, std::vector<double>((size_t)nsub + 1, INF));
            std::vector<std::vector<int>> from((size_t)G + 1, std::vector<int>((size_t)nsub + 1, -1));
            cost[0][0] = 0.0;
            for (int g = 1; g <= G; ++g)
                for (int j = 1; j <= nsub; ++j)
                    for (int i = g - 1; i < j; ++i) {
                        if (cost[g - 1][i] >= INF) continue;
                        const double c = cost[g - 1][i] + (double)(j - i) * (double)nov[i];
                        if (c < cost[g][j]) { cost[g][j] = c; from[g][j] = i; }
                    }
            int gbest = 1;
            for (int g = 2; g <= G; ++g)
                if (cost[g][nsub] < cost[gbest][nsub]) gbest = g;
            std::vector<int> cuts;
            for (int g = gbest, j = nsub; g >= 1; --g) {
                cuts.push_back(from[g][j]);
                j = from[g][j];
            }
            std::reverse(cuts.begin(), cuts.end());
            for (size_t k = 0; k < cuts.size(); ++k) {
                const int a = cuts[k], b = k + 1 < cuts.size() ? cuts[k + 1] : nsub;
                if (!grp.empty() && nov[a] == grp.back().nov) grp.back().n += b - a;   // same overlap: one group
                else grp.push_back({a, b - a, nfft0, nov[a]});
            }
        }
        cdmt_multiplan *mp = new cdmt_multiplan();
        mp->nsub = nsub; mp->nchan = nchan; mp->ndec = ndec; mp->ndm = ndm; mp->in_dtype = in_dtype; mp->last_launches = 0;
        for (const Grp &g : grp) {
            cdmt_plan *p = nullptr;
            const int rc = cdmt_plan_create(&p, g.n, fcen_mhz + g.s0, bw_mhz, g.nfft, g.nov, nchan, ndec, ndm, dm, in_dtype,
                                            chirp_ref);
            if (rc) {
                cdmt_multiplan_destroy(mp);
                return rc;
            }
            mp->plans.push_back(p);
            mp->sub0.push_back(g.s0);
            mp->nsubg.push_back(g.n);
        }
        *mplan = mp;
    } catch (...) {
        return CDMT_ERR_ALLOC;
    }
    return CDMT_OK;
}

extern "C" int cdmt_multiplan_query(const cdmt_multiplan *mp, long long nsamp, int *ngroups, long long *nout_valid,
                                    long long *nout_alloc, size_t *out_bytes, size_t *workspace_bytes,
                                    double *kept_fraction)
{
    if (!mp) return CDMT_ERR_ARG;
    MultiSizes z;
    const int rc = multi_sizes(mp, nsamp, &z);
    if (rc) return rc;
    if (ngroups) *ngroups = (int)mp->plans.size();
    if (nout_valid) *nout_valid = z.rows_valid;
    if (nout_alloc) *nout_alloc = z.rows_alloc;
    if (out_bytes) *out_bytes = (size_t)mp->ndm * (size_t)z.rows_alloc * (size_t)mp->nsub * mp->nchan * sizeof(float);
    if (workspace_bytes) *workspace_bytes = z.workspace;
    if (kept_fraction) *kept_fraction = z.kept;
    return CDMT_OK;
}

extern "C" int cdmt_multiplan_group(const cdmt_multiplan *mp, int group, long long nsamp, int *first_subband, int *nsub,
                                    int *nfft, int *noverlap, long long *first_sample, long long *nout)
{
    if (!mp || group < 0 || group >= (int)mp->plans.size()) return CDMT_ERR_ARG;
    MultiSizes z;
    const int rc = multi_sizes(mp, nsamp, &z);
    if (rc) return rc;
    const Geometry &g = mp->plans[group]->g;
    if (first_subband) *first_subband = mp->sub0[group];
    if (nsub) *nsub = g.nsub;
    if (nfft) *nfft = g.nfft;
    if (noverlap) *noverlap = g.noverlap;
    if (first_sample) *first_sample = z.delta[group];
    if (nout) *nout = z.rows[group];
    return CDMT_OK;
}

extern "C" int cdmt_multiplan_execute(cdmt_multiplan *mp, const void *d_in, long long nsamp, long long in_stride_pol,
                                      float *d_out, long long out_stride_dm, void *d_workspace, size_t workspace_bytes,
                                      void *cuda_stream)
{
    if (!mp || !d_in || !d_out || !d_workspace) return CDMT_ERR_ARG;
    if ((reinterpret_cast<uintptr_t>(d_workspace) & 255) != 0 || (reinterpret_cast<uintptr_t>(d_out) & 3) != 0)
        return CDMT_ERR_ARG;
    const uintptr_t word = (uintptr_t)in_word_bytes(mp->in_dtype), rps = (uintptr_t)in_rows_per_sub(mp->in_dtype);
    if ((reinterpret_cast<uintptr_t>(d_in) & (word - 1)) != 0) return CDMT_ERR_ARG;
    if (in_stride_pol < nsamp) return CDMT_ERR_SIZE;
    MultiSizes z;
    int rc = multi_sizes(mp, nsamp, &z);
    if (rc) return rc;
    const long long pitch = (long long)mp->nsub * mp->nchan;
    if (pitch > 0x7fffffffLL || out_stride_dm < z.rows_alloc * pitch) return CDMT_ERR_SIZE;
    if (workspace_bytes < z.workspace) return CDMT_ERR_WORKSPACE;
    mp->last_launches = 0;
    for (size_t i = 0; i < mp->plans.size(); ++i) {
        cdmt_plan *p = mp->plans[i];
        const char *in = static_cast<const char *>(d_in) + ((size_t)rps * mp->sub0[i] * (size_t)in_stride_pol + (size_t)z.delta[i]) * word;
        // descending frequency: the highest group comes first in a row
        float *out = d_out + (size_t)(mp->nsub - mp->sub0[i] - mp->nsubg[i]) * mp->nchan;
        rc = run_chunks(p, in, in_stride_pol, z.nblock[i], out, out_stride_dm, nullptr, d_workspace, workspace_bytes,
                        static_cast<cudaStream_t>(cuda_stream), nullptr, (int)pitch);
        mp->last_launches += p->last_launches;
        if (rc) return rc;
    }
    return CDMT_OK;
}

extern "C" long long cdmt_multiplan_last_launch_count(const cdmt_multiplan *mp) { return mp ? mp->last_launches : -1; }

extern "C" long long cdmt_last_launch_count(const cdmt_plan *plan) { return plan ? plan->last_launches : -1; }

extern "C" int cdmt_measure_fp32_peak(void *d_scratch, size_t scratch_bytes, int iters, double *tflops,
                                      void *cuda_stream)
{
    if (!d_scratch || !tflops || iters < 1) return CDMT_ERR_ARG;
    const int nblocks = 148 * 2, inner = 4096;
    if (scratch_bytes < sizeof(float) * (size_t)nblocks * 1024) return CDMT_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaEvent_t e0, e1;
    if (check_cuda(cudaEventCreate(&e0)) || check_cuda(cudaEventCreate(&e1))) return CDMT_ERR_CUDA;
    int rc = check_cuda(launch_fp32_peak(reinterpret_cast<float *>(d_scratch), nblocks, 64, st));  // warm-up
    double best = 0.0;
    for (int i = 0; i < iters && !rc; ++i) {
        cudaEventRecord(e0, st);
        rc = check_cuda(launch_fp32_peak(reinterpret_cast<float *>(d_scratch), nblocks, inner, st));
        cudaEventRecord(e1, st);
        if (rc) break;
        rc = check_cuda(cudaEventSynchronize(e1));
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = (double)nblocks * 1024.0 * inner * 16.0 * 8.0 * 2.0;
        const double tf = flops / (ms * 1e-3) * 1e-12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *tflops = best;
    return rc;
}
