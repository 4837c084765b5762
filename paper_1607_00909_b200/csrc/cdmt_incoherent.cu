// cdmt_incoherent.cu -- second stage of the semi-coherent search: every
// coherently dedispersed filterbank is incoherently dedispersed over a grid of fine DM offsets
// ("brute force dedispersion"), while it is still in HBM.
//
//   shift[k][j] = rint(ddm_k (f_j^-2 - f_0^-2) / 2.41e-4 / tsamp)      (Eq. 2 between channel centres,
//                 f_0 = highest channel; fp64 on the host)
//   ts[d][k][t] = sum_j fb[d][t + shift[k][j] - smin][j],  t < nt - (smax - smin)
//
// The filterbank is time-major, channel-fastest; dedispersion wants runs along time.
// The sums are those of the brute-force definition above, but they are not formed trial by trial.
// The host orders the trials by DM offset and cuts them into groups of up to 8 in which the shift of
// any channel grows by at most 4 samples.  Inside a group a channel's shifts are fixed by its first
// shift s0 and seven 2-bit increments, and neighbouring channels share the increment pattern over
// runs of typically 10-100 channels.  For a run R the kernel forms
//     P_o[t] = sum_{j in R} fb[t + s0_j + o - smin][j],   o = 0 .. spread(R) <= 4
// -- one add per channel, sample and DISTINCT shift instead of one per trial -- and at the end of the
// run adds P_{o_R(k)} into trial k (o_R(k) = the pattern's cumulative increment).  Same terms, other
// order of additions; exact on integer data.
//
// A CTA (16 warps = 16 trial groups = 128 trials) owns 256 output samples: it walks the channels in
// chunks of 32, transposing each chunk's tile [32][256 + range] into shared memory (coalesced float4
// loads along channels, row length = 1 mod 32 so that the transposing stores are conflict-free); a
// thread keeps 8 trials x 8 samples (t = lane + 32 i) plus the five run sums in registers and reads 8
// samples per channel and distinct shift with conflict-free LDS.32.  The table words of a (group,
// channel) are made warp-uniform for the compiler by a shuffle, so every test on them is a uniform
// branch.  Measured on c3 (251 fine trials x 96 coherent DMs): 54 ms against 66 ms for the
// trial-by-trial kernel it replaces (16 x 8 trials: 54 ms, 8 x 8: 58 ms, 4 x 8: 69 ms).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>

#include "cdmt_internal.h"

namespace cdmt {

constexpr int IC_TILE = 256;     // output samples per CTA
constexpr int IC_GROUP = 8;      // trials per warp
constexpr int IC_WARPS = 16;     // warps (trial groups) per CTA
constexpr int IC_MAXSTEP = 3;    // largest growth of a channel's shift from one trial to the next (2-bit table field)
constexpr int IC_MAXSPREAD = 4;  // largest growth of a channel's shift inside a group (five run sums P_0..P_4)

// ------------------------------------------------------------------------------------------ host
bool incoherent_plan(const Geometry &g, const double *h_fcen, int nfine, const double *ddm, IncoherentTables *T)
{
    for (int k = 1; k < nfine; ++k)
        if (!(ddm[k] > ddm[k - 1])) return false;
    const int nch = g.nsub * g.nchan;
    incoherent_release(T);   // page-locked copy of the previous tables
    T->nfine = nfine;
    T->nch = nch;
    // channel centres in the order of the filterbank: descending frequency
    std::vector<double> f((size_t)nch);
    for (int s = 0; s < g.nsub; ++s)
        for (int c = 0; c < g.nchan; ++c)
            f[(size_t)nch - 1 - ((size_t)s * g.nchan + c)] =
                h_fcen[s] + ((double)c + 0.5 - 0.5 * (double)g.nchan) * g.bw_mhz / (double)g.nchan;
    const double tsamp = (double)g.nchan * (double)g.ndec / (g.bw_mhz * 1e6);
    T->shifts.assign((size_t)nfine * nch, 0);
    int smin = 0, smax = 0;
    for (int k = 0; k < nfine; ++k)
        for (int j = 0; j < nch; ++j) {
            const double tau = ddm[k] * (1.0 / (f[j] * f[j]) - 1.0 / (f[0] * f[0])) / 2.41e-4;
            const int s = (int)std::nearbyint(tau / tsamp);
            T->shifts[(size_t)k * nch + j] = s;
            smin = std::min(smin, s);
            smax = std::max(smax, s);
        }
    T->smin = smin;
    T->range = smax - smin;
    // groups of up to 8 consecutive trials whose shifts grow by at most 3 samples per trial and 4 in all
    T->groups.clear();
    T->entries.clear();
    int k0 = 0;
    while (k0 < nfine) {
        int n = 1;
        while (n < IC_GROUP && k0 + n < nfine) {
            bool ok = true;
            const int *a = &T->shifts[(size_t)(k0 + n) * nch], *p = &T->shifts[(size_t)(k0 + n - 1) * nch];
            const int *b = &T->shifts[(size_t)k0 * nch];
            for (int j = 0; j < nch && ok; ++j)
                ok = a[j] >= p[j] && a[j] - p[j] <= IC_MAXSTEP && a[j] - b[j] <= IC_MAXSPREAD;
            if (!ok) break;
            ++n;
        }
        T->groups.push_back(make_int2(k0, n));
        // entry of channel j: x = (s0 - smin) | spread << 24 | end-of-run << 28, y = 2-bit increments
        const size_t e0 = T->entries.size();
        for (int j = 0; j < nch; ++j) {
            uint2 e;
            e.x = (unsigned)(T->shifts[(size_t)k0 * nch + j] - smin);
            e.y = 0;
            for (int k = 1; k < n; ++k) {
                const unsigned inc = (unsigned)(T->shifts[(size_t)(k0 + k) * nch + j] - T->shifts[(size_t)(k0 + k - 1) * nch + j]);
                e.y |= inc << (2 * k);
            }
            const unsigned spread = (unsigned)(T->shifts[(size_t)(k0 + n - 1) * nch + j] - T->shifts[(size_t)k0 * nch + j]);
            e.x |= spread << 24;
            T->entries.push_back(e);
        }
        // a run ends where the next channel has another increment pattern, and at the last channel
        for (int j = 0; j < nch; ++j)
            if (j == nch - 1 || T->entries[e0 + j].y != T->entries[e0 + j + 1].y) T->entries[e0 + j].x |= 1u << 28;
        k0 += n;
    }
    return true;
}

static size_t ic_align(size_t x) { return (x + 255) & ~(size_t)255; }

size_t incoherent_workspace_bytes(const IncoherentTables &T)
{
    return ic_align(T.entries.size() * sizeof(uint2)) + ic_align(T.groups.size() * sizeof(int2));
}

// ---------------------------------------------------------------------------------------- device
struct IcArgs {
    const float *fb;        // [ndm] planes of [nt_in][nch]
    long long fb_stride_dm;
    float *ts;              // [ndm] planes of [nfine] rows of ts_pitch
    long long ts_stride_dm, ts_pitch;
    const uint2 *entries;   // [ngroups][nch]
    const int2 *groups;     // [ngroups]
    int nt_in, nt_out, nch, ngroups, cc, tw, vec_in;
    int gpc, tt;            // trial groups and 256-sample time tiles per CTA: gpc * tt <= IC_WARPS warps are live
};

// Run sums of the distinct shifts O1 and O2 = O1 + 1 of one channel: if spread >= O1 add this lane's
// 8 samples at s0 + O1 into PA, and if spread >= O2 those at s0 + O2 into PB.  PTX so that the tests
// stay two-instruction branches (`bra.uni`: every lane holds the same table word) instead of sixteen
// predicated loads and adds on the common path, where spread is 0 and only the first test executes.
template <int O1>
__device__ __forceinline__ void ic_run_add2(float (&PA)[8], float (&PB)[8], unsigned sp, unsigned spread)
{
    asm volatile(
        "{\n\t"
        ".reg .pred q;\n\t"
        ".reg .f32 t<8>;\n\t"
        ".reg .b32 a;\n\t"
        "setp.lt.u32 q, %17, %18;\n\t"
        "@q bra.uni IC_END;\n\t"
        "add.u32 a, %16, %20;\n\t"
        "ld.shared.f32 t0, [a];\n\t"
        "ld.shared.f32 t1, [a+128];\n\t"
        "ld.shared.f32 t2, [a+256];\n\t"
        "ld.shared.f32 t3, [a+384];\n\t"
        "ld.shared.f32 t4, [a+512];\n\t"
        "ld.shared.f32 t5, [a+640];\n\t"
        "ld.shared.f32 t6, [a+768];\n\t"
        "ld.shared.f32 t7, [a+896];\n\t"
        "add.f32 %0, %0, t0;\n\t"
        "add.f32 %1, %1, t1;\n\t"
        "add.f32 %2, %2, t2;\n\t"
        "add.f32 %3, %3, t3;\n\t"
        "add.f32 %4, %4, t4;\n\t"
        "add.f32 %5, %5, t5;\n\t"
        "add.f32 %6, %6, t6;\n\t"
        "add.f32 %7, %7, t7;\n\t"
        "setp.lt.u32 q, %17, %19;\n\t"
        "@q bra.uni IC_END;\n\t"
        "add.u32 a, %16, %21;\n\t"
        "ld.shared.f32 t0, [a];\n\t"
        "ld.shared.f32 t1, [a+128];\n\t"
        "ld.shared.f32 t2, [a+256];\n\t"
        "ld.shared.f32 t3, [a+384];\n\t"
        "ld.shared.f32 t4, [a+512];\n\t"
        "ld.shared.f32 t5, [a+640];\n\t"
        "ld.shared.f32 t6, [a+768];\n\t"
        "ld.shared.f32 t7, [a+896];\n\t"
        "add.f32 %8, %8, t0;\n\t"
        "add.f32 %9, %9, t1;\n\t"
        "add.f32 %10, %10, t2;\n\t"
        "add.f32 %11, %11, t3;\n\t"
        "add.f32 %12, %12, t4;\n\t"
        "add.f32 %13, %13, t5;\n\t"
        "add.f32 %14, %14, t6;\n\t"
        "add.f32 %15, %15, t7;\n\t"
        "IC_END:\n\t"
        "}"
        : "+f"(PA[0]), "+f"(PA[1]), "+f"(PA[2]), "+f"(PA[3]), "+f"(PA[4]), "+f"(PA[5]), "+f"(PA[6]), "+f"(PA[7]),
          "+f"(PB[0]), "+f"(PB[1]), "+f"(PB[2]), "+f"(PB[3]), "+f"(PB[4]), "+f"(PB[5]), "+f"(PB[6]), "+f"(PB[7])
        : "r"(sp), "r"(spread), "n"(O1), "n"(O1 + 1), "n"(4 * O1), "n"(4 * (O1 + 1))
        : "memory");
}

// grid (ceil(nt_out / (256 tt)), ceil(ngroups / gpc), ndm), 32 IC_WARPS threads; warp w works on trial group
// w % gpc and time tile w / gpc of the CTA (few trial groups: several time tiles share one staged tile,
// so that the warps stay busy and the halo is re-read less).  Dynamic shared memory: float tile[cc][tw]
// and uint2 tab[gpc][cc]
template <bool MULTI>   // false: gpc = IC_WARPS, tt = 1 as compile-time constants (the common, register-tight case)
__global__ void __launch_bounds__(32 * IC_WARPS, 1) k_incoherent(const IcArgs a)
{
    const int gpc = MULTI ? a.gpc : IC_WARPS, tt = MULTI ? a.tt : 1;
    extern __shared__ float4 ic_smem4[];
    float *tile = reinterpret_cast<float *>(ic_smem4);
    const int cc = a.cc, tw = a.tw, quads = cc >> 2;
    uint2 *tab = reinterpret_cast<uint2 *>(tile + (((size_t)cc * tw + 3) & ~(size_t)3));
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tbase = blockIdx.x * IC_TILE * tt;           // first sample of the staged tile
    const int gsel = MULTI ? warp % gpc : warp, sub = MULTI ? warp / gpc : 0;
    const int t0 = tbase + sub * IC_TILE;                  // first output sample of this warp
    const int grp = blockIdx.y * gpc + gsel;
    const bool live = sub < tt && grp < a.ngroups && t0 < a.nt_out;
    const float *fb = a.fb + (size_t)blockIdx.z * (size_t)a.fb_stride_dm;
    const int rows = tw;                     // input samples staged per chunk
    const int rstep = (32 * IC_WARPS) / quads;
    const int r0 = tid / quads, q = tid % quads;

    float acc[IC_GROUP][8];        // trial k of the group, output sample t0 + lane + 32 i
    float P[IC_MAXSPREAD + 1][8];  // sums of the current run of channels at shifts s0 + o
#pragma unroll
    for (int k = 0; k < IC_GROUP; ++k)
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[k][i] = 0.f;
#pragma unroll
    for (int o = 0; o <= IC_MAXSPREAD; ++o)
#pragma unroll
        for (int i = 0; i < 8; ++i) P[o][i] = 0.f;

    for (int c0 = 0; c0 < a.nch; c0 += cc) {
        __syncthreads();  // the previous chunk has been consumed
        // ---- stage the transposed tile: tile[c][i] = fb[t0 + i][c0 + c]; four rows per thread in
        //      flight (the loads of a batch are issued before its stores); tw = 1 mod 32 keeps the
        //      transposing stores of a warp (8 channel quads x 4 rows) on 32 different banks
        for (int ib = r0; ib < rows; ib += 4 * rstep) {
            float gq[4][4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int i = ib + u * rstep, t = tbase + i;
#pragma unroll
                for (int e = 0; e < 4; ++e) gq[u][e] = 0.f;
                if (i < rows && t < a.nt_in) {
                    const float *src = fb + (size_t)t * a.nch + c0 + 4 * q;
                    if (a.vec_in && c0 + 4 * q + 3 < a.nch) {
                        const float4 w = __ldg(reinterpret_cast<const float4 *>(src));
                        gq[u][0] = w.x; gq[u][1] = w.y; gq[u][2] = w.z; gq[u][3] = w.w;
                    } else {
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            if (c0 + 4 * q + e < a.nch) gq[u][e] = __ldg(src + e);
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int i = ib + u * rstep;
                if (i < rows) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) tile[(size_t)(4 * q + e) * tw + i] = gq[u][e];
                }
            }
        }
        for (int e = tid; e < gpc * cc; e += 32 * IC_WARPS) {
            const int w = e / cc, c = e % cc;
            const int gw = blockIdx.y * gpc + w;
            uint2 v = make_uint2(0u, 0u);
            if (gw < a.ngroups && c0 + c < a.nch) v = a.entries[(size_t)gw * a.nch + c0 + c];
            tab[w * cc + c] = v;
        }
        __syncthreads();
        if (!live) continue;
        // ---- add the chunk's channels into the run sums; at the end of a run, into the trials
#pragma unroll 1
        for (int c = 0; c < cc; ++c) {
            const uint2 e0 = tab[gsel * cc + c];
            // the table words are the same in every lane; the shuffles let the compiler know it
            uint2 e;
            e.x = __shfl_sync(0xffffffffu, e0.x, 0);
            e.y = __shfl_sync(0xffffffffu, e0.y, 0);
            const unsigned s0 = e.x & 0xffffffu, spread = (e.x >> 24) & 7u;
            const float *p = tile + (size_t)c * tw + s0 + lane + sub * IC_TILE;
#pragma unroll
            for (int i = 0; i < 8; ++i) P[0][i] += p[32 * i];
            const unsigned sp = (unsigned)__cvta_generic_to_shared(p);
            ic_run_add2<1>(P[1], P[2], sp, spread);
            ic_run_add2<3>(P[3], P[4], sp, spread);
            if (e.x & (1u << 28)) {
                // end of the run: trial k takes the sum at its cumulative increment o_k
                unsigned o = 0;
#pragma unroll
                for (int k = 0; k < IC_GROUP; ++k) {
                    if (k > 0) o += (e.y >> (2 * k)) & 3u;
                    if (o == 0u) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) acc[k][i] += P[0][i];
                    } else if (o == 1u) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) acc[k][i] += P[1][i];
                    } else if (o == 2u) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) acc[k][i] += P[2][i];
                    } else if (o == 3u) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) acc[k][i] += P[3][i];
                    } else {
#pragma unroll
                        for (int i = 0; i < 8; ++i) acc[k][i] += P[4][i];
                    }
                }
#pragma unroll
                for (int oo = 0; oo <= IC_MAXSPREAD; ++oo)
#pragma unroll
                    for (int i = 0; i < 8; ++i) P[oo][i] = 0.f;
            }
        }
    }
    if (!live) return;
    const int2 gi = a.groups[grp];
    float *out = a.ts + (size_t)blockIdx.z * (size_t)a.ts_stride_dm;
#pragma unroll
    for (int k = 0; k < IC_GROUP; ++k) {
        if (k >= gi.y) break;
        float *row = out + (size_t)(gi.x + k) * (size_t)a.ts_pitch;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int t = t0 + lane + 32 * i;
            if (t < a.nt_out) row[t] = acc[k][i];
        }
    }
}

// the last `nrows` rows of every DM plane move to its front (cdmt_incoherent_carry)
__global__ void __launch_bounds__(256) k_carry_rows(float *fb, long long fb_stride_dm, long long src_off, long long n)
{
    float *p = fb + (size_t)blockIdx.y * (size_t)fb_stride_dm;
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256) p[i] = p[src_off + i];
}

cudaError_t launch_carry_rows(float *d_fb, long long fb_stride_dm, long long nt_in, int nrows, int nch, int ndm,
                              cudaStream_t st, long long *launches)
{
    const long long n = (long long)nrows * nch;
    if (n == 0) return cudaSuccess;
    dim3 grid((unsigned)((n + 256 * 8 - 1) / (256 * 8) > 4096 ? 4096 : (n + 256 * 8 - 1) / (256 * 8)), (unsigned)ndm);
    k_carry_rows<<<grid, 256, 0, st>>>(d_fb, fb_stride_dm, (nt_in - nrows) * (long long)nch, n);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) ++*launches;
    return e;
}

// ---------------------------------------------------------------------------------------- launch
// Launch geometry: trial groups and time tiles per CTA, the row length of the staged tile and the channels
// per chunk that fit shared memory; false if even four channels of 256 + range samples do not fit
// (range > ~14000) or there are more trial groups than a grid dimension holds.
bool incoherent_config(const IncoherentTables &T, int *cc_out, int *tw_out, int *gpc_out, int *tt_out, size_t *smem_out)
{
    const int ngroups = (int)T.groups.size();
    if (ngroups < 1) return false;
    // trial groups per CTA (balanced over grid.y) and, where they do not fill the warps, time tiles per CTA
    const int ny = (ngroups + IC_WARPS - 1) / IC_WARPS;
    if (ny > 65535) return false;
    const int gpc = (ngroups + ny - 1) / ny;
    int tt = IC_WARPS / gpc;
    for (;; --tt) {
        const int tw = ((T.range + tt * IC_TILE + 30) & ~31) + 1;   // >= range + 256 tt and = 1 mod 32
        auto smem_for = [&](int cc) { return sizeof(float) * (((size_t)cc * tw + 3) & ~(size_t)3) + sizeof(uint2) * gpc * cc; };
        // channels per chunk: 32 if the tile stays below 72 KB, else fewer time tiles; at one time tile
        // whatever number of channels fits shared memory
        int cc = 0;
        if (smem_for(32) <= 72 * 1024) cc = 32;
        else if (tt == 1)
            for (int c : {32, 16, 8, 4})
                if (smem_for(c) <= 227 * 1024) { cc = c; break; }
        if (cc) {
            if (cc_out) *cc_out = cc;
            if (tw_out) *tw_out = tw;
            if (gpc_out) *gpc_out = gpc;
            if (tt_out) *tt_out = tt;
            if (smem_out) *smem_out = smem_for(cc);
            return true;
        }
        if (tt == 1) return false;   // even four channels of 256 + range samples do not fit
    }
}

void incoherent_release(IncoherentTables *T)
{
    if (T->pinned) cudaFreeHost(T->pinned);
    T->pinned = nullptr;
}

cudaError_t launch_incoherent(const Geometry &g, IncoherentTables &T, const float *d_fb, long long fb_stride_dm,
                              long long nt_in, float *d_ts, long long ts_stride_dm, long long ts_pitch,
                              void *d_workspace, cudaStream_t st, long long *launches)
{
    const int nch = T.nch, ngroups = (int)T.groups.size();
    const long long nt_out = nt_in - T.range;
    char *ws = reinterpret_cast<char *>(d_workspace);
    const size_t nb_e = T.entries.size() * sizeof(uint2), nb_g = T.groups.size() * sizeof(int2);
    uint2 *d_entries = reinterpret_cast<uint2 *>(ws);
    int2 *d_groups = reinterpret_cast<int2 *>(ws + ic_align(nb_e));
    // the tables travel from page-locked memory the plan keeps for them: a plain asynchronous copy on the
    // caller's stream, also inside a stream capture
    if (!T.pinned) {
        cudaError_t e = cudaMallocHost(&T.pinned, ic_align(nb_e) + nb_g);
        if (e != cudaSuccess) return e;
        memcpy(T.pinned, T.entries.data(), nb_e);
        memcpy(static_cast<char *>(T.pinned) + ic_align(nb_e), T.groups.data(), nb_g);
    }
    cudaError_t e = cudaMemcpyAsync(d_entries, T.pinned, nb_e, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(d_groups, static_cast<char *>(T.pinned) + ic_align(nb_e), nb_g, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;

    IcArgs a;
    a.fb = d_fb; a.fb_stride_dm = fb_stride_dm; a.ts = d_ts; a.ts_stride_dm = ts_stride_dm; a.ts_pitch = ts_pitch;
    a.entries = d_entries; a.groups = d_groups;
    a.nt_in = (int)nt_in; a.nt_out = (int)nt_out; a.nch = nch; a.ngroups = ngroups;
    size_t smem = 0;
    if (!incoherent_config(T, &a.cc, &a.tw, &a.gpc, &a.tt, &smem)) return cudaErrorInvalidValue;
    a.vec_in = (nch % 4 == 0 && fb_stride_dm % 4 == 0 && (reinterpret_cast<uintptr_t>(d_fb) & 15) == 0) ? 1 : 0;
    const bool multi = !(a.gpc == IC_WARPS && a.tt == 1);
    e = multi ? cudaFuncSetAttribute(k_incoherent<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
              : cudaFuncSetAttribute(k_incoherent<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)((nt_out + IC_TILE * a.tt - 1) / (IC_TILE * a.tt)), (unsigned)((ngroups + a.gpc - 1) / a.gpc), (unsigned)g.ndm);
    if (multi) k_incoherent<true><<<grid, 32 * IC_WARPS, smem, st>>>(a);
    else k_incoherent<false><<<grid, 32 * IC_WARPS, smem, st>>>(a);
    e = cudaGetLastError();
    if (e == cudaSuccess) ++*launches;
    return e;
}

}  // namespace cdmt
