// cdmt_incoherent.cu -- second stage of the semi-coherent search: every
// coherently dedispersed filterbank is incoherently dedispersed over a grid of fine DM offsets
// ("brute force dedispersion"), while it is still in HBM.
//
//   shift[k][j] = rint(ddm_k (f_j^-2 - f_0^-2) / 2.41e-4 / tsamp)      (Eq. 2 between channel centres,
//                 f_0 = highest channel; fp64 on the host)
//   ts[d][k][t] = sum_j fb[d][t + shift[k][j] - smin][j],  t < nt - (smax - smin)
//
// The filterbank is time-major, channel-fastest; dedispersion wants runs along time.
// A CTA (4 warps) owns 256 output samples of 64 trials: it walks the channels in chunks of CC,
// transposing each chunk's tile [CC][256 + range + ...] into shared memory (coalesced loads along
// channels), and every warp adds the chunk into the 16 trials x 8 samples it keeps in registers.
// Per channel a thread loads two 8-sample windows (4 x LDS.128) that serve all 16 trials of its
// group: the host orders the trials by DM offset and cuts groups so that, inside a group, the shift
// of any channel grows by at most 4 samples, so the window only ever slides forward by register
// moves (2-bit increments per trial from a table).  Four copies of the tile, displaced by 0..3
// samples, make every window start 16-byte aligned.  128 FADD per 16 floats read from shared memory:
// the kernel is bound by the FP32 pipe, not by shared-memory bandwidth (4 adds per float would be
// the break-even).
#include <algorithm>
#include <cmath>
#include <cstdint>

#include "cdmt_internal.h"

namespace cdmt {

constexpr int IC_TILE = 256;     // output samples per CTA
constexpr int IC_GROUP = 16;     // trials per warp
constexpr int IC_WARPS = 4;      // warps (trial groups) per CTA
constexpr int IC_MAXSPREAD = 4;  // growth of a channel's shift inside a group the 8-sample window allows

// ------------------------------------------------------------------------------------------ host
bool incoherent_plan(const Geometry &g, const double *h_fcen, int nfine, const double *ddm, IncoherentTables *T)
{
    for (int k = 1; k < nfine; ++k)
        if (!(ddm[k] > ddm[k - 1])) return false;
    const int nch = g.nsub * g.nchan;
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
    // groups of up to 16 consecutive trials whose shifts stay inside the sliding window
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
                ok = a[j] >= p[j] && a[j] - p[j] <= 3 && a[j] - b[j] <= IC_MAXSPREAD;
            if (!ok) break;
            ++n;
        }
        T->groups.push_back(make_int2(k0, n));
        for (int j = 0; j < nch; ++j) {
            uint2 e;
            e.x = (unsigned)(T->shifts[(size_t)k0 * nch + j] - smin);
            e.y = 0;
            for (int k = 1; k < n; ++k) {
                const unsigned inc = (unsigned)(T->shifts[(size_t)(k0 + k) * nch + j] - T->shifts[(size_t)(k0 + k - 1) * nch + j]);
                e.y |= inc << (2 * k);
            }
            T->entries.push_back(e);
        }
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
    int nt_in, nt_out, nch, ngroups, cc, tw, vec_in, vec_out;
};

__device__ __forceinline__ void ic_slide(float (&v)[8])
{
#pragma unroll
    for (int i = 0; i < 7; ++i) v[i] = v[i + 1];
}

// grid (ceil(nt_out / 256), ceil(ngroups / 4), ndm), 128 threads; dynamic shared memory:
// float tile[cc][4 copies][tw] (+ skew) and uint2 tab[4][cc]
__global__ void __launch_bounds__(32 * IC_WARPS, 2) k_incoherent(const IcArgs a)
{
    extern __shared__ float4 ic_smem4[];
    float *tile = reinterpret_cast<float *>(ic_smem4);
    const int cc = a.cc, tw = a.tw, quads = cc >> 2;
    uint2 *tab = reinterpret_cast<uint2 *>(tile + (size_t)cc * 4 * tw + 32);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int t0 = blockIdx.x * IC_TILE;
    const int grp = blockIdx.y * IC_WARPS + warp;
    const bool live = grp < a.ngroups;
    const float *fb = a.fb + (size_t)blockIdx.z * (size_t)a.fb_stride_dm;
    const int rows = tw + 3;                 // input samples staged per chunk
    const int rstep = (32 * IC_WARPS) / quads;
    const int r0 = tid / quads, q = tid % quads;

    float acc[IC_GROUP][8];
#pragma unroll
    for (int k = 0; k < IC_GROUP; ++k)
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[k][i] = 0.f;

    for (int c0 = 0; c0 < a.nch; c0 += cc) {
        __syncthreads();  // the previous chunk has been consumed
        // ---- stage: tile copy j of channel c holds fb[t0 + i + j][c0 + c] at index i
        for (int i = r0; i < rows; i += rstep) {
            const int t = t0 + i;
            float gq[4] = {0.f, 0.f, 0.f, 0.f};
            if (t < a.nt_in) {
                const float *src = fb + (size_t)t * a.nch + c0 + 4 * q;
                if (a.vec_in && c0 + 4 * q + 3 < a.nch) {
                    const float4 w = __ldg(reinterpret_cast<const float4 *>(src));
                    gq[0] = w.x; gq[1] = w.y; gq[2] = w.z; gq[3] = w.w;
                } else {
#pragma unroll
                    for (int e = 0; e < 4; ++e)
                        if (c0 + 4 * q + e < a.nch) gq[e] = __ldg(src + e);
                }
            }
#pragma unroll
            for (int e = 0; e < 4; ++e)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int idx = i - j;
                    if (idx >= 0 && idx < tw) tile[(size_t)((4 * q + e) * 4 + j) * tw + 8 * q + idx] = gq[e];
                }
        }
        for (int e = tid; e < IC_WARPS * cc; e += 32 * IC_WARPS) {
            const int w = e / cc, c = e % cc;
            const int gw = blockIdx.y * IC_WARPS + w;
            uint2 v = make_uint2(0u, 0u);
            if (gw < a.ngroups && c0 + c < a.nch) v = a.entries[(size_t)gw * a.nch + c0 + c];
            tab[w * cc + c] = v;
        }
        __syncthreads();
        if (!live) continue;
        // ---- accumulate the chunk: two 8-sample windows per channel serve the 16 trials
#pragma unroll 1
        for (int c = 0; c < cc; ++c) {
            const uint2 e = tab[warp * cc + c];
            const float *p = tile + (size_t)(c * 4 + (int)(e.x & 3u)) * tw + 8 * (c >> 2) + (e.x & ~3u) + 4 * lane;
            float v0[8], v1[8];
            {
                const float4 x0 = *reinterpret_cast<const float4 *>(p), x1 = *reinterpret_cast<const float4 *>(p + 4);
                const float4 y0 = *reinterpret_cast<const float4 *>(p + 128), y1 = *reinterpret_cast<const float4 *>(p + 132);
                v0[0] = x0.x; v0[1] = x0.y; v0[2] = x0.z; v0[3] = x0.w; v0[4] = x1.x; v0[5] = x1.y; v0[6] = x1.z; v0[7] = x1.w;
                v1[0] = y0.x; v1[1] = y0.y; v1[2] = y0.z; v1[3] = y0.w; v1[4] = y1.x; v1[5] = y1.y; v1[6] = y1.z; v1[7] = y1.w;
            }
            if (e.y == 0u) {
                // every trial of the group has the same shift in this channel (the usual case)
#pragma unroll
                for (int k = 0; k < IC_GROUP; ++k)
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        acc[k][i] += v0[i];
                        acc[k][4 + i] += v1[i];
                    }
            } else {
#pragma unroll
                for (int k = 0; k < IC_GROUP; ++k) {
                    if (k > 0) {
                        const unsigned n = (e.y >> (2 * k)) & 3u;
                        if (n >= 1u) { ic_slide(v0); ic_slide(v1); }
                        if (n >= 2u) { ic_slide(v0); ic_slide(v1); }
                        if (n == 3u) { ic_slide(v0); ic_slide(v1); }
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        acc[k][i] += v0[i];
                        acc[k][4 + i] += v1[i];
                    }
                }
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
        for (int h = 0; h < 2; ++h) {
            const int t = t0 + 128 * h + 4 * lane;
            if (a.vec_out && t + 3 < a.nt_out) {
                *reinterpret_cast<float4 *>(row + t) = make_float4(acc[k][4 * h], acc[k][4 * h + 1], acc[k][4 * h + 2], acc[k][4 * h + 3]);
            } else {
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    if (t + i < a.nt_out) row[t + i] = acc[k][4 * h + i];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------- launch
cudaError_t launch_incoherent(const Geometry &g, const IncoherentTables &T, const float *d_fb, long long fb_stride_dm,
                              long long nt_in, float *d_ts, long long ts_stride_dm, long long ts_pitch,
                              void *d_workspace, cudaStream_t st, long long *launches)
{
    const int nch = T.nch, ngroups = (int)T.groups.size();
    const long long nt_out = nt_in - T.range;
    char *ws = reinterpret_cast<char *>(d_workspace);
    uint2 *d_entries = reinterpret_cast<uint2 *>(ws);
    int2 *d_groups = reinterpret_cast<int2 *>(ws + ic_align(T.entries.size() * sizeof(uint2)));
    cudaError_t e = cudaMemcpyAsync(d_entries, T.entries.data(), T.entries.size() * sizeof(uint2), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(d_groups, T.groups.data(), T.groups.size() * sizeof(int2), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;

    IcArgs a;
    a.fb = d_fb; a.fb_stride_dm = fb_stride_dm; a.ts = d_ts; a.ts_stride_dm = ts_stride_dm; a.ts_pitch = ts_pitch;
    a.entries = d_entries; a.groups = d_groups;
    a.nt_in = (int)nt_in; a.nt_out = (int)nt_out; a.nch = nch; a.ngroups = ngroups;
    a.tw = ((T.range + 3) & ~3) + IC_TILE + 8;
    a.vec_in = (nch % 4 == 0 && fb_stride_dm % 4 == 0 && (reinterpret_cast<uintptr_t>(d_fb) & 15) == 0) ? 1 : 0;
    a.vec_out = (ts_pitch % 4 == 0 && ts_stride_dm % 4 == 0 && (reinterpret_cast<uintptr_t>(d_ts) & 15) == 0) ? 1 : 0;
    // channels per chunk: the largest of 16, 8, 4 whose tile lets two CTAs share an SM, else whatever fits
    auto smem_for = [&](int cc) { return sizeof(float) * ((size_t)cc * 4 * a.tw + 32) + sizeof(uint2) * IC_WARPS * cc; };
    int cc = 0;
    for (int c : {16, 8, 4})
        if (smem_for(c) <= 110 * 1024) { cc = c; break; }
    if (!cc)
        for (int c : {16, 8, 4})
            if (smem_for(c) <= 227 * 1024) { cc = c; break; }
    if (!cc) return cudaErrorInvalidValue;
    a.cc = cc;
    const size_t smem = smem_for(cc);
    e = cudaFuncSetAttribute(k_incoherent, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)((nt_out + IC_TILE - 1) / IC_TILE), (unsigned)((ngroups + IC_WARPS - 1) / IC_WARPS), (unsigned)g.ndm);
    k_incoherent<<<grid, 32 * IC_WARPS, smem, st>>>(a);
    e = cudaGetLastError();
    if (e == cudaSuccess) ++*launches;
    return e;
}

}  // namespace cdmt
