// cdmt_incoherent.cu -- second stage of the semi-coherent search: every
// coherently dedispersed filterbank is incoherently dedispersed over a grid of fine DM offsets
// ("brute force dedispersion"), while it is still in HBM.
//
//   shift[k][j] = rint(ddm_k (f_j^-2 - f_0^-2) / 2.41e-4 / tsamp)      (Eq. 2 between channel centres,
//                 f_0 = highest channel; fp64 on the host)
//   ts[d][k][t] = sum_j fb[d][t + shift[k][j] - smin][j],  t < nt - (smax - smin)
//
// The filterbank is time-major, channel-fastest; dedispersion wants runs along time.
// A CTA (8 warps) owns 256 output samples of 64 trials: it walks the channels in chunks of CC,
// transposing each chunk's tile [CC][256 + range] into shared memory (coalesced loads along
// channels), and every warp adds the chunk into the 8 trials x 8 samples (t = lane + 32 i) it
// keeps in registers.  The host orders the trials by DM offset and cuts them into groups of 8, so
// inside a group the shift of a channel only grows, and by little: per channel a thread reads its 8
// samples at the first trial's shift (conflict-free LDS.32) and re-reads them only where a trial's
// shift differs from the previous one (2-bit increments per trial from a table).  64 FADD per 8-16
// floats read from shared memory: the kernel is bound by the FP32 pipe (4 adds per float read would
// be the break-even with shared-memory bandwidth).
#include <algorithm>
#include <cmath>
#include <cstdint>

#include "cdmt_internal.h"

namespace cdmt {

constexpr int IC_TILE = 256;     // output samples per CTA
constexpr int IC_GROUP = 8;      // trials per warp (measured on c3: 16 x 4 warps 85 ms, 8 x 8 warps 72 ms, 4 x 8 warps 74 ms)
constexpr int IC_WARPS = 8;      // warps (trial groups) per CTA
constexpr int IC_MAXSTEP = 3;    // largest growth of a channel's shift from one trial to the next (2-bit table field)

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
    // groups of up to IC_GROUP consecutive trials whose shifts grow by at most 3 samples per trial
    T->groups.clear();
    T->entries.clear();
    int k0 = 0;
    while (k0 < nfine) {
        int n = 1;
        while (n < IC_GROUP && k0 + n < nfine) {
            bool ok = true;
            const int *a = &T->shifts[(size_t)(k0 + n) * nch], *p = &T->shifts[(size_t)(k0 + n - 1) * nch];
            for (int j = 0; j < nch && ok; ++j)
                ok = a[j] >= p[j] && a[j] - p[j] <= IC_MAXSTEP;
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
    int nt_in, nt_out, nch, ngroups, cc, tw, vec_in;
};

// this lane's 8 samples t = lane + 32 i of one channel at the current shift
__device__ __forceinline__ void ic_window(float (&v)[8], const float *p)
{
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = p[32 * i];
}

// Trial K of the group: if its 2-bit field of `ey` is non-zero, advance the shared-memory address by
// that many samples and re-read the window.  Written in PTX so that the test is one predicate-setting
// logic instruction and the branch is declared warp-uniform (`bra.uni`: every lane holds the same
// table word) -- no reconvergence bookkeeping, nothing but two instructions on the common path.
template <int K>
__device__ __forceinline__ void ic_step(float (&v)[8], unsigned &sp, unsigned ey)
{
    asm volatile(
        "{\n\t"
        ".reg .pred q;\n\t"
        ".reg .b32 t;\n\t"
        "and.b32 t, %9, %10;\n\t"
        "setp.eq.u32 q, t, 0;\n\t"
        "@q bra.uni IC_SKIP;\n\t"
        "shr.u32 t, t, %11;\n\t"
        "shl.b32 t, t, 2;\n\t"
        "add.u32 %8, %8, t;\n\t"
        "ld.shared.f32 %0, [%8];\n\t"
        "ld.shared.f32 %1, [%8+128];\n\t"
        "ld.shared.f32 %2, [%8+256];\n\t"
        "ld.shared.f32 %3, [%8+384];\n\t"
        "ld.shared.f32 %4, [%8+512];\n\t"
        "ld.shared.f32 %5, [%8+640];\n\t"
        "ld.shared.f32 %6, [%8+768];\n\t"
        "ld.shared.f32 %7, [%8+896];\n\t"
        "IC_SKIP:\n\t"
        "}"
        : "+f"(v[0]), "+f"(v[1]), "+f"(v[2]), "+f"(v[3]), "+f"(v[4]), "+f"(v[5]), "+f"(v[6]), "+f"(v[7]), "+r"(sp)
        : "r"(ey), "n"(3u << (2 * K)), "n"(2 * K)
        : "memory");
}

template <int K>
__device__ __forceinline__ void ic_trials(float (&acc)[IC_GROUP][8], float (&v)[8], unsigned &sp, unsigned ey)
{
    if constexpr (K < IC_GROUP) {
        if constexpr (K > 0) ic_step<K>(v, sp, ey);
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[K][i] += v[i];
        ic_trials<K + 1>(acc, v, sp, ey);
    }
}

// grid (ceil(nt_out / 256), ceil(ngroups / IC_WARPS), ndm), 32 IC_WARPS threads; dynamic shared memory:
// float tile[cc][tw] and uint2 tab[IC_WARPS][cc]
__global__ void __launch_bounds__(32 * IC_WARPS, 2) k_incoherent(const IcArgs a)
{
    extern __shared__ float4 ic_smem4[];
    float *tile = reinterpret_cast<float *>(ic_smem4);
    const int cc = a.cc, tw = a.tw, quads = cc >> 2;
    uint2 *tab = reinterpret_cast<uint2 *>(tile + (((size_t)cc * tw + 3) & ~(size_t)3));
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int t0 = blockIdx.x * IC_TILE;
    const int grp = blockIdx.y * IC_WARPS + warp;
    const bool live = grp < a.ngroups;
    const float *fb = a.fb + (size_t)blockIdx.z * (size_t)a.fb_stride_dm;
    const int rows = tw;                     // input samples staged per chunk
    const int rstep = (32 * IC_WARPS) / quads;
    const int r0 = tid / quads, q = tid % quads;

    float acc[IC_GROUP][8];  // trial k of the group, output sample t0 + lane + 32 i
#pragma unroll
    for (int k = 0; k < IC_GROUP; ++k)
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[k][i] = 0.f;

    for (int c0 = 0; c0 < a.nch; c0 += cc) {
        __syncthreads();  // the previous chunk has been consumed
        // ---- stage the transposed tile: tile[c][i] = fb[t0 + i][c0 + c]; four rows per thread in
        //      flight (the loads of a batch are issued before its stores); tw = 1 mod 32 keeps the
        //      transposing stores of a warp (8 channel quads x 4 rows) on 32 different banks
        for (int ib = r0; ib < rows; ib += 4 * rstep) {
            float gq[4][4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int i = ib + u * rstep, t = t0 + i;
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
        for (int e = tid; e < IC_WARPS * cc; e += 32 * IC_WARPS) {
            const int w = e / cc, c = e % cc;
            const int gw = blockIdx.y * IC_WARPS + w;
            uint2 v = make_uint2(0u, 0u);
            if (gw < a.ngroups && c0 + c < a.nch) v = a.entries[(size_t)gw * a.nch + c0 + c];
            tab[w * cc + c] = v;
        }
        __syncthreads();
        if (!live) continue;
        // ---- accumulate the chunk.  Per channel: the window of the group's first trial (8 conflict-free
        //      LDS.32), then blocks of four trials -- usually no trial of a block moves the shift (one
        //      test, 32 straight adds); where one does, the window is re-read at the new shift
#pragma unroll 1
        for (int c = 0; c < cc; ++c) {
            const uint2 e = tab[warp * cc + c];
            const float *p = tile + (size_t)c * tw + e.x + lane;
            float v[8];
            ic_window(v, p);
            unsigned sp = (unsigned)__cvta_generic_to_shared(p);
            // the table word is the same in every lane; the shuffle lets the compiler know it
            ic_trials<0>(acc, v, sp, __shfl_sync(0xffffffffu, e.y, 0));
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
    a.tw = ((T.range + IC_TILE + 30) & ~31) + 1;  // >= range + 256 and = 1 mod 32
    a.vec_in = (nch % 4 == 0 && fb_stride_dm % 4 == 0 && (reinterpret_cast<uintptr_t>(d_fb) & 15) == 0) ? 1 : 0;
    // channels per chunk: the largest of 32, 16, 8, 4 whose tile lets two CTAs share an SM, else whatever fits
    auto smem_for = [&](int cc) { return sizeof(float) * (((size_t)cc * a.tw + 3) & ~(size_t)3) + sizeof(uint2) * IC_WARPS * cc; };
    int cc = 0;
    for (int c : {32, 16, 8, 4})
        if (smem_for(c) <= 72 * 1024) { cc = c; break; }
    if (!cc)
        for (int c : {32, 16, 8, 4})
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
