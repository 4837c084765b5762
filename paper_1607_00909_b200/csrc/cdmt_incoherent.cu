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
// samples per channel and distinct shift with conflict-free LDS.32.
//
// The first trial's shift s0 of a channel changes every ~90 channels at most (c3: 15 us of delay between
// neighbouring channels against 1.3 ms samples), so the host cuts every run further into SEGMENTS of
// channels that also share s0.  A warp walks the segment list of its trial group: inside a segment the
// window address only moves by one tile row per channel, so the channel loop holds nothing but the
// loads and adds (no table word, no shuffle, no test per channel), specialised by the run's spread; the
// segment records (one uint4 per ~30 channels) are read from global memory and made warp-uniform by a
// shuffle.  k_incoherent below is the general form (any channel count and alignment, shift ranges up to
// ~14 000 samples); k_incoherent_v4 further down is the fast form for filterbanks whose rows can be read
// in 16-byte pieces.  Measured on c3 (251 fine trials x 96 coherent DMs): 39.0 ms (k_incoherent_v4) against
// 54 ms for the per-channel table walk of round 1 and 66 ms for the trial-by-trial kernel before that.
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
    T->segs.clear();
    T->seg_off.clear();
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
    // Heaviest groups first: the 16 groups of a CTA meet at a block barrier once per chunk, so a CTA runs
    // at the pace of its slowest warp.  The work of a group -- (1 + spread) window reads per channel plus
    // the hand-over at every run end -- grows with |ddm| (offsets near zero move no channel by a sample),
    // so groups sorted by work share a CTA with their like.  (Each group carries its own first trial, so
    // the order of the records is free.)
    const int ngroups = (int)T->groups.size();
    std::vector<double> work((size_t)ngroups, 0.0);
    for (int gi = 0; gi < ngroups; ++gi)
        for (int j = 0; j < nch; ++j) {
            const uint2 e = T->entries[(size_t)gi * nch + j];
            work[gi] += 1.0 + (double)((e.x >> 24) & 7u) + ((e.x & (1u << 28)) ? 8.0 : 0.0);
        }
    std::vector<int> order((size_t)ngroups);
    for (int gi = 0; gi < ngroups; ++gi) order[gi] = gi;
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return work[x] > work[y]; });
    std::vector<int2> sorted_groups;
    sorted_groups.reserve(ngroups);
    for (int gi : order) {
        sorted_groups.push_back(T->groups[gi]);
        const size_t e0 = (size_t)gi * nch;
        // segments: maximal channel ranges [c0, c1) with the same first shift and increment pattern;
        // z = (s0 - smin) | spread << 24 | (the segment closes its run) << 28, w = the pattern
        T->seg_off.push_back((int)T->segs.size());
        for (int j = 0; j < nch;) {
            const uint2 e = T->entries[e0 + j];
            int j1 = j;
            while (!(T->entries[e0 + j1].x & (1u << 28)) && (T->entries[e0 + j1 + 1].x & 0xffffffu) == (e.x & 0xffffffu)) ++j1;
            uint4 sg;
            sg.x = (unsigned)j;
            sg.y = (unsigned)(j1 + 1);
            sg.z = (e.x & 0x07ffffffu) | (T->entries[e0 + j1].x & (1u << 28));
            sg.w = e.y;
            T->segs.push_back(sg);
            j = j1 + 1;
        }
    }
    T->groups.swap(sorted_groups);
    T->seg_off.push_back((int)T->segs.size());
    return true;
}

static size_t ic_align(size_t x) { return (x + 255) & ~(size_t)255; }

size_t incoherent_workspace_bytes(const IncoherentTables &T)
{
    return ic_align(T.segs.size() * sizeof(uint4)) + ic_align(T.seg_off.size() * sizeof(int)) + ic_align(T.groups.size() * sizeof(int2));
}

// ---------------------------------------------------------------------------------------- device
struct IcArgs {
    const float *fb;        // [ndm] planes of [nt_in][nch]
    long long fb_stride_dm;
    float *ts;              // [ndm] planes of [nfine] rows of ts_pitch
    long long ts_stride_dm, ts_pitch;
    const uint4 *segs;      // segment records, group after group
    const int *seg_off;     // [ngroups + 1] first segment of a group
    const int2 *groups;     // [ngroups]
    int nt_in, nt_out, nch, ngroups, cc, tw, vec_in;
    int gpc, tt;            // trial groups and 256-sample time tiles per CTA: gpc * tt <= IC_WARPS warps are live
};

// Run sums over the n channels of a segment: P_o[i] += tile[c][s0 + o + lane + 32 i], o <= SP (the run's spread)
template <int SP>
__device__ __forceinline__ void ic_seg_add(float (&P)[IC_MAXSPREAD + 1][8], const float *p, int n, int tw)
{
#pragma unroll 1
    for (int c = 0; c < n; ++c) {
#pragma unroll
        for (int o = 0; o <= SP; ++o)
#pragma unroll
            for (int i = 0; i < 8; ++i) P[o][i] += p[32 * i + o];
        p += tw;
    }
}

__device__ __forceinline__ uint4 ic_uniform(uint4 v)
{
    // the record is the same in every lane; the shuffles let the compiler know it (uniform branches)
    v.x = __shfl_sync(0xffffffffu, v.x, 0);
    v.y = __shfl_sync(0xffffffffu, v.y, 0);
    v.z = __shfl_sync(0xffffffffu, v.z, 0);
    v.w = __shfl_sync(0xffffffffu, v.w, 0);
    return v;
}

// grid (ceil(nt_out / (256 tt)), ceil(ngroups / gpc), ndm), 32 IC_WARPS threads; warp w works on trial group
// w % gpc and time tile w / gpc of the CTA (few trial groups: several time tiles share one staged tile,
// so that the warps stay busy and the halo is re-read less).  Dynamic shared memory: float tile[cc][tw]
template <bool MULTI>   // false: gpc = IC_WARPS, tt = 1 as compile-time constants (the common, register-tight case)
__global__ void __launch_bounds__(32 * IC_WARPS, 1) k_incoherent(const IcArgs a)
{
    const int gpc = MULTI ? a.gpc : IC_WARPS, tt = MULTI ? a.tt : 1;
    extern __shared__ float4 ic_smem4[];
    float *tile = reinterpret_cast<float *>(ic_smem4);
    const int cc = a.cc, tw = a.tw, quads = cc >> 2;
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

    int cur = 0, cur_end = 0;
    if (live) {
        cur = a.seg_off[grp];
        cur_end = a.seg_off[grp + 1];
    }
    uint4 sg = cur < cur_end ? ic_uniform(__ldg(a.segs + cur)) : make_uint4(0x7fffffffu, 0x7fffffffu, 0u, 0u);

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
        __syncthreads();
        if (!live) continue;
        // ---- the segments of this warp's trial group that reach into the chunk
        while ((int)sg.x < c0 + cc) {
            const int a0 = max((int)sg.x, c0), a1 = min((int)sg.y, c0 + cc);
            const unsigned s0 = sg.z & 0xffffffu, spread = (sg.z >> 24) & 7u;
            const float *p = tile + (size_t)(a0 - c0) * tw + s0 + lane + sub * IC_TILE;
            switch (spread) {
            case 0: ic_seg_add<0>(P, p, a1 - a0, tw); break;
            case 1: ic_seg_add<1>(P, p, a1 - a0, tw); break;
            case 2: ic_seg_add<2>(P, p, a1 - a0, tw); break;
            case 3: ic_seg_add<3>(P, p, a1 - a0, tw); break;
            default: ic_seg_add<4>(P, p, a1 - a0, tw); break;
            }
            if ((int)sg.y > c0 + cc) break;   // goes on in the next chunk
            if (sg.z & (1u << 28)) {
                // end of the run: trial k takes the sum at its cumulative increment o_k
                unsigned o = 0;
#pragma unroll
                for (int k = 0; k < IC_GROUP; ++k) {
                    if (k > 0) o += (sg.w >> (2 * k)) & 3u;
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
            ++cur;
            sg = cur < cur_end ? ic_uniform(__ldg(a.segs + cur)) : make_uint4(0x7fffffffu, 0x7fffffffu, 0u, 0u);
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

// ------------------------------------------------------------------------------------------------
// k_incoherent_v4: the same sums for filterbanks whose rows can be read in 16-byte pieces (channel count
// a multiple of 4, aligned planes) and whose shift range lets two tiles fit shared memory.
//
//  * The tile keeps the filterbank's own order, [time][CC channels] (CC = 32 or 64: 128- or 256-byte rows), and is filled by
//    16-byte cp.async copies (no registers, no transposing stores) into one of TWO buffers: the copies of
//    chunk c+1 fly while chunk c is summed.  (One CTA of 16 warps x 128 registers fills an SM, so in
//    k_incoherent the global loads of a chunk -- two batches, ~1.5 us each -- are exposed once per chunk,
//    about as long as the summing itself.)
//  * The 16-byte pieces of a row are XOR-swizzled with the row number (piece j of row r sits at
//    j ^ (r & 7)), so that a quarter warp -- 8 lanes = 8 consecutive time samples of one channel quad --
//    reads 8 different pieces: LDS.128 without bank conflicts.  A lane therefore takes FOUR channels of a
//    sample at once (they share the segment's first shift) and adds (x + y) + (z + w) into the run sum:
//    a quarter of the shared-memory instructions for the same bytes.  Where a segment starts or ends inside
//    a quad, the same 16-byte load is used and the channels of the neighbouring segment are replaced by
//    zeros (single LDS.32 column reads would meet 4-way bank conflicts in this layout).
//  * Everything else -- trial groups, runs, segments, end-of-run hand-over -- as in k_incoherent; the
//    additions of a run happen in another order (pairs inside a quad first), exact on integer data.
//  * The swizzle acts on the low three bits of the piece number for either row length (what a quarter
//    warp needs); 64 channels per chunk halve the block barriers per channel.
// ------------------------------------------------------------------------------------------------

__device__ __forceinline__ void ic_cp16(unsigned dst, const void *src, int bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}

// P_o[i] += sum of the four channels of quad j at rows s0 + o + lane + 32 i (+ the warp's time tile)
template <int SP, int NS, int RB>
__device__ __forceinline__ void ic4_quads(float (&P)[IC_MAXSPREAD + 1][NS], unsigned rowaddr, unsigned row7, int j0, int nq)
{
#pragma unroll 1
    for (int j = j0; j < j0 + nq; ++j) {
#pragma unroll
        for (int o = 0; o <= SP; ++o) {
            // row r = r_lane + o: its swizzle term is ((row7 + o) & 7); 32 i more rows do not change it
            const unsigned a = rowaddr + (unsigned)RB * o + (((unsigned)j ^ ((row7 + o) & 7u)) << 4);
#pragma unroll
            for (int i = 0; i < NS; ++i) {
                float x, y, z, w;
                asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x), "=f"(y), "=f"(z), "=f"(w) : "r"(a + 32u * RB * i));
                P[o][i] += (x + y) + (z + w);
            }
        }
    }
}
// a quad of which only channels [lo, hi) belong to the segment: the same LDS.128, the other components
// are replaced by zero (lo, hi are warp-uniform, so the selects cost no divergence)
template <int SP, int NS, int RB>
__device__ __forceinline__ void ic4_partial(float (&P)[IC_MAXSPREAD + 1][NS], unsigned rowaddr, unsigned row7, int j, int lo, int hi)
{
    const bool m0 = lo <= 0 && 0 < hi, m1 = lo <= 1 && 1 < hi, m2 = lo <= 2 && 2 < hi, m3 = lo <= 3 && 3 < hi;
#pragma unroll
    for (int o = 0; o <= SP; ++o) {
        const unsigned a = rowaddr + (unsigned)RB * o + (((unsigned)j ^ ((row7 + o) & 7u)) << 4);
#pragma unroll
        for (int i = 0; i < NS; ++i) {
            float x, y, z, w;
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x), "=f"(y), "=f"(z), "=f"(w) : "r"(a + 32u * RB * i));
            P[o][i] += ((m0 ? x : 0.f) + (m1 ? y : 0.f)) + ((m2 ? z : 0.f) + (m3 ? w : 0.f));
        }
    }
}
// channels [a0, a1) of the staged chunk (chunk-relative), all with the first shift of `rowaddr`
template <int SP, int NS, int RB>
__device__ __forceinline__ void ic4_seg_add(float (&P)[IC_MAXSPREAD + 1][NS], unsigned rowaddr, unsigned row7, int a0, int a1)
{
    if (a0 & 3) {   // head: the rest of the quad a0 sits in (or the whole segment, if it ends inside that quad)
        const int qe = min((a0 | 3) + 1, a1);
        ic4_partial<SP, NS, RB>(P, rowaddr, row7, a0 >> 2, a0 & 3, qe - (a0 & ~3));
        a0 = qe;
    }
    const int nq = (a1 - a0) >> 2;
    if (nq > 0) ic4_quads<SP, NS, RB>(P, rowaddr, row7, a0 >> 2, nq);
    a0 += 4 * nq;
    if (a0 < a1) ic4_partial<SP, NS, RB>(P, rowaddr, row7, a0 >> 2, 0, a1 - a0);
}

// NS = samples per lane: 8 (256-sample tiles, 128 registers, one CTA per SM) or 4 (128-sample tiles, 64
// registers, two CTAs = 32 warps per SM: the kernel waits on shared-memory latency and on the block barrier,
// and twice the resident warps cover both)
template <bool MULTI, int NS, int CC>
__global__ void __launch_bounds__(32 * IC_WARPS, NS == 8 ? 1 : 2) k_incoherent_v4(const IcArgs a)
{
    constexpr int TILE = 32 * NS;                           // output samples per warp
    const int gpc = MULTI ? a.gpc : IC_WARPS, tt = MULTI ? a.tt : 1;
    extern __shared__ float4 ic_smem4[];
    const int rows = a.tw;                                  // input samples staged per chunk: range + 256 tt
    const unsigned tile0 = (unsigned)__cvta_generic_to_shared(ic_smem4), tile_bytes = (unsigned)(4 * CC) * (unsigned)rows;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tbase = blockIdx.x * TILE * tt;
    const int gsel = MULTI ? warp % gpc : warp, sub = MULTI ? warp / gpc : 0;
    const int t0 = tbase + sub * TILE;
    const int grp = blockIdx.y * gpc + gsel;
    const bool live = sub < tt && grp < a.ngroups && t0 < a.nt_out;
    const float *fb = a.fb + (size_t)blockIdx.z * (size_t)a.fb_stride_dm;

    float acc[IC_GROUP][NS];
    float P[IC_MAXSPREAD + 1][NS];
#pragma unroll
    for (int k = 0; k < IC_GROUP; ++k)
#pragma unroll
        for (int i = 0; i < NS; ++i) acc[k][i] = 0.f;
#pragma unroll
    for (int o = 0; o <= IC_MAXSPREAD; ++o)
#pragma unroll
        for (int i = 0; i < NS; ++i) P[o][i] = 0.f;

    int cur = 0, cur_end = 0;
    if (live) {
        cur = a.seg_off[grp];
        cur_end = a.seg_off[grp + 1];
    }
    const uint4 seg_none = make_uint4(0x7fffffffu, 0x7fffffffu, 0u, 0u);
    uint4 sg = cur < cur_end ? ic_uniform(__ldg(a.segs + cur)) : seg_none;
    uint4 sg_next = cur + 1 < cur_end ? __ldg(a.segs + cur + 1) : seg_none;   // read one record ahead

    // 16-byte pieces of chunk c0 -> buffer `buf`; rows beyond the filterbank and channels beyond nch are zero
    auto stage = [&](int c0, int buf) {
        const unsigned dst0 = tile0 + (unsigned)buf * tile_bytes;
        for (int e = tid; e < rows * (CC / 4); e += 32 * IC_WARPS) {
            const int r = e / (CC / 4), j = e % (CC / 4), t = tbase + r, c = c0 + 4 * j;
            const bool ok = t < a.nt_in && c < a.nch;      // nch is a multiple of 4: a quad is in or out
            const float *src = ok ? fb + (size_t)t * a.nch + c : fb;
            ic_cp16(dst0 + (unsigned)(4 * CC) * r + ((unsigned)(j ^ (r & 7)) << 4), src, ok ? 16 : 0);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    // Two buffers, two block barriers per chunk.  (Three buffers need only one barrier per chunk -- the copies
    // of chunk c+1 then go where chunk c-2 was summed from -- but measured slower: c3 47.4 against 46.0 ms.)
    stage(0, 0);
    int buf = 0;
    for (int c0 = 0; c0 < a.nch; c0 += CC, buf ^= 1) {
        __syncthreads();                                   // the other buffer has been consumed
        if (c0 + CC < a.nch) {
            stage(c0 + CC, buf ^ 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();                                   // every thread's pieces of this chunk have landed
        if (!live) continue;
        while ((int)sg.x < c0 + CC) {
            const int a0 = max((int)sg.x, c0) - c0, a1 = min((int)sg.y, c0 + CC) - c0;
            const unsigned s0 = sg.z & 0xffffffu, spread = (sg.z >> 24) & 7u;
            const unsigned r_lane = s0 + lane + sub * TILE;
            const unsigned rowaddr = tile0 + (unsigned)buf * tile_bytes + (unsigned)(4 * CC) * r_lane, row7 = r_lane & 7u;
            switch (spread) {
            case 0: ic4_seg_add<0, NS, 4 * CC>(P, rowaddr, row7, a0, a1); break;
            case 1: ic4_seg_add<1, NS, 4 * CC>(P, rowaddr, row7, a0, a1); break;
            case 2: ic4_seg_add<2, NS, 4 * CC>(P, rowaddr, row7, a0, a1); break;
            case 3: ic4_seg_add<3, NS, 4 * CC>(P, rowaddr, row7, a0, a1); break;
            default: ic4_seg_add<4, NS, 4 * CC>(P, rowaddr, row7, a0, a1); break;
            }
            if ((int)sg.y > c0 + CC) break;
            if (sg.z & (1u << 28)) {
                unsigned o = 0;
#pragma unroll
                for (int k = 0; k < IC_GROUP; ++k) {
                    if (k > 0) o += (sg.w >> (2 * k)) & 3u;
                    if (o == 0u) {
#pragma unroll
                        for (int i = 0; i < NS; ++i) acc[k][i] += P[0][i];
                    } else if (o == 1u) {
#pragma unroll
                        for (int i = 0; i < NS; ++i) acc[k][i] += P[1][i];
                    } else if (o == 2u) {
#pragma unroll
                        for (int i = 0; i < NS; ++i) acc[k][i] += P[2][i];
                    } else if (o == 3u) {
#pragma unroll
                        for (int i = 0; i < NS; ++i) acc[k][i] += P[3][i];
                    } else {
#pragma unroll
                        for (int i = 0; i < NS; ++i) acc[k][i] += P[4][i];
                    }
                }
#pragma unroll
                for (int oo = 0; oo <= IC_MAXSPREAD; ++oo)
#pragma unroll
                    for (int i = 0; i < NS; ++i) P[oo][i] = 0.f;
            }
            ++cur;
            sg = ic_uniform(sg_next);
            sg_next = cur + 1 < cur_end ? __ldg(a.segs + cur + 1) : seg_none;
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
        for (int i = 0; i < NS; ++i) {
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
        auto smem_for = [&](int cc) { return sizeof(float) * (((size_t)cc * tw + 3) & ~(size_t)3); };
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

// k_incoherent_v4: trial groups and time tiles per CTA as above; two tiles of (range + tile tt) rows of 128 bytes
static bool incoherent_config_v4(const IncoherentTables &T, int tile, int cc, size_t smem_max, int *rows_out, int *gpc_out, int *tt_out, size_t *smem_out)
{
    const int ngroups = (int)T.groups.size();
    if (ngroups < 1) return false;
    const int ny = (ngroups + IC_WARPS - 1) / IC_WARPS;
    if (ny > 65535) return false;
    const int gpc = (ngroups + ny - 1) / ny;
    for (int tt = IC_WARPS / gpc; tt >= 1; --tt) {
        const int rows = T.range + tt * tile;
        const size_t smem = 2 * (size_t)rows * 4 * cc;
        if (smem <= smem_max) {
            *rows_out = rows; *gpc_out = gpc; *tt_out = tt; *smem_out = smem;
            return true;
        }
    }
    return false;
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
    const size_t nb_s = T.segs.size() * sizeof(uint4), nb_o = T.seg_off.size() * sizeof(int), nb_g = T.groups.size() * sizeof(int2);
    const size_t off_o = ic_align(nb_s), off_g = off_o + ic_align(nb_o), total = off_g + nb_g;
    // the tables travel from page-locked memory the plan keeps for them: one plain asynchronous copy on the
    // caller's stream, also inside a stream capture
    if (!T.pinned) {
        cudaError_t e = cudaMallocHost(&T.pinned, total);
        if (e != cudaSuccess) return e;
        memset(T.pinned, 0, total);
        memcpy(T.pinned, T.segs.data(), nb_s);
        memcpy(static_cast<char *>(T.pinned) + off_o, T.seg_off.data(), nb_o);
        memcpy(static_cast<char *>(T.pinned) + off_g, T.groups.data(), nb_g);
    }
    cudaError_t e = cudaMemcpyAsync(ws, T.pinned, total, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;

    IcArgs a;
    a.fb = d_fb; a.fb_stride_dm = fb_stride_dm; a.ts = d_ts; a.ts_stride_dm = ts_stride_dm; a.ts_pitch = ts_pitch;
    a.segs = reinterpret_cast<const uint4 *>(ws);
    a.seg_off = reinterpret_cast<const int *>(ws + off_o);
    a.groups = reinterpret_cast<const int2 *>(ws + off_g);
    a.nt_in = (int)nt_in; a.nt_out = (int)nt_out; a.nch = nch; a.ngroups = ngroups;
    size_t smem = 0;
    a.vec_in = (nch % 4 == 0 && fb_stride_dm % 4 == 0 && (reinterpret_cast<uintptr_t>(d_fb) & 15) == 0) ? 1 : 0;
    // rows readable in 16-byte pieces and two tiles in shared memory: the cp.async / LDS.128 kernel, with
    // 128-sample tiles and two CTAs per SM where two such tiles take at most half of shared memory
    // (the 256-sample form where both apply: c3 48.6 against 41.5 ms, c4 237 / 204, c5 122 / 115; 64-sample
    // tiles with three CTAs per SM spill at 40 registers: c3 49.8 ms)
    if (a.vec_in) {
        // 64 channels per chunk halve the block barriers per channel (c3 41.5 -> 39.0 ms, c4 204 -> 162 ms) unless
        // the larger tiles leave room for fewer time tiles per CTA (c5: 7 trial groups x 2 time tiles only with 32)
        int ns = 0, cc = 0;
        {
            int tw64 = 0, gpc64 = 0, tt64 = 0, tw32 = 0, gpc32 = 0, tt32 = 0;
            size_t sm64 = 0, sm32 = 0;
            const bool ok64 = incoherent_config_v4(T, 128, 64, 110u * 1024, &tw64, &gpc64, &tt64, &sm64);
            const bool ok32 = incoherent_config_v4(T, 128, 32, 110u * 1024, &tw32, &gpc32, &tt32, &sm32);
            if (ok64 && (!ok32 || tt64 >= tt32)) ns = 4, cc = 64, a.tw = tw64, a.gpc = gpc64, a.tt = tt64, smem = sm64;
            else if (ok32) ns = 4, cc = 32, a.tw = tw32, a.gpc = gpc32, a.tt = tt32, smem = sm32;
            else if (incoherent_config_v4(T, 256, 32, 224u * 1024, &a.tw, &a.gpc, &a.tt, &smem)) ns = 8, cc = 32;
        }
        if (ns) {
            a.cc = cc;
            const bool multi = !(a.gpc == IC_WARPS && a.tt == 1);
            const void *fn = ns == 8 ? (multi ? (const void *)k_incoherent_v4<true, 8, 32> : (const void *)k_incoherent_v4<false, 8, 32>)
                           : cc == 64 ? (multi ? (const void *)k_incoherent_v4<true, 4, 64> : (const void *)k_incoherent_v4<false, 4, 64>)
                                      : (multi ? (const void *)k_incoherent_v4<true, 4, 32> : (const void *)k_incoherent_v4<false, 4, 32>);
            e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            const int tile = 32 * ns;
            dim3 grid((unsigned)((nt_out + tile * a.tt - 1) / (tile * a.tt)), (unsigned)((ngroups + a.gpc - 1) / a.gpc), (unsigned)g.ndm);
            void *args[] = {&a};
            e = cudaLaunchKernel(fn, grid, dim3(32 * IC_WARPS), args, smem, st);
            if (e == cudaSuccess) ++*launches;
            return e;
        }
    }
    if (!incoherent_config(T, &a.cc, &a.tw, &a.gpc, &a.tt, &smem)) return cudaErrorInvalidValue;
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
