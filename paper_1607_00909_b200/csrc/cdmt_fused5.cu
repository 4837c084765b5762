// cdmt_fused5.cu -- k_fused_ws: the fused per-DM kernel (Alg. 1 l.99-103 + time integration,
// PAPER.md:117-123), warp-specialised.
//
// Same arithmetic as k_fused_x2 (cdmt_fused2.cu): the length-M backward FFT of a channel as two
// half transforms of length L = M/2 = 16 * 16 * R2 in the two lanes of f32x2 registers, radix-2
// combine, detection, Stokes I, time integration.  What changes is WHO forms the chirp of Eq. 1
// and how the trial is ordered:
//
//  * The chirp does not depend on the data block (one transfer function per DM and
//    channel, applied to every block).  A CTA therefore takes TWO blocks of the same (subband,
//    channel) -- FFT group A = warps 0-3, FFT group B = warps 4-7 -- and a third warp group
//    (warps 8-11, "chirp warps") forms H(DM_d) once for both: FP64 phase polynomial, mod-1
//    reduction, MUFU sin/cos, exactly as in k_fused_x2.  Chirp warp q and warp q of either FFT
//    group own the same 32 lanes of tensor memory, and thread l of all three works on the same
//    bins, so H travels through TMEM (tcgen05.st by the producer, tcgen05.ld by the two
//    consumers; two buffers, full/empty mbarriers) without touching shared memory.  The FP64 and
//    XU pipes now run beside the FP32 pipe instead of in turn with it, and the chirp is computed
//    once per two blocks.  `setmaxnreg` moves the registers the chirp warps do not need to the
//    FFT warps (104 / 200 of the 3 x 168 the CTA is launched with).
//  * An FFT group never waits at its block barrier: the two polarisations have their own
//    exchange buffers and their own mbarriers, and are staggered --
//        pass 0 (X * H, radix 16) pol 0, pol 1 | pass 1 pol 0, arrive A0 | pass 1 pol 1, arrive A1
//        | wait A0, pass 2 + combine + detect pol 0 | wait A1, the same for pol 1 | integrate, store
//    so every wait has a whole pass of the other polarisation in front of it.
//
// TMEM map of a lane (512 columns): [0,128) X of group A, [128,256) X of group B, [256,384) the
// pass-1 / pass-2 / combine twiddles (the same for both groups), [384,448) and [448,512) H.
#include <cstdint>

#include "cdmt_fft2.cuh"
#include "cdmt_fused_common.cuh"
#include "cdmt_internal.h"
#include "cdmt_tmem.cuh"

namespace cdmt {

template <int M>
struct WS {
    static constexpr int L = M / 2;        // length of the two half transforms
    static constexpr int NT = L / 16;      // threads of one FFT group: 16 packed points each
    static constexpr int R2 = L / 256;     // radix of the last pass
    static constexpr int U2 = 16 / R2;     // last-pass butterflies per thread
    static constexpr int NWARP = NT / 32;  // warps per group (4)
    static constexpr int NGRP = 2;         // FFT groups (blocks) per CTA
    static constexpr int NTHREADS = (NGRP + 1) * NT;
    static constexpr int PITCH = 17;       // float4 per d1 row: conflict-free 16-byte accesses
    static constexpr int RHO = 16 * PITCH; // float4 per j2 plane
    static constexpr int EX = R2 * RHO;    // float4 per exchange buffer (one per polarisation and group)
    static constexpr int IROW = 34;        // float2 per integration row: 32 lanes + 16 bytes
    static constexpr int INTEG = 16 * IROW;
    static constexpr int COL_XA = 0, COL_TW1 = 256, COL_TW2 = 288, COL_TWF = 320, COL_H = 384;
    static constexpr int NBAR = 8 + 16 + 32;  // per group A0 A1 F0 F1; per quadrant H full[2] empty[2]; per (group, quadrant) tile full[2] empty[2]
    static constexpr size_t group_bytes = sizeof(float4) * 2 * EX + sizeof(float2) * 2 * NWARP * INTEG;  // two tiles per warp
    static constexpr size_t smem_bytes = 2 * group_bytes + sizeof(uint64_t) * NBAR + 16 + sizeof(double2) * 2 * NGRP * NWARP;
    static constexpr int REGS_FFT = 200, REGS_CHIRP = 104;  // 2 x 200 + 104 = 3 x 168: what the CTA holds at launch
};

__device__ __forceinline__ unsigned ws_f2u(float x) { return __float_as_uint(x); }
__device__ __forceinline__ float ws_u2f(unsigned x) { return __uint_as_float(x); }
__device__ __forceinline__ P2 ws_pku(unsigned lo, unsigned hi) { return pk(ws_u2f(lo), ws_u2f(hi)); }
__device__ __forceinline__ P2 ws_lo2(P2 v) { return bc(lo_of(v)); }
__device__ __forceinline__ P2 ws_hi2(P2 v) { return bc(hi_of(v)); }
__device__ __forceinline__ float4 ws_c2_to_f4(const C2 &v)
{
    float4 q;
    upk(v.re, q.x, q.y);
    upk(v.im, q.z, q.w);
    return q;
}
__device__ __forceinline__ C2 ws_f4_to_c2(const float4 &q) { return C2{pk(q.x, q.y), pk(q.z, q.w)}; }

// one lane of the warp arrives for all of it, after every lane's earlier TMEM traffic has been fenced
__device__ __forceinline__ void ws_warp_arrive(uint64_t *bar, int lane)
{
    tmem_fence_before_sync();
    __syncwarp();
    if (lane == 0) mbar_arrive(bar);
}

template <int M, int LOGD, bool SUMS>
__global__ void __launch_bounds__(WS<M>::NTHREADS, 1)
k_fused_ws(const FusedArgs a, const __grid_constant__ DmParams dmp)
{
    using G = WS<M>;
    constexpr int L = G::L, NT = G::NT, R2 = G::R2, U2 = G::U2;
    constexpr int D = 1 << LOGD;
    constexpr int DG = D > 16 ? 16 : D;  // lanes summed through the shared-memory tile
    static_assert(LOGD >= 3 && LOGD <= 5, "ndec 8, 16 or 32");
    static_assert(NT == 128, "one warpgroup per role");
    extern __shared__ float4 smem4[];
    uint64_t *bars = reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(smem4) + 2 * G::group_bytes);
    uint32_t *tslot = reinterpret_cast<uint32_t *>(bars + G::NBAR);
    double2 *psum = reinterpret_cast<double2 *>(tslot + 4);   // [parity][group][q]: the chirp warps' (sum I, sum I^2)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int role = warp >> 2;          // 0, 1: FFT group A, B; NGRP: chirp warps
    const int q = warp & 3;              // TMEM lane quadrant
    const int t = tid & (NT - 1);        // thread index inside the role: the same bins in all three
    const int bx = (int)blockIdx.x + a.cta0;
    const int c = bx % a.nchan;
    const int pl = bx / a.nchan;         // pair index inside the chunk: (bp, s)
    const int s = pl % a.nsub, bp = pl / a.nsub;
    const int nb_chunk = a.nb_chunk;     // whole blocks in this chunk (units = nb_chunk * nsub)
    const bool has_b = 2 * bp + 1 < nb_chunk;
    const int d_begin = a.dm_first + blockIdx.y * a.dm_tile;
    const int d_end = min(a.ndm, d_begin + a.dm_tile);

    if (warp == 0) tmem_alloc<512>(tslot);
    if (tid == 0) {
        for (int g = 0; g < 2; ++g)
            for (int k = 0; k < 4; ++k) mbar_init(bars + 4 * g + k, NT);
        for (int k = 0; k < 8; ++k) mbar_init(bars + 8 + k, 1);                       // full[q][buf]: the chirp warp
        for (int k = 0; k < 8; ++k) mbar_init(bars + 16 + k, has_b ? 2 : 1);          // empty[q][buf]: the consumers
        for (int k = 0; k < 32; ++k) mbar_init(bars + 24 + k, 1);                     // tile full / empty[g][q][buf]
    }
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tbase = *tslot;
    const uint32_t tcol = tbase + ((uint32_t)(32 * q) << 16);
    uint64_t *full = bars + 8 + 2 * q, *empty = bars + 16 + 2 * q;
    // tile hand-over between FFT warp (g, q) and chirp warp q: bars[24 + 4 (4 g + q) + 2 buf] = full, + 1 = empty

    const int j1 = t & 15, j2 = t >> 4;      // pass-0 role; pass 1: (j2, t0 = t & 15)
    const int rest = j1 * R2 + j2;           // half-transform input index j = j0 L/16 + rest

    if (role == G::NGRP) {
        // ------------------------------------------------------------------ chirp warps
        {
            // pass twiddles of thread t: w1[r] = exp(2 pi i r t0 / 256), w2[u][r] = exp(2 pi i r beta_u / L)
            unsigned r[32];
#pragma unroll
            for (int rr = 0; rr < 16; ++rr) {
                float sn, cs;
                sincospif((float)(2 * rr * (t & 15)) * (1.0f / 256.0f), &sn, &cs);
                r[2 * rr] = ws_f2u(cs);
                r[2 * rr + 1] = ws_f2u(sn);
            }
            tmem_st32(tcol + G::COL_TW1, r);
#pragma unroll
            for (int u = 0; u < U2; ++u)
#pragma unroll
                for (int rr = 0; rr < R2; ++rr) {
                    float sn, cs;
                    sincospif((float)(2 * rr * (t + NT * u)) * (1.0f / (float)L), &sn, &cs);
                    r[2 * (u * R2 + rr)] = ws_f2u(cs);
                    r[2 * (u * R2 + rr) + 1] = ws_f2u(sn);
                }
            tmem_st32(tcol + G::COL_TW2, r);
            // combine twiddles in the order the last pass leaves its outputs: k = u R2 + t2 holds
            // t' = t + NT n, n = u + U2 t2, as the pairs (wr, -wr), (wi, -wi) of w_M^t'
#pragma unroll
            for (int h = 0; h < 2; ++h) {
#pragma unroll
                for (int kk = 0; kk < 8; ++kk) {
                    const int k = 8 * h + kk;
                    const int n = (k / R2) + U2 * (k % R2);
                    float sn, cs;
                    sincospif((float)(2 * (t + NT * n)) * (1.0f / (float)M), &sn, &cs);
                    r[4 * kk + 0] = ws_f2u(cs);
                    r[4 * kk + 1] = ws_f2u(-cs);
                    r[4 * kk + 2] = ws_f2u(sn);
                    r[4 * kk + 3] = ws_f2u(-sn);
                }
                tmem_st32(tcol + G::COL_TWF + 32 * h, r);
            }
        }
        // Eq. 1 along this thread's bins m = 2 rest + e + r M/16 (e = 0 even lane, 1 odd lane):
        // g(f_a + bb r) = sum_k c_k r^k, Taylor in bb r / (f0 + f_a) <= 1e-3 (host checks the r^6 term)
        double ce[6], co[6];
        {
            double f0, fb0, df;
            chirp_axes(a, s, c, M, &f0, &fb0, &df);
            const double kc = 1.0 / (2.41e-10 * f0 * f0), bb = (double)(M / 16) * df;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const double fa = fb0 + (double)(2 * rest + e) * df;
                const double sa = f0 + fa, ee = bb / sa, pp = kc * f0 * f0 / sa;
                const double c2 = pp * ee * ee, c3 = -c2 * ee, c4 = -c3 * ee, c5 = -c4 * ee;
                double *cc = e ? co : ce;
                cc[0] = kc * fa * fa / sa;
                cc[1] = kc * (fa * fa + 2.0 * fa * f0) / (sa * sa) * bb;
                cc[2] = c2;
                cc[3] = c3;
                cc[4] = c4;
                cc[5] = c5;
            }
        }
        tmem_fence_before_sync();
        __syncthreads();  // X and twiddles are in TMEM
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(G::REGS_CHIRP));
        // Epilogue of trial index j, for both FFT groups: the FFT warp (g, q) left the 32 powers of each of its
        // lanes (times t + NT n [+ L]) in a tile; here one lane sums the D adjacent samples of a row (time
        // integration, north_star), scales and stores them time-major, and -- SUMS -- the warp
        // adds the stored values and their squares in fp64 (block sums of Alg. 1 l.104), the four chirp warps
        // meet at a named barrier and one thread per group adds the four pairs in quadrant order.
        const int nchan_total = a.nsub * a.nchan;
        const int ochan = nchan_total - 1 - (s * a.nchan + c);
        const int il = lane & (DG - 1), g0 = lane - il;
        const int tgrp = (D > 16) ? (t & ~31) : (t - il);  // first sample of a lane's group, before + NT n
        auto epilogue = [&](unsigned j) {
            const unsigned tb = j & 1u, tpar = (j >> 1) & 1u;
            double2 *ps = psum + (size_t)tb * G::NGRP * G::NWARP;
#pragma unroll
            for (int g = 0; g < G::NGRP; ++g) {
                if (g == 1 && !has_b) break;
                uint64_t *tbar = bars + 24 + 4 * (4 * g + q) + 2 * tb;
                const float2 *ib = reinterpret_cast<const float2 *>(smem4 + (size_t)g * (G::group_bytes / sizeof(float4)) + 2 * G::EX) +
                                   (size_t)(2 * q + tb) * G::INTEG;
                const int b = a.unit0 / a.nsub + 2 * bp + g;
                float *outd = a.out + (size_t)(d_begin + (int)j) * (size_t)a.out_stride_dm + (size_t)b * a.vdec * a.out_pitch + ochan;
                mbar_wait(tbar, tpar);  // the FFT warp has filled the tile
                double sum1 = 0.0, sum2 = 0.0;
#pragma unroll
                for (int kk = 0; kk < 16 / DG; ++kk) {
                    const int n = il + DG * kk;
                    const float4 *row = reinterpret_cast<const float4 *>(ib + n * G::IROW + g0);
                    P2 acc = pk(0.f, 0.f);
#pragma unroll
                    for (int qq = 0; qq < DG / 2; ++qq) {
                        const float4 f = row[qq];
                        acc = add2(acc, add2(pk(f.x, f.y), pk(f.z, f.w)));
                    }
                    float s0, s1;
                    upk(acc, s0, s1);
                    if (D > 16) {
                        s0 += __shfl_xor_sync(0xffffffffu, s0, 16);
                        s1 += __shfl_xor_sync(0xffffffffu, s1, 16);
                    }
                    const int t0 = tgrp + NT * n;
                    if (D <= 16 || lane < 16) {
                        if (t0 >= a.hdisc && t0 < M - a.hdisc) {
                            const float f = s0 * a.scale;
                            outd[(size_t)((t0 - a.hdisc) >> LOGD) * a.out_pitch] = f;
                            if (SUMS) { sum1 += (double)f; sum2 = fma((double)f, (double)f, sum2); }
                        }
                        const int t1 = t0 + L;
                        if (t1 >= a.hdisc && t1 < M - a.hdisc) {
                            const float f = s1 * a.scale;
                            outd[(size_t)((t1 - a.hdisc) >> LOGD) * a.out_pitch] = f;
                            if (SUMS) { sum1 += (double)f; sum2 = fma((double)f, (double)f, sum2); }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(tbar + 1);  // the tile may be filled again
                if (SUMS) {
                    warp_sum_pair(sum1, sum2);
                    if (lane == 0) ps[g * G::NWARP + q] = make_double2(sum1, sum2);
                }
            }
            if (SUMS) {
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (t < G::NGRP && (t == 0 || has_b)) {
                    double a1 = 0.0, a2 = 0.0;
#pragma unroll
                    for (int w = 0; w < G::NWARP; ++w) {
                        a1 += ps[t * G::NWARP + w].x;
                        a2 += ps[t * G::NWARP + w].y;
                    }
                    const int b = a.unit0 / a.nsub + 2 * bp + t;
                    a.segsum[((size_t)(d_begin + (int)j) * a.nblock_total + b) * nchan_total + ochan] = make_double2(a1, a2);
                }
            }
        };
#pragma unroll 1
        for (int d = d_begin; d < d_end; ++d) {
            const unsigned i = (unsigned)(d - d_begin), buf = i & 1u;
            if (i >= 2u) {
                mbar_wait(empty + buf, ((i >> 1) & 1u) ^ 1u);  // both consumers have read H(d-2)
                tmem_fence_after_sync();
            }
            const double dm = dmp.dm[d - a.dm_param0];
            double pe[6], po[6];
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                pe[k] = dm * ce[k];
                po[k] = dm * co[k];
            }
#pragma unroll
            for (int part = 0; part < 4; ++part) {
                unsigned h[16];
#pragma unroll
                for (int rr = 0; rr < 4; ++rr) {
                    const double x = (double)(4 * part + rr);
                    const double phe = fma(fma(fma(fma(fma(pe[5], x, pe[4]), x, pe[3]), x, pe[2]), x, pe[1]), x, pe[0]);
                    const double pho = fma(fma(fma(fma(fma(po[5], x, po[4]), x, po[3]), x, po[2]), x, po[1]), x, po[0]);
                    // adding 1.5 * 2^20 leaves round(phi * 2^32) mod 2^32 in the low mantissa word: the
                    // fraction of a cycle as a signed fixed-point number (|phi| < 2^19, checked on the host)
                    const float xe = __int2float_rn(__double2loint(phe + 1572864.0)) * 1.4629180792671596e-9f;
                    const float xo = __int2float_rn(__double2loint(pho + 1572864.0)) * 1.4629180792671596e-9f;
                    h[4 * rr + 0] = ws_f2u(__cosf(xe));
                    h[4 * rr + 1] = ws_f2u(__cosf(xo));
                    h[4 * rr + 2] = ws_f2u(__sinf(xe));
                    h[4 * rr + 3] = ws_f2u(__sinf(xo));
                }
                tmem_st16(tcol + G::COL_H + 64 * buf + 16 * part, h);
            }
            ws_warp_arrive(full + buf, lane);
            // while the FFT warps work on trial i with the chirp just delivered: the epilogue of trial i - 1
            if (i >= 1u) epilogue(i - 1u);
        }
        if (d_begin < d_end) epilogue((unsigned)(d_end - d_begin) - 1u);
    } else {
        // ------------------------------------------------------------------ FFT groups
        const bool active = role == 0 || has_b;
        const int g = role;
        float4 *ex0 = smem4 + (size_t)g * (G::group_bytes / sizeof(float4)), *ex1 = ex0 + G::EX;
        float2 *ib0 = reinterpret_cast<float2 *>(ex0 + 2 * G::EX) + (size_t)(2 * (warp & 3)) * G::INTEG;  // this warp's two tiles
        uint64_t *tbar = bars + 24 + 4 * (4 * g + q);
        uint64_t *barA0 = bars + 4 * g, *barA1 = barA0 + 1, *barF0 = barA0 + 2, *barF1 = barA0 + 3;
        const int blk = 2 * bp + g;                               // block inside the chunk
        const int ulocal = blk * a.nsub + s;
        const uint32_t tX = tcol + (uint32_t)(128 * g);
        if (active) {
            // this thread's bins 2j, 2j+1 of both polarisations -> TMEM as (re_e, re_o, im_e, im_o)
            const float4 *src = reinterpret_cast<const float4 *>(a.spec + ((size_t)ulocal * 2) * a.nfft + (size_t)c * M);
#pragma unroll
            for (int pol = 0; pol < 2; ++pol) {
                unsigned r[64];
#pragma unroll
                for (int j0 = 0; j0 < 16; ++j0) {
                    const float4 v = __ldg(src + (size_t)pol * (a.nfft / 2) + j0 * (L / 16) + rest);
                    r[4 * j0 + 0] = ws_f2u(v.x);
                    r[4 * j0 + 1] = ws_f2u(v.z);
                    r[4 * j0 + 2] = ws_f2u(v.y);
                    r[4 * j0 + 3] = ws_f2u(v.w);
                }
                tmem_st64(tX + 64 * pol, r);
            }
        }
        tmem_fence_before_sync();
        __syncthreads();
        tmem_fence_after_sync();
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(G::REGS_FFT));
        if (active) {
#pragma unroll 1
            for (int d = d_begin; d < d_end; ++d) {
                const unsigned i = (unsigned)(d - d_begin), buf = i & 1u, par = i & 1u;
                const uint32_t tH = tcol + G::COL_H + 64 * buf;
                // ---- pass 0: Z = X * H(d), radix 16 over j0, both polarisations.  X and H come from TMEM in
                //      pieces of four bins, the next piece in flight while this one is multiplied.
                mbar_wait(full + buf, (i >> 1) & 1u);  // H(d) written by the chirp warp
                tmem_fence_after_sync();
                unsigned hq[2][16], xq[2][16];
                tmem_ld16_async(hq[0], tH);
                tmem_ld16_async(xq[0], tX);
#pragma unroll
                for (int pol = 0; pol < 2; ++pol) {
                    C2 v[16];
#pragma unroll
                    for (int cq = 0; cq < 4; ++cq) {
                        const int cur = cq & 1, nxt = cur ^ 1;
                        tmem_ld_wait();
                        tmem_regs16(hq[cur]);
                        tmem_regs16(xq[cur]);
                        if (cq < 3 || pol == 0) {
                            const int pn = cq < 3 ? pol : 1, cn = cq < 3 ? cq + 1 : 0;
                            tmem_ld16_async(hq[nxt], tH + 16 * cn);
                            tmem_ld16_async(xq[nxt], tX + 64 * pn + 16 * cn);
                        }
#pragma unroll
                        for (int rr = 0; rr < 4; ++rr) {
                            const int r = 4 * cq + rr;
                            v[r] = cmulp(C2{ws_pku(xq[cur][4 * rr], xq[cur][4 * rr + 1]), ws_pku(xq[cur][4 * rr + 2], xq[cur][4 * rr + 3])},
                                         ws_pku(hq[cur][4 * rr], hq[cur][4 * rr + 1]), ws_pku(hq[cur][4 * rr + 2], hq[cur][4 * rr + 3]));
                        }
                    }
                    PDft<16>::run(v);
                    if (i != 0u) mbar_wait(pol ? barF1 : barF0, par ^ 1u);  // pass-2 loads of trial d-1 are done
                    float4 *dst = (pol ? ex1 : ex0) + j2 * G::RHO + j1 * G::PITCH;
#pragma unroll
                    for (int t0 = 0; t0 < 16; ++t0) dst[t0] = ws_c2_to_f4(v[t0]);
                }
                ws_warp_arrive(empty + buf, lane);  // H(d) consumed; also orders the half-warp exchange below
                // ---- pass 1: along j1, in place, half-warp local; both polarisations' loads up front
                unsigned w2[32];
                {
                    unsigned w1[32];
                    tmem_ld32_async(w1, tcol + G::COL_TW1);
                    float4 *p0 = ex0 + j2 * G::RHO + (t & 15), *p1 = ex1 + j2 * G::RHO + (t & 15);
                    C2 v0[16], v1[16];
#pragma unroll
                    for (int d1 = 0; d1 < 16; ++d1) v0[d1] = ws_f4_to_c2(p0[d1 * G::PITCH]);
#pragma unroll
                    for (int d1 = 0; d1 < 16; ++d1) v1[d1] = ws_f4_to_c2(p1[d1 * G::PITCH]);
                    tmem_ld_wait();
                    tmem_regs32(w1);
#pragma unroll
                    for (int d1 = 1; d1 < 16; ++d1) v0[d1] = cmuls(v0[d1], ws_u2f(w1[2 * d1]), ws_u2f(w1[2 * d1 + 1]));
                    PDft<16>::run(v0);
#pragma unroll
                    for (int t1 = 0; t1 < 16; ++t1) p0[t1 * G::PITCH] = ws_c2_to_f4(v0[t1]);
                    mbar_arrive(barA0);
#pragma unroll
                    for (int d1 = 1; d1 < 16; ++d1) v1[d1] = cmuls(v1[d1], ws_u2f(w1[2 * d1]), ws_u2f(w1[2 * d1 + 1]));
                    tmem_ld32_async(w2, tcol + G::COL_TW2);  // for pass 2, in flight during this butterfly
                    PDft<16>::run(v1);
#pragma unroll
                    for (int t1 = 0; t1 < 16; ++t1) p1[t1 * G::PITCH] = ws_c2_to_f4(v1[t1]);
                    mbar_arrive(barA1);
                }
                // ---- pass 2 along j2, radix-2 combine, detection, polarisation sum
                P2 pw[16];  // (|y[t']|^2, |y[t' + L]|^2) summed over polarisations, order k = u R2 + t2
#pragma unroll
                for (int pol = 0; pol < 2; ++pol) {
                    const float4 *ex = pol ? ex1 : ex0;
                    mbar_wait(pol ? barA1 : barA0, par);
                    C2 v[16];
#pragma unroll
                    for (int u = 0; u < U2; ++u) {
                        const int beta = t + NT * u;
                        const float4 *p = ex + (beta >> 4) * G::PITCH + (beta & 15);
#pragma unroll
                        for (int rr = 0; rr < R2; ++rr) v[u * R2 + rr] = ws_f4_to_c2(p[rr * G::RHO]);
                    }
                    if (pol == 0) {
                        tmem_ld_wait();
                        tmem_regs32(w2);
                    }
                    unsigned wf[2][16];
                    tmem_ld16_async(wf[0], tcol + G::COL_TWF);
#pragma unroll
                    for (int u = 0; u < U2; ++u) {
#pragma unroll
                        for (int rr = 1; rr < R2; ++rr)
                            v[u * R2 + rr] = cmuls(v[u * R2 + rr], ws_u2f(w2[2 * (u * R2 + rr)]), ws_u2f(w2[2 * (u * R2 + rr) + 1]));
                    }
                    mbar_arrive(pol ? barF1 : barF0);  // this thread's loads of the trial have been consumed
#pragma unroll
                    for (int u = 0; u < U2; ++u) PDft<R2>::run(v + u * R2);
#pragma unroll
                    for (int cq = 0; cq < 4; ++cq) {
                        const int cur = cq & 1, nxt = cur ^ 1;
                        tmem_ld_wait();
                        tmem_regs16(wf[cur]);
                        if (cq < 3) tmem_ld16_async(wf[nxt], tcol + G::COL_TWF + 16 * (cq + 1));
#pragma unroll
                        for (int kk = 0; kk < 4; ++kk) {
                            const int k = 4 * cq + kk;
                            const P2 Wr = ws_pku(wf[cur][4 * kk], wf[cur][4 * kk + 1]), Wi = ws_pku(wf[cur][4 * kk + 2], wf[cur][4 * kk + 3]);
                            const P2 re = v[k].re, im = v[k].im;  // lanes (A, B)
                            const P2 yr = fma2(ws_hi2(im), neg2(Wi), fma2(ws_hi2(re), Wr, ws_lo2(re)));
                            const P2 yi = fma2(ws_hi2(re), Wi, fma2(ws_hi2(im), Wr, ws_lo2(im)));
                            pw[k] = pol ? fma2(yi, yi, fma2(yr, yr, pw[k])) : fma2(yi, yi, mul2(yr, yr));
                        }
                    }
                }
                // ---- hand-over to the chirp warp of this quadrant, which integrates and stores: the 32 powers of
                //      this thread (times t + NT n [+ L]) go to one of the warp's two tiles
                if (i >= 2u) mbar_wait(tbar + 2 * buf + 1, ((i >> 1) & 1u) ^ 1u);  // tile of trial d - 2 has been read
                {
                    float2 *ib = ib0 + (size_t)buf * G::INTEG;
#pragma unroll
                    for (int k = 0; k < 16; ++k) {
                        const int n = (k / R2) + U2 * (k % R2);
                        float2 v2;
                        upk(pw[k], v2.x, v2.y);
                        ib[n * G::IROW + lane] = v2;
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(tbar + 2 * buf);
            }
        }
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(tbase);
}

// ------------------------------------------------------------------------------------
// launch
// ------------------------------------------------------------------------------------
template <int M, int LOGD>
static cudaError_t launch_ws_MD(FusedArgs fa, const double *h_dm, int nunits, cudaStream_t st, long long *launches)
{
    using G = WS<M>;
    const bool sums = fa.segsum != nullptr;
    cudaError_t e = sums ? cudaFuncSetAttribute(k_fused_ws<M, LOGD, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem_bytes)
                         : cudaFuncSetAttribute(k_fused_ws<M, LOGD, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem_bytes);
    if (e != cudaSuccess) return e;
    const int ndm_total = fa.ndm;
    fa.nb_chunk = nunits / fa.nsub;
    const int npairs = (fa.nb_chunk + 1) / 2 * fa.nsub;
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    for (int d0 = 0; d0 < ndm_total; d0 += DM_PARAM_MAX) {
        const int cnt = ndm_total - d0 < DM_PARAM_MAX ? ndm_total - d0 : DM_PARAM_MAX;
        DmParams dmp;
        for (int i = 0; i < cnt; ++i) dmp.dm[i] = h_dm[d0 + i];
        for (int i = cnt; i < DM_PARAM_MAX; ++i) dmp.dm[i] = 0.0;
        fa.dm_first = d0;
        fa.dm_param0 = d0;
        fa.ndm = d0 + cnt;
        // Every CTA runs all its trials on one SM for the same time, so a launch of n CTAs on S SMs costs
        // ceil(n / S) waves: a small launch (a host group of two blocks of c3 is 4608 CTAs = 31.1 waves) idles
        // through most of its last wave.  Where that matters the CTAs beyond the last full wave are launched
        // apart, each cut into DM tiles, as many as fill the SMs once: one short wave instead of a long one.
        const int nctas = npairs * fa.nchan;
        const int full = nctas / nsm * nsm, rem = nctas - full;
        const bool split = fa.dm_tile >= cnt && rem > 0 && full > 0 && nctas / nsm < 100 && 2 * rem <= nsm && cnt >= 16;
        auto launch = [&](int cta0, int n, int tile) {
            FusedArgs la = fa;
            la.cta0 = cta0;
            la.dm_tile = tile;
            dim3 grid((unsigned)n, (unsigned)((cnt + tile - 1) / tile));
            if (sums) k_fused_ws<M, LOGD, true><<<grid, G::NTHREADS, G::smem_bytes, st>>>(la, dmp);
            else k_fused_ws<M, LOGD, false><<<grid, G::NTHREADS, G::smem_bytes, st>>>(la, dmp);
            ++*launches;
            return cudaGetLastError();
        };
        if (!split) {
            e = launch(0, nctas, fa.dm_tile);
        } else {
            e = launch(0, full, fa.dm_tile);
            if (e != cudaSuccess) return e;
            int ny = nsm / rem;
            if (ny > cnt / 8) ny = cnt / 8;   // at least 8 trials per CTA: its set-up costs about one
            e = launch(full, rem, (cnt + ny - 1) / ny);
        }
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// whole blocks only: the chunk must start at a block boundary and hold every subband of its blocks
bool fused_ws_supported(int M, int ndec, int hdisc, int nsub, int unit0, int nunits)
{
    if (M != 4096) return false;
    if (ndec != 8 && ndec != 16 && ndec != 32) return false;
    if (hdisc % ndec != 0) return false;
    return unit0 % nsub == 0 && nunits % nsub == 0;
}

cudaError_t launch_fused_ws(int M, int logd, const FusedArgs &fa, const double *h_dm, int nunits, cudaStream_t st,
                            long long *launches)
{
    if (M != 4096) return cudaErrorInvalidValue;
    switch (logd) {
    case 3: return launch_ws_MD<4096, 3>(fa, h_dm, nunits, st, launches);
    case 4: return launch_ws_MD<4096, 4>(fa, h_dm, nunits, st, launches);
    case 5: return launch_ws_MD<4096, 5>(fa, h_dm, nunits, st, launches);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace cdmt
