// kernels_fused.cu -- fused forward step: E update + H update (+ CPML psi, sources, detectors) in ONE
// pass over the grid (rows F1-F7 of DESIGN.md; Eq. 1-2).
//
// Design:
//   * ping-pong: step n reads buffer n&1 and writes buffer (n+1)&1, so tiles are independent;
//   * the xy plane is cut into TX x TY tiles, a tile's z column into segments; a persistent CTA
//     (one per SM) marches its segments plane by plane (2.5-D blocking);
//   * one producer warp streams each plane's boxes (6 fields, inv_eps, psi slabs) global->shared with
//     TMA (cp.async.bulk.tensor, zero fill outside the grid = the zero-pad wall convention) through an
//     mbarrier full/empty ring; consumer warps hold a float4 of cells per thread;
//   * plane kk: phase A computes E'(kk) on the tile plus a +x halo column and +y halo row (recomputed,
//     not exchanged), phase B computes H'(kk-1) from E'(kk-1) (registers + shared ring) and E'(kk);
//   * algorithmic traffic: 6 reads + 6 writes + inv_eps per cell, psi read+write on slab cells only.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "fdtd_grid.h"
#include "fused_common.cuh"

using namespace fdtd;

namespace {

constexpr int MAX_SRC = 4, MAX_DET = 4;
constexpr int MAX_THREADS = 512;      // 128 registers per thread at one CTA per SM

struct FwdParams {
    Dims G;
    Tables T;
    const CUtensorMap *maps;
    const Segment *segs;
    const int *seg_begin;          // [n_cta + 1]
    float *buf[2];                 // ping-pong field buffers, [6][nc] each
    PsiSet psiE[2], psiH[2];
    const int *step;
    int TX, TY, TX4, NT, NCW;      // tile, float4s per row, active consumer threads, consumer warps
    int PW, ROWS, XW;              // box width / rows, narrow x-psi box width
    int big_bytes, small_bytes, stage_bytes, nstages;
    int slot_off[SA_COUNT];        // byte offset of each logical array inside a stage
    int ring_off, bar_off;         // byte offsets in dynamic smem
    int RP;                        // ring row pitch (floats)
    int has_mu;
    int n_src, n_det, total_freq;
    SourceDev src[MAX_SRC];
    DetectorDev det[MAX_DET];
    const float *cs;
};

__device__ __forceinline__ float4 lds4(const uint8_t *base, int off_bytes)
{
    return *reinterpret_cast<const float4 *>(base + off_bytes);
}
__device__ __forceinline__ float lds1(const uint8_t *base, int off_bytes)
{
    return *reinterpret_cast<const float *>(base + off_bytes);
}
__device__ __forceinline__ float4 ldg4(const float *p) { return __ldg(reinterpret_cast<const float4 *>(p)); }
__device__ __forceinline__ void stg4(float *p, float4 v) { *reinterpret_cast<float4 *>(p) = v; }

__device__ __forceinline__ bool in_zslab(const Dims &G, int k) { return G.d > 0 && k >= 0 && k < G.nz && (k < G.d || k >= G.nz - G.d); }
__device__ __forceinline__ int zslab_index(const Dims &G, int k) { return k < G.d ? k : k - (G.nz - 2 * G.d); }

// additive source contribution to component `comp` at cell (i,j,k) during this step
__device__ __forceinline__ float source_at(const FwdParams &P, int n, int comp, int i, int j, int k)
{
    float acc = 0.f;
    for (int s = 0; s < P.n_src; ++s) {
        const SourceDev &q = P.src[s];
        if (q.comp != comp) continue;
        if (i < q.lo[0] || i >= q.hi[0] || j < q.lo[1] || j >= q.hi[1] || k < q.lo[2] || k >= q.hi[2]) continue;
        const int bx = q.hi[0] - q.lo[0], by = q.hi[1] - q.lo[1];
        const float pr = q.profile ? __ldg(q.profile + ((long long)(k - q.lo[2]) * by + (j - q.lo[1])) * bx + (i - q.lo[0])) : 1.f;
        acc += pr * __ldg(q.waveform + n);
    }
    return acc;
}

__device__ __forceinline__ bool any_source_plane(const FwdParams &P, int family, int k)
{
    for (int s = 0; s < P.n_src; ++s)
        if ((P.src[s].comp >= 3) == (family != 0) && k >= P.src[s].lo[2] && k < P.src[s].hi[2]) return true;
    return false;
}

// running DFT of component `comp` (value v) at cell (i,j,k): P_f += v (cos - i sin)
__device__ __forceinline__ void detect_cell(const FwdParams &P, int n, int comp, float v, int i, int j, int k)
{
    for (int s = 0; s < P.n_det; ++s) {
        const DetectorDev &q = P.det[s];
        if (!((q.mask >> comp) & 1)) continue;
        if (i < q.lo[0] || i >= q.hi[0] || j < q.lo[1] || j >= q.hi[1] || k < q.lo[2] || k >= q.hi[2]) continue;
        const int bx = q.hi[0] - q.lo[0], by = q.hi[1] - q.lo[1], bz = q.hi[2] - q.lo[2];
        const long long bc = (long long)bx * by * bz;
        const long long cell = ((long long)(k - q.lo[2]) * by + (j - q.lo[1])) * bx + (i - q.lo[0]);
        int ci = 0;
        for (int c = 0; c < comp; ++c) ci += (q.mask >> c) & 1;
        const float *csn = P.cs + ((long long)n * P.total_freq + q.cs_off) * 2;
        for (int f = 0; f < q.n_freq; ++f) {
            float2 *ph = reinterpret_cast<float2 *>(q.phasor) + ((long long)f * q.ncomp + ci) * bc + cell;
            float2 acc = *ph;
            acc.x += v * __ldg(csn + 2 * f);
            acc.y -= v * __ldg(csn + 2 * f + 1);
            *ph = acc;
        }
    }
}

__device__ __forceinline__ bool any_detector_plane(const FwdParams &P, int family, int k)
{
    for (int s = 0; s < P.n_det; ++s) {
        const int m = family ? (P.det[s].mask >> 3) : (P.det[s].mask & 7);
        if (m && k >= P.det[s].lo[2] && k < P.det[s].hi[2]) return true;
    }
    return false;
}

__device__ __forceinline__ float &f4at(float4 &v, int q) { return q == 0 ? v.x : (q == 1 ? v.y : (q == 2 ? v.z : v.w)); }

// ================================================================================================
__global__ void __launch_bounds__(MAX_THREADS, 1) k_fused_forward(const __grid_constant__ FwdParams P)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const Dims &G = P.G;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + P.bar_off);
    uint64_t *empty = full + P.nstages;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = *P.step;
    const int par = n & 1;

    if (threadIdx.x == 0) {
        for (int s = 0; s < P.nstages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], P.NCW); }
        fence_mbar_init();
    }
    __syncthreads();

    const int seg_lo = P.seg_begin[blockIdx.x], seg_hi = P.seg_begin[blockIdx.x + 1];

    // ============================================================================== producer warp
    if (warp == P.NCW) {
        if (lane != 0) return;
        const CUtensorMap *M = P.maps;
        int ld = 0;
        for (int sg = seg_lo; sg < seg_hi; ++sg) {
            const Segment S = P.segs[sg];
            const int x = S.i0 - 4, y = S.j0 - 1;
            const bool xs = (S.flags & (SEG_X_LO | SEG_X_HI)) != 0, ys = (S.flags & (SEG_Y_LO | SEG_Y_HI)) != 0;
            const int xhi = (S.flags & SEG_X_HI) ? 1 : 0, yhi = (S.flags & SEG_Y_HI) ? 1 : 0;
            const int xv = (xhi ? S.xbase - (G.nx - G.dpx) : S.xbase) - 4;     // x-psi box start in view coordinates
            const int yv = yhi ? y - (G.ny - G.d) : y;                          // y-psi box start in view coordinates
            for (int kk = S.k0 - 1; kk <= S.k1; ++kk, ++ld) {
                const int s = ld % P.nstages;
                mbar_wait(&empty[s], ((ld / P.nstages) & 1) ^ 1);
                uint8_t *st = smem + (size_t)s * P.stage_bytes;
                const bool prolog = kk == S.k0 - 1;
                const bool doB = kk >= S.k0 + 1;
                const bool zE = !prolog && in_zslab(G, kk), zH = doB && in_zslab(G, kk - 1);
                uint32_t bytes = 3 * P.big_bytes;
                if (!prolog) {
                    bytes += 4 * P.big_bytes;
                    if (zE) bytes += 2 * P.big_bytes;
                    if (ys) bytes += 2 * P.big_bytes;
                    if (xs) bytes += 2 * P.small_bytes;
                }
                if (doB) {
                    if (P.has_mu) bytes += P.big_bytes;
                    if (zH) bytes += 2 * P.big_bytes;
                    if (ys) bytes += 2 * P.big_bytes;
                    if (xs) bytes += 2 * P.small_bytes;
                }
                mbar_expect_tx(&full[s], bytes);
                for (int c = 3; c < 6; ++c) tma_load_3d(st + P.slot_off[c], M + TM_FIELD + par * 6 + c, x, y, kk, &full[s]);
                if (!prolog) {
                    for (int c = 0; c < 3; ++c) tma_load_3d(st + P.slot_off[c], M + TM_FIELD + par * 6 + c, x, y, kk, &full[s]);
                    tma_load_3d(st + P.slot_off[SA_IE], M + TM_IE, x, y, kk, &full[s]);
                    if (zE) {
                        const int kz = zslab_index(G, kk);
                        tma_load_3d(st + P.slot_off[SA_PE_Z0], M + tm_psi(par, 0, 8), x, y, kz, &full[s]);
                        tma_load_3d(st + P.slot_off[SA_PE_Z1], M + tm_psi(par, 0, 9), x, y, kz, &full[s]);
                    }
                    if (ys) {
                        tma_load_3d(st + P.slot_off[SA_PE_Y0], M + tm_psi(par, 0, 4 + 2 * yhi), x, yv, kk, &full[s]);
                        tma_load_3d(st + P.slot_off[SA_PE_Y1], M + tm_psi(par, 0, 5 + 2 * yhi), x, yv, kk, &full[s]);
                    }
                    if (xs) {
                        tma_load_3d(st + P.slot_off[SA_PE_X0], M + tm_psi(par, 0, 0 + 2 * xhi), xv, y, kk, &full[s]);
                        tma_load_3d(st + P.slot_off[SA_PE_X1], M + tm_psi(par, 0, 1 + 2 * xhi), xv, y, kk, &full[s]);
                    }
                }
                if (doB) {
                    if (P.has_mu) tma_load_3d(st + P.slot_off[SA_IM], M + TM_IM, x, y, kk - 1, &full[s]);
                    if (zH) {
                        const int kz = zslab_index(G, kk - 1);
                        tma_load_3d(st + P.slot_off[SA_PH_Z0], M + tm_psi(par, 1, 8), x, y, kz, &full[s]);
                        tma_load_3d(st + P.slot_off[SA_PH_Z1], M + tm_psi(par, 1, 9), x, y, kz, &full[s]);
                    }
                    if (ys) {
                        tma_load_3d(st + P.slot_off[SA_PH_Y0], M + tm_psi(par, 1, 4 + 2 * yhi), x, yv, kk - 1, &full[s]);
                        tma_load_3d(st + P.slot_off[SA_PH_Y1], M + tm_psi(par, 1, 5 + 2 * yhi), x, yv, kk - 1, &full[s]);
                    }
                    if (xs) {
                        tma_load_3d(st + P.slot_off[SA_PH_X0], M + tm_psi(par, 1, 0 + 2 * xhi), xv, y, kk - 1, &full[s]);
                        tma_load_3d(st + P.slot_off[SA_PH_X1], M + tm_psi(par, 1, 1 + 2 * xhi), xv, y, kk - 1, &full[s]);
                    }
                }
            }
        }
        return;
    }

    // ============================================================================== consumer warps
    const int t = threadIdx.x;
    const bool active = t < P.NT;
    const int ty = active ? t / P.TX4 : 0;
    const int tx = active ? t - ty * P.TX4 : 0;
    const bool halo_row = ty == P.TY;
    const bool last_col = tx == P.TX4 - 1;
    const int o_own = ((1 + ty) * P.PW + 4 + 4 * tx) * 4;        // byte offset of my float4 inside a big box
    const int o_my = o_own - P.PW * 4;                           // row below (-y)
    const int o_mx = o_own - 4;                                  // cell to the left (-x)
    const int o_hc = o_own + 16;                                 // +x halo column cell (for last_col threads)
    float *ring = reinterpret_cast<float *>(smem + P.ring_off);
    const int ring_comp = (P.TY + 1) * P.RP, ring_slot = 3 * ring_comp;
    const int r_own = ty * P.RP + 4 * tx;
    float *dst = P.buf[par ^ 1];
    const PsiSet &pE = P.psiE[par ^ 1], &pH = P.psiH[par ^ 1];
    const float S = G.S;
    const long long nc = G.nc;
    const int consumer_threads = P.NCW * 32;

    int ld = 0;
    for (int sg = seg_lo; sg < seg_hi; ++sg) {
        const Segment Sg = P.segs[sg];
        const int i = Sg.i0 + 4 * tx, j = Sg.j0 + ty;
        const bool in_x = i < G.nx, in_y = j < G.ny;
        const bool own_ok = active && !halo_row && in_x && in_y;
        const bool ypml = G.d > 0 && in_y && (j < G.d || j >= G.ny - G.d);
        const bool xpml = G.d > 0 && in_x && (i < G.dpx || i >= G.nx - G.dpx);
        const int ih = i + 4;                                     // +x halo column
        const bool xpml_h = G.d > 0 && ih < G.nx && (ih < G.dpx || ih >= G.nx - G.dpx);
        const int o_x = ((1 + ty) * P.XW + (i - Sg.xbase + 4)) * 4;   // my float4 inside a narrow x-psi box
        // per-thread coefficients (constant along z)
        const float4 ikEx = in_x ? ldg4(P.T.ik[0][0] + i) : splat(1.f);
        const float4 ikHx = in_x ? ldg4(P.T.ik[1][0] + i) : splat(1.f);
        const float ikEx_h = ih < G.nx ? __ldg(P.T.ik[0][0] + ih) : 1.f;
        const float ikEy = in_y ? __ldg(P.T.ik[0][1] + j) : 1.f, ikHy = in_y ? __ldg(P.T.ik[1][1] + j) : 1.f;
        float bEy = 1.f, aEy = 0.f, bHy = 1.f, aHy = 0.f;
        if (ypml) { bEy = __ldg(P.T.b[0][1] + j); aEy = __ldg(P.T.a[0][1] + j); bHy = __ldg(P.T.b[1][1] + j); aHy = __ldg(P.T.a[1][1] + j); }
        const int sy = j < G.d ? j : j - (G.ny - 2 * G.d);
        const int sx = i < G.dpx ? i : i - (G.nx - 2 * G.dpx);
        const long long own_xy = (long long)j * G.nx + i;

        float4 hxk = splat(0.f), hyk = splat(0.f), hzk = splat(0.f);      // H(kk-1) at my cells
        float4 e1x = splat(0.f), e1y = splat(0.f), e1z = splat(0.f);      // E'(kk-1) at my cells
        float hxk_h = 0.f;                                                // H_x(kk-1) at the +x halo column

        for (int kk = Sg.k0 - 1; kk <= Sg.k1; ++kk, ++ld) {
            const int s = ld % P.nstages;
            mbar_wait(&full[s], (ld / P.nstages) & 1);
            const uint8_t *st = smem + (size_t)s * P.stage_bytes;
            const bool prolog = kk == Sg.k0 - 1;
            if (prolog) {
                if (active) {
                    hxk = lds4(st + P.slot_off[SA_HX], o_own);
                    hyk = lds4(st + P.slot_off[SA_HY], o_own);
                    hzk = lds4(st + P.slot_off[SA_HZ], o_own);
                    hxk_h = lds1(st + P.slot_off[SA_HX], o_hc);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[s]);
                continue;
            }
            const bool storeE = kk < Sg.k1;
            const bool doB = kk >= Sg.k0 + 1;
            float4 hx = splat(0.f), hy = hx, hz = hx, e2x = hx, e2y = hx, e2z = hx;
            if (active) {
                // ---------------------------------------------------------------- phase A: E'(kk)
                const bool zE = in_zslab(G, kk);
                const int kc = kk < G.nz ? kk : G.nz;                 // tables are padded past N
                const float ikEz = __ldg(P.T.ik[0][2] + kc);
                float bEz = 1.f, aEz = 0.f;
                if (zE) { bEz = __ldg(P.T.b[0][2] + kk); aEz = __ldg(P.T.a[0][2] + kk); }
                const float4 ex = lds4(st + P.slot_off[SA_EX], o_own), ey = lds4(st + P.slot_off[SA_EY], o_own),
                             ez = lds4(st + P.slot_off[SA_EZ], o_own);
                const float4 sie = S * lds4(st + P.slot_off[SA_IE], o_own);
                hx = lds4(st + P.slot_off[SA_HX], o_own);
                hy = lds4(st + P.slot_off[SA_HY], o_own);
                hz = lds4(st + P.slot_off[SA_HZ], o_own);
                const float4 hx_my = lds4(st + P.slot_off[SA_HX], o_my), hz_my = lds4(st + P.slot_off[SA_HZ], o_my);
                const float hy_mx = lds1(st + P.slot_off[SA_HY], o_mx), hz_mx = lds1(st + P.slot_off[SA_HZ], o_mx);
                const float4 dHz_dy = hz - hz_my, dHx_dy = hx - hx_my;
                const float4 dHy_dz = hy - hyk, dHx_dz = hx - hxk;
                const float4 dHy_dx = dminus_x(hy, hy_mx), dHz_dx = dminus_x(hz, hz_mx);
                const bool wr = own_ok && storeE;                      // I own these cells: write E' and psi_E
                const long long zoff = (long long)kk * G.ny * G.nx;
                float4 bEx = splat(1.f), aEx = splat(0.f);
                if (xpml) { bEx = ldg4(P.T.b[0][0] + i); aEx = ldg4(P.T.a[0][0] + i); }
                const long long ix = ((long long)kk * G.ny + j) * (2 * G.dpx) + sx;      // x-slab psi index
                const long long iy = ((long long)kk * (2 * G.d) + sy) * G.nx + i;        // y-slab psi index
                const long long iz = zE ? ((long long)zslab_index(G, kk) * G.ny + j) * G.nx + i : 0;

                // E'_x: a = y (psiE_x0), b = z (psiE_x1)
                float4 tE = ikEy * dHz_dy - ikEz * dHy_dz;
                if (ypml) { const float4 p = bEy * lds4(st + P.slot_off[SA_PE_Y0], o_own) + aEy * dHz_dy; tE = tE + p; if (wr) stg4(pE.p[0][0] + iy, p); }
                if (zE)   { const float4 p = bEz * lds4(st + P.slot_off[SA_PE_Z1], o_own) + aEz * dHy_dz; tE = tE - p; if (wr) stg4(pE.p[0][1] + iz, p); }
                e2x = ex + sie * tE;
                // E'_y: a = z (psiE_y0), b = x (psiE_y1)
                tE = ikEz * dHx_dz - ikEx * dHz_dx;
                if (zE)   { const float4 p = bEz * lds4(st + P.slot_off[SA_PE_Z0], o_own) + aEz * dHx_dz; tE = tE + p; if (wr) stg4(pE.p[1][0] + iz, p); }
                if (xpml) { const float4 p = bEx * lds4(st + P.slot_off[SA_PE_X1], o_x) + aEx * dHz_dx; tE = tE - p; if (wr) stg4(pE.p[1][1] + ix, p); }
                e2y = ey + sie * tE;
                // E'_z: a = x (psiE_z0), b = y (psiE_z1)
                tE = ikEx * dHy_dx - ikEy * dHx_dy;
                if (xpml) { const float4 p = bEx * lds4(st + P.slot_off[SA_PE_X0], o_x) + aEx * dHy_dx; tE = tE + p; if (wr) stg4(pE.p[2][0] + ix, p); }
                if (ypml) { const float4 p = bEy * lds4(st + P.slot_off[SA_PE_Y1], o_own) + aEy * dHx_dy; tE = tE - p; if (wr) stg4(pE.p[2][1] + iy, p); }
                e2z = ez + sie * tE;

                const bool src_plane = P.n_src && any_source_plane(P, 0, kk);
                if (src_plane) {
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        f4at(e2x, q) += source_at(P, n, 0, i + q, j, kk);
                        f4at(e2y, q) += source_at(P, n, 1, i + q, j, kk);
                        f4at(e2z, q) += source_at(P, n, 2, i + q, j, kk);
                    }
                }
                float *rg = ring + (kk & 1) * ring_slot + r_own;
                *reinterpret_cast<float4 *>(rg) = e2x;
                *reinterpret_cast<float4 *>(rg + ring_comp) = e2y;
                *reinterpret_cast<float4 *>(rg + 2 * ring_comp) = e2z;
                if (wr) {
                    stg4(dst + 0 * nc + zoff + own_xy, e2x);
                    stg4(dst + 1 * nc + zoff + own_xy, e2y);
                    stg4(dst + 2 * nc + zoff + own_xy, e2z);
                    if (P.n_det && any_detector_plane(P, 0, kk)) {
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            detect_cell(P, n, 0, f4at(e2x, q), i + q, j, kk);
                            detect_cell(P, n, 1, f4at(e2y, q), i + q, j, kk);
                            detect_cell(P, n, 2, f4at(e2z, q), i + q, j, kk);
                        }
                    }
                }
                // +x halo column: E'_y and E'_z at (i+4, j, kk), recomputed for my row (not stored)
                if (last_col) {
                    const float hx_h = lds1(st + P.slot_off[SA_HX], o_hc);
                    if (!halo_row) {
                        const float hy_h = lds1(st + P.slot_off[SA_HY], o_hc), hz_h = lds1(st + P.slot_off[SA_HZ], o_hc);
                        const float hx_h_my = lds1(st + P.slot_off[SA_HX], o_hc - P.PW * 4);
                        const float sie_h = S * lds1(st + P.slot_off[SA_IE], o_hc);
                        const float dHx_dz_h = hx_h - hxk_h, dHz_dx_h = hz_h - hz.w, dHy_dx_h = hy_h - hy.w, dHx_dy_h = hx_h - hx_h_my;
                        float bx_h = 1.f, ax_h = 0.f;
                        if (xpml_h) { bx_h = __ldg(P.T.b[0][0] + ih); ax_h = __ldg(P.T.a[0][0] + ih); }
                        float tH = ikEz * dHx_dz_h - ikEx_h * dHz_dx_h;
                        if (zE)     tH += bEz * lds1(st + P.slot_off[SA_PE_Z0], o_hc) + aEz * dHx_dz_h;
                        if (xpml_h) tH -= bx_h * lds1(st + P.slot_off[SA_PE_X1], o_x + 16) + ax_h * dHz_dx_h;
                        float ey_h = lds1(st + P.slot_off[SA_EY], o_hc) + sie_h * tH;
                        tH = ikEx_h * dHy_dx_h - ikEy * dHx_dy_h;
                        if (xpml_h) tH += bx_h * lds1(st + P.slot_off[SA_PE_X0], o_x + 16) + ax_h * dHy_dx_h;
                        if (ypml)   tH -= bEy * lds1(st + P.slot_off[SA_PE_Y1], o_hc) + aEy * dHx_dy_h;
                        float ez_h = lds1(st + P.slot_off[SA_EZ], o_hc) + sie_h * tH;
                        if (src_plane) { ey_h += source_at(P, n, 1, ih, j, kk); ez_h += source_at(P, n, 2, ih, j, kk); }
                        rg[ring_comp + 4] = ey_h;
                        rg[2 * ring_comp + 4] = ez_h;
                    }
                    hxk_h = hx_h;
                }
            }
            // ---------------------------------------------------------------- phase B: H'(kk-1)
            if (active && doB && !halo_row) {
                const int km = kk - 1;
                const bool zH = in_zslab(G, km);
                const float ikHz = __ldg(P.T.ik[1][2] + km);
                float bHz = 1.f, aHz = 0.f;
                if (zH) { bHz = __ldg(P.T.b[1][2] + km); aHz = __ldg(P.T.a[1][2] + km); }
                const float4 sim = P.has_mu ? S * lds4(st + P.slot_off[SA_IM], o_own) : splat(S);
                const float *rg = ring + (km & 1) * ring_slot + r_own;
                const float4 ex_py = *reinterpret_cast<const float4 *>(rg + P.RP);
                const float4 ez_py = *reinterpret_cast<const float4 *>(rg + 2 * ring_comp + P.RP);
                const float ey_px = rg[ring_comp + 4], ez_px = rg[2 * ring_comp + 4];
                const float4 dEz_dy = ez_py - e1z, dEx_dy = ex_py - e1x;
                const float4 dEy_dz = e2y - e1y, dEx_dz = e2x - e1x;
                const float4 dEz_dx = dplus_x(e1z, ez_px), dEy_dx = dplus_x(e1y, ey_px);
                float4 bHx = splat(1.f), aHx = splat(0.f);
                if (xpml) { bHx = ldg4(P.T.b[1][0] + i); aHx = ldg4(P.T.a[1][0] + i); }
                const long long zoff = (long long)km * G.ny * G.nx;
                const long long ix = ((long long)km * G.ny + j) * (2 * G.dpx) + sx;
                const long long iy = ((long long)km * (2 * G.d) + sy) * G.nx + i;
                const long long iz = zH ? ((long long)zslab_index(G, km) * G.ny + j) * G.nx + i : 0;
                const bool wr = own_ok;
                // H'_x: a = y (psiH_x0), b = z (psiH_x1)
                float4 tH = ikHy * dEz_dy - ikHz * dEy_dz;
                if (ypml) { const float4 p = bHy * lds4(st + P.slot_off[SA_PH_Y0], o_own) + aHy * dEz_dy; tH = tH + p; if (wr) stg4(pH.p[0][0] + iy, p); }
                if (zH)   { const float4 p = bHz * lds4(st + P.slot_off[SA_PH_Z1], o_own) + aHz * dEy_dz; tH = tH - p; if (wr) stg4(pH.p[0][1] + iz, p); }
                float4 h2x = hxk - sim * tH;
                // H'_y: a = z (psiH_y0), b = x (psiH_y1)
                tH = ikHz * dEx_dz - ikHx * dEz_dx;
                if (zH)   { const float4 p = bHz * lds4(st + P.slot_off[SA_PH_Z0], o_own) + aHz * dEx_dz; tH = tH + p; if (wr) stg4(pH.p[1][0] + iz, p); }
                if (xpml) { const float4 p = bHx * lds4(st + P.slot_off[SA_PH_X1], o_x) + aHx * dEz_dx; tH = tH - p; if (wr) stg4(pH.p[1][1] + ix, p); }
                float4 h2y = hyk - sim * tH;
                // H'_z: a = x (psiH_z0), b = y (psiH_z1)
                tH = ikHx * dEy_dx - ikHy * dEx_dy;
                if (xpml) { const float4 p = bHx * lds4(st + P.slot_off[SA_PH_X0], o_x) + aHx * dEy_dx; tH = tH + p; if (wr) stg4(pH.p[2][0] + ix, p); }
                if (ypml) { const float4 p = bHy * lds4(st + P.slot_off[SA_PH_Y1], o_own) + aHy * dEx_dy; tH = tH - p; if (wr) stg4(pH.p[2][1] + iy, p); }
                float4 h2z = hzk - sim * tH;
                if (wr) {
                    if (P.n_src && any_source_plane(P, 1, km)) {
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            f4at(h2x, q) += source_at(P, n, 3, i + q, j, km);
                            f4at(h2y, q) += source_at(P, n, 4, i + q, j, km);
                            f4at(h2z, q) += source_at(P, n, 5, i + q, j, km);
                        }
                    }
                    stg4(dst + 3 * nc + zoff + own_xy, h2x);
                    stg4(dst + 4 * nc + zoff + own_xy, h2y);
                    stg4(dst + 5 * nc + zoff + own_xy, h2z);
                    if (P.n_det && any_detector_plane(P, 1, km)) {
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            detect_cell(P, n, 3, f4at(h2x, q), i + q, j, km);
                            detect_cell(P, n, 4, f4at(h2y, q), i + q, j, km);
                            detect_cell(P, n, 5, f4at(h2z, q), i + q, j, km);
                        }
                    }
                }
            }
            e1x = e2x; e1y = e2y; e1z = e2z;
            hxk = hx; hyk = hy; hzk = hz;
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
            named_bar_sync(1, consumer_threads);      // ring slot (kk-1)&1 may be overwritten next iteration
        }
    }
}

// ================================================================================================
// host side
// ================================================================================================
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode()
{
    static EncodeTiledFn fn = nullptr;
    if (fn) return fn;
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || !p) {
        (void)cudaGetLastError();
        return nullptr;
    }
    fn = (EncodeTiledFn)p;
    return fn;
}

// 3-D fp32 tensor (dx fastest) with row pitch / plane pitch in floats
bool encode3d(CUtensorMap *out, const float *base, long long dx, long long dy, long long dz, long long pitch_y,
              long long pitch_z, int bx, int by)
{
    EncodeTiledFn fn = get_encode();
    if (!fn) return false;
    cuuint64_t dims[3] = { (cuuint64_t)dx, (cuuint64_t)dy, (cuuint64_t)dz };
    cuuint64_t strides[2] = { (cuuint64_t)pitch_y * 4, (cuuint64_t)pitch_z * 4 };
    cuuint32_t box[3] = { (cuuint32_t)bx, (cuuint32_t)by, 1 };
    cuuint32_t es[3] = { 1, 1, 1 };
    return fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int align_up(int v, int a) { return (v + a - 1) / a * a; }

}  // namespace

struct FusedState {
    int TX = 0, TY = 0, nst = 0, n_cta = 0, threads = 0;
    size_t smem = 0;
    FwdParams fp{};
    float *bufB = nullptr;                 // second field buffer
    CUtensorMap *d_maps = nullptr;
    CUtensorMap *h_maps = nullptr;         // pinned staging
    cudaEvent_t maps_done = nullptr;
    Segment *d_segs = nullptr;
    int *d_seg_begin = nullptr;
    const float *maps_fields = nullptr, *maps_ie = nullptr, *maps_im = nullptr;   // pointers the maps were built for
};

namespace {

struct TileChoice { int TX, TY, nst; size_t smem; int stage_bytes, big, small, XW; double score; };

// smem layout for a candidate tile; returns false if it does not fit
bool layout(const Dims &G, bool has_mu, int TX, int TY, int nst, int smem_cap, TileChoice &c)
{
    const int PW = TX + 8, ROWS = TY + 2;
    c.TX = TX; c.TY = TY; c.nst = nst;
    c.big = align_up(PW * ROWS * 4, 128);
    c.XW = G.dpx + 8;
    c.small = align_up(c.XW * ROWS * 4, 128);
    int n_big = 7 + (has_mu ? 1 : 0) + (G.d > 0 ? 8 : 0);
    int n_small = G.d > 0 ? 4 : 0;
    c.stage_bytes = align_up(n_big * c.big + n_small * c.small, 1024);
    const int RP = TX + 4;
    const size_t ring = (size_t)2 * 3 * (TY + 1) * RP * 4;
    c.smem = (size_t)nst * c.stage_bytes + align_up((int)ring, 128) + 128;
    return c.smem <= (size_t)smem_cap;
}

}  // namespace

int fused_setup(fdtd_grid *g)
{
    const Dims &G = g->G;
    if (g->desc.path == FDTD_PATH_GENERIC) { g->fused_why_not = "generic path requested"; return FDTD_OK; }
    if (G.periodic) { g->fused_why_not = "periodic grids use the generic kernels"; return FDTD_OK; }
    if (G.nx % 4) { g->fused_why_not = "nx is not a multiple of 4"; return FDTD_OK; }
    if (G.d > 0 && (G.dpx % 4)) { g->fused_why_not = "x-slab psi storage is not float4 aligned (nx < 2*roundup4(d))"; return FDTD_OK; }
    if (!get_encode()) { g->fused_why_not = "cuTensorMapEncodeTiled is not available"; return FDTD_OK; }
    int dev = 0, smem_cap = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&smem_cap, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        g->fused_why_not = "cannot query the device";
        return FDTD_OK;
    }
    const bool has_mu = true;   // the stage layout always reserves the inv_mu slot (8 big arrays); cheap and keeps one kernel

    // ---- tile choice: maximise useful work per byte staged, subject to shared memory and slab rules -------------
    const int tx_max = G.d > 0 ? std::min(248, G.nx - 2 * G.dpx - 4) / 4 * 4 : std::min(248, G.nx);
    const int ty_max = G.d > 0 ? std::min(64, G.ny - 2 * G.d - 2) : std::min(64, G.ny);
    TileChoice best{}; best.score = -1;
    int fTX = 0, fTY = 0, fNST = 0;
    if (const char *e = getenv("FDTD_TILE")) sscanf(e, "%d,%d,%d", &fTX, &fTY, &fNST);
    for (int TX = 4; TX <= tx_max; TX += 4)
        for (int TY = 1; TY <= ty_max; ++TY) {
            if (fTX && (TX != fTX || TY != fTY)) continue;
            const int NT = (TX / 4) * (TY + 1);
            if (align_up(NT, 32) + 32 > MAX_THREADS) continue;
            for (int nst = 4; nst >= 2; --nst) {
                if (fNST && nst != fNST) continue;
                TileChoice c{};
                if (!layout(G, has_mu, TX, TY, nst, smem_cap, c)) continue;
                const double eff_x = (double)G.nx / (((G.nx + TX - 1) / TX) * TX);
                const double eff_y = (double)G.ny / (((G.ny + TY - 1) / TY) * TY);
                const double halo = (double)(TX + 8) * (TY + 2) / ((double)TX * TY);
                const double thr = (double)NT / (align_up(NT, 32));
                // bytes through L2 per useful cell (7 loads * halo + 6 stores), wasted thread slots, sync depth bonus
                c.score = eff_x * eff_y * thr / (28.0 * halo + 24.0) * (nst >= 3 ? 1.0 : 0.93) * (NT >= 192 ? 1.0 : 0.85);
                if (c.score > best.score) best = c;
                break;
            }
        }
    if (best.score < 0) { g->fused_why_not = "no tile fits (grid too small for its PML)"; return FDTD_OK; }

    FusedState *F = new FusedState();
    g->fused = F;
    F->TX = best.TX; F->TY = best.TY; F->nst = best.nst; F->smem = best.smem;
    int rc;
    if ((rc = g->alloc((void **)&F->bufB, (size_t)G.nc * 6 * sizeof(float)))) return rc;
    if ((rc = g->alloc_psi(g->psiE[1])) || (rc = g->alloc_psi(g->psiH[1]))) return rc;
    if ((rc = g->alloc((void **)&F->d_maps, sizeof(CUtensorMap) * TM_COUNT))) return rc;
    if (cudaMallocHost((void **)&F->h_maps, sizeof(CUtensorMap) * TM_COUNT) != cudaSuccess ||
        cudaEventCreateWithFlags(&F->maps_done, cudaEventDisableTiming) != cudaSuccess) {
        (void)cudaGetLastError();
        return fdtd_fail(FDTD_ENOMEM, "pinned tensor-map staging allocation failed");
    }

    // ---- segments: flatten (tile, plane) and cut into n_cta equal-cost runs ------------------------------------
    const int ntx = (G.nx + F->TX - 1) / F->TX, nty = (G.ny + F->TY - 1) / F->TY;
    const long long total = (long long)ntx * nty * G.nz;
    int n_cta = (int)std::min<long long>(n_sm, std::max<long long>(1, total / 6));
    if (const char *e = getenv("FDTD_NCTA")) n_cta = std::max(1, atoi(e));
    std::vector<Segment> segs;
    std::vector<int> seg_begin(n_cta + 1, 0);
    {
        long long done = 0;
        int cta = 0;
        for (int txi = 0; txi < ntx; ++txi)
            for (int tyi = 0; tyi < nty; ++tyi) {
                int k = 0;
                while (k < G.nz) {
                    // planes left for the current CTA
                    long long quota_end = (total * (cta + 1)) / n_cta;
                    long long room = quota_end - done;
                    if (room <= 0) { ++cta; seg_begin[cta] = (int)segs.size(); continue; }
                    int len = (int)std::min<long long>(room, G.nz - k);
                    Segment s{};
                    s.i0 = txi * F->TX; s.j0 = tyi * F->TY; s.k0 = k; s.k1 = k + len;
                    if (G.d > 0) {
                        if (s.i0 < G.dpx) s.flags |= SEG_X_LO;
                        if (s.i0 + F->TX >= G.nx - G.dpx) s.flags |= SEG_X_HI;
                        if (s.j0 < G.d) s.flags |= SEG_Y_LO;
                        if (s.j0 + F->TY >= G.ny - G.d) s.flags |= SEG_Y_HI;
                    }
                    s.xbase = (s.flags & SEG_X_HI) ? std::max(s.i0, G.nx - G.dpx) : s.i0;
                    segs.push_back(s);
                    k += len; done += len;
                }
            }
        for (int c = cta + 1; c <= n_cta; ++c) seg_begin[c] = (int)segs.size();
    }
    for (const Segment &s : segs)
        if (((s.flags & SEG_X_LO) && (s.flags & SEG_X_HI)) || ((s.flags & SEG_Y_LO) && (s.flags & SEG_Y_HI))) {
            g->fused_why_not = "a tile touches both slabs of an axis";
            return FDTD_OK;
        }
    F->n_cta = n_cta;
    if ((rc = g->alloc((void **)&F->d_segs, segs.size() * sizeof(Segment)))) return rc;
    if ((rc = g->alloc((void **)&F->d_seg_begin, seg_begin.size() * sizeof(int)))) return rc;
    if (cudaMemcpy(F->d_segs, segs.data(), segs.size() * sizeof(Segment), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(F->d_seg_begin, seg_begin.data(), seg_begin.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
        (void)cudaGetLastError();
        return fdtd_fail(FDTD_ECUDA, "upload of the segment table failed");
    }

    // ---- kernel parameters that do not depend on the call -----------------------------------------------------------
    FwdParams &P = F->fp;
    P.G = G; P.T = g->T; P.maps = F->d_maps; P.segs = F->d_segs; P.seg_begin = F->d_seg_begin;
    P.step = g->d_step;
    P.TX = F->TX; P.TY = F->TY; P.TX4 = F->TX / 4; P.NT = P.TX4 * (F->TY + 1); P.NCW = (P.NT + 31) / 32;
    P.PW = F->TX + 8; P.ROWS = F->TY + 2; P.XW = best.XW;
    P.big_bytes = P.PW * P.ROWS * 4; P.small_bytes = P.XW * P.ROWS * 4;
    P.stage_bytes = best.stage_bytes; P.nstages = F->nst;
    {
        int off = 0;
        const int bigs[] = { SA_EX, SA_EY, SA_EZ, SA_HX, SA_HY, SA_HZ, SA_IE, SA_IM, SA_PE_Y0, SA_PE_Y1, SA_PE_Z0, SA_PE_Z1,
                             SA_PH_Y0, SA_PH_Y1, SA_PH_Z0, SA_PH_Z1 };
        const int n_big = G.d > 0 ? 16 : 8;
        for (int q = 0; q < SA_COUNT; ++q) P.slot_off[q] = 0;
        for (int q = 0; q < n_big; ++q) { P.slot_off[bigs[q]] = off; off += best.big; }
        if (G.d > 0)
            for (int q = SA_PE_X0; q <= SA_PH_X1; ++q) { P.slot_off[q] = off; off += best.small; }
    }
    P.RP = F->TX + 4;
    P.ring_off = F->nst * best.stage_bytes;
    P.bar_off = P.ring_off + align_up(2 * 3 * (F->TY + 1) * P.RP * 4, 128);
    F->threads = (P.NCW + 1) * 32;
    if (cudaFuncSetAttribute(k_fused_forward, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F->smem) != cudaSuccess) {
        (void)cudaGetLastError();
        g->fused_why_not = "cannot reserve shared memory";
        return FDTD_OK;
    }
    g->path = FDTD_PATH_FUSED;
    g->tile_x = F->TX; g->tile_y = F->TY; g->tile_z = (int)(total / n_cta / std::max(1, ntx * nty / std::max(1, ntx * nty)));
    g->tile_z = (int)std::min<long long>(G.nz, total / n_cta);
    return FDTD_OK;
}

void fused_teardown(fdtd_grid *g)
{
    if (g->fused) {
        if (g->fused->h_maps) cudaFreeHost(g->fused->h_maps);
        if (g->fused->maps_done) cudaEventDestroy(g->fused->maps_done);
    }
    delete g->fused;
    g->fused = nullptr;
}

namespace {

// (re)builds the tensor maps when the caller's pointers changed
int build_maps(fdtd_grid *g, float *fields, const float *ie, const float *im, cudaStream_t st)
{
    FusedState *F = g->fused;
    const Dims &G = g->G;
    if (F->maps_fields == fields && F->maps_ie == ie && F->maps_im == im) return FDTD_OK;
    const int PW = F->TX + 8, ROWS = F->TY + 2, XW = F->fp.XW;
    if (cudaEventSynchronize(F->maps_done) != cudaSuccess) { (void)cudaGetLastError(); }   // earlier upload finished
    bool ok = true;
    float *bufs[2] = { fields, F->bufB };
    for (int set = 0; set < 2; ++set)
        for (int c = 0; c < 6; ++c)
            ok &= encode3d(&F->h_maps[TM_FIELD + set * 6 + c], bufs[set] + (long long)c * G.nc, G.nx, G.ny, G.nz, G.nx,
                           (long long)G.nx * G.ny, PW, ROWS);
    ok &= encode3d(&F->h_maps[TM_IE], ie, G.nx, G.ny, G.nz, G.nx, (long long)G.nx * G.ny, PW, ROWS);
    ok &= encode3d(&F->h_maps[TM_IM], im ? im : ie, G.nx, G.ny, G.nz, G.nx, (long long)G.nx * G.ny, PW, ROWS);
    if (G.d > 0) {
        for (int set = 0; set < 2; ++set)
            for (int fam = 0; fam < 2; ++fam) {
                const PsiSet &ps = fam ? g->psiH[set] : g->psiE[set];
                // x axis arrays: (c=z,s=0) and (c=y,s=1); layout [nz][ny][2*dpx]
                const float *xa[2] = { ps.p[2][0], ps.p[1][1] };
                for (int q = 0; q < 2; ++q)
                    for (int view = 0; view < 2; ++view)
                        ok &= encode3d(&F->h_maps[tm_psi(set, fam, q + 2 * view)], xa[q] + view * G.dpx, G.dpx, G.ny, G.nz,
                                       2 * G.dpx, (long long)2 * G.dpx * G.ny, XW, ROWS);
                // y axis arrays: (c=x,s=0) and (c=z,s=1); layout [nz][2*d][nx]
                const float *ya[2] = { ps.p[0][0], ps.p[2][1] };
                for (int q = 0; q < 2; ++q)
                    for (int view = 0; view < 2; ++view)
                        ok &= encode3d(&F->h_maps[tm_psi(set, fam, 4 + q + 2 * view)], ya[q] + (long long)view * G.d * G.nx, G.nx,
                                       G.d, G.nz, G.nx, (long long)2 * G.d * G.nx, PW, ROWS);
                // z axis arrays: (c=y,s=0) and (c=x,s=1); layout [2*d][ny][nx]
                const float *za[2] = { ps.p[1][0], ps.p[0][1] };
                for (int q = 0; q < 2; ++q)
                    ok &= encode3d(&F->h_maps[tm_psi(set, fam, 8 + q)], za[q], G.nx, G.ny, 2 * G.d, G.nx, (long long)G.nx * G.ny, PW, ROWS);
            }
    }
    if (!ok) return fdtd_fail(FDTD_ECUDA, "cuTensorMapEncodeTiled failed");
    // the previous maps may still be in use by kernels of an earlier call on another stream: the copy is stream ordered
    // on `st`, and callers that switch streams between calls must synchronise them (documented in DESIGN.md)
    cudaError_t e = cudaMemcpyAsync(F->d_maps, F->h_maps, sizeof(CUtensorMap) * TM_COUNT, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaEventRecord(F->maps_done, st);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, std::string("tensor map upload: ") + cudaGetErrorString(e)); }
    F->maps_fields = fields; F->maps_ie = ie; F->maps_im = im;
    return FDTD_OK;
}

}  // namespace

// run_steps lives in fdtd_api.cu; re-declared here through a small trampoline
int fdtd_run_steps_fwd(fdtd_grid *g, const std::string &key, int n_steps, int launches_per_step, cudaStream_t st,
                       void (*enqueue)(void *, cudaStream_t), void *ctx);

namespace {
struct FwdCtx {
    fdtd_grid *g; FwdParams P; bool recording; float *A; float *B;
};
void enqueue_fwd(void *vctx, cudaStream_t cs)
{
    FwdCtx *c = (FwdCtx *)vctx;
    fdtd_grid *g = c->g;
    FusedState *F = g->fused;
    { ProfScope p(g, fdtd_grid::PC_FUSED_FWD, cs);
      k_fused_forward<<<F->n_cta, F->threads, F->smem, cs>>>(c->P); }
    if (c->recording) {
        // step n read buffer n&1 (pre-step H) and wrote buffer (n+1)&1 (E'); the record kernel picks them by parity
        ProfScope p(g, fdtd_grid::PC_RECORD, cs);
        launch_record_pp(g->G, g->R, c->A, c->B, g->rec, g->d_step, cs);
    }
    { ProfScope p(g, fdtd_grid::PC_OTHER, cs); launch_advance(g->d_step, 1, cs); }
}
}  // namespace

int fused_forward(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                  const std::vector<SourceDev> &S, const std::vector<DetectorDev> &D, int total_freq, int n_steps,
                  bool recording, cudaStream_t st)
{
    FusedState *F = g->fused;
    if ((int)S.size() > MAX_SRC || (int)D.size() > MAX_DET)
        return fdtd_fail(FDTD_EINVAL, "the fused path takes at most 4 sources and 4 detectors (use FDTD_PATH_GENERIC)");
    int rc = build_maps(g, fields, inv_eps, inv_mu, st);
    if (rc) return rc;
    for (int q = 0; q < 2; ++q)
        if ((rc = g->zero_psi(g->psiE[q], st)) || (rc = g->zero_psi(g->psiH[q], st))) return rc;
    FwdCtx ctx{ g, F->fp, recording, fields, F->bufB };
    FwdParams &P = ctx.P;
    P.buf[0] = fields; P.buf[1] = F->bufB;
    for (int q = 0; q < 2; ++q) { P.psiE[q] = g->psiE[q]; P.psiH[q] = g->psiH[q]; }
    P.has_mu = inv_mu ? 1 : 0;
    P.n_src = (int)S.size(); P.n_det = (int)D.size(); P.total_freq = total_freq;
    for (size_t q = 0; q < S.size(); ++q) P.src[q] = S[q];
    for (size_t q = 0; q < D.size(); ++q) P.det[q] = D[q];
    P.cs = g->d_cs;
    std::string key("ff");
    key.append((const char *)&P, sizeof(P));
    key.push_back(recording ? 1 : 0);
    rc = fdtd_run_steps_fwd(g, key, n_steps, 2 + (recording ? 1 : 0), st, enqueue_fwd, &ctx);
    if (rc) return rc;
    if (n_steps & 1) {
        cudaError_t e = cudaMemcpyAsync(fields, F->bufB, (size_t)g->G.nc * 6 * sizeof(float), cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, cudaGetErrorString(e)); }
    }
    return FDTD_OK;
}

int fused_backward(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                   const std::vector<SourceDev> &S, const std::vector<DetectorDev> &D, int total_freq, int n_steps,
                   float *dL_dinv_eps, cudaStream_t st)
{
    (void)g; (void)fields; (void)inv_eps; (void)inv_mu; (void)S; (void)D; (void)total_freq; (void)n_steps; (void)dL_dinv_eps; (void)st;
    return fdtd_fail(FDTD_ESTATE, "fused backward: not reached (the API falls back to the generic reverse kernels)");
}
