// kernels_fused.cu -- fused forward step: E update + H update (+ CPML psi, sources, detectors) in ONE
// pass over the grid (rows F1-F7 of DESIGN.md; Eq. 1-2).
//
// Design:
//   * ping-pong: step n reads buffer n&1 and writes buffer (n+1)&1, so tiles are independent;
//   * the xy plane is cut into TX x TY tiles, a tile's z column into segments; a persistent CTA
//     (one per SM) marches its segments plane by plane (2.5-D blocking);
//   * one producer thread streams each plane's boxes (6 fields, inv_eps, psi slabs) global->shared with
//     TMA (cp.async.bulk.tensor; zero fill outside the grid IS the zero-pad wall convention) into a ring
//     of equally sized slots; a plane takes as many slots as it has arrays (7 in the interior, up to 18 in
//     a CPML corner), so interior planes are prefetched ~5 deep; mbarrier full/empty per plane;
//   * consumer threads own a float4 of cells; plane kk: phase A computes E'(kk) on the tile plus a +y halo
//     row and a +x halo column (recomputed, not exchanged), phase B computes H'(kk-1) from E'(kk-1)
//     (registers + a shared E' ring) and E'(kk);
//   * the update is written as  base curl  +  per-axis CPML corrections  (ik-1)*d + psi  that only run
//     on planes / warps that touch a slab;
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
constexpr int NBAR = 16;                // plane-loads in flight (mbarrier ring)

struct FwdParams {
    Dims G;
    Tables T;
    const CUtensorMap *maps;
    const Segment *segs;           // [n_rot][...]
    const int *seg_begin;          // [n_rot][n_cta + 1]
    int n_rot, seg_stride, n_cta;
    float *buf[2];                 // ping-pong field buffers, [6][nc] each
    PsiSet psiE[2], psiH[2];
    const int *step;
    int nslots;                    // slots in the shared-memory ring
    int XW, small_bytes;           // narrow x-psi box: width (floats) and exact byte size (TMA transaction bytes)
    int small_off, xslots;         // a pair of narrow boxes sits at offsets 0 / small_off of `xslots` consecutive slots
    int has_mu;
    int n_src, n_det, total_freq;
    SourceDev src[MAX_SRC];
    DetectorDev det[MAX_DET];
    const float *cs;
};

template <int TX4_, int TY_>
struct Cfg {
    static constexpr int TX4 = TX4_, TY = TY_, TX = 4 * TX4_;
    static constexpr int PW = TX + 8, ROWS = TY + 2;
    static constexpr int BOX_BYTES = PW * ROWS * 4;                    // TMA transaction bytes of a big box
    static constexpr int SLOT = (BOX_BYTES + 127) / 128 * 128;          // slot pitch
    static constexpr int RP = TX + 4;                                   // E' ring row pitch (floats)
    static constexpr int RING_COMP = (TY + 1) * RP, RING_SLOT = 3 * RING_COMP;
    static constexpr int RING_BYTES = (2 * RING_SLOT * 4 + 127) / 128 * 128;
    static constexpr int NT = TX4 * (TY + 1);                           // float4 threads (incl. the +y halo row)
    static constexpr int NCW = (NT + TY + 31) / 32;                     // consumer warps (halo-column threads appended)
    static constexpr int THREADS = NCW * 32 + 32;
};

__device__ __forceinline__ float4 lds4(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float lds1(uint32_t addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts4(uint32_t addr, float4 v)
{
    asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void sts1(uint32_t addr, float v)
{
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ float4 ldg4(const float *p) { return __ldg(reinterpret_cast<const float4 *>(p)); }
__device__ __forceinline__ void stg4(float *p, float4 v) { *reinterpret_cast<float4 *>(p) = v; }

__device__ __forceinline__ bool in_zslab(const Dims &G, int k) { return G.d > 0 && k >= 0 && k < G.nz && (k < G.d || k >= G.nz - G.d); }
__device__ __forceinline__ int zslab_index(const Dims &G, int k) { return k < G.d ? k : k - (G.nz - 2 * G.d); }

// Which arrays a plane-load carries and where they sit (slot ordinals).  Shared by producer and consumers.
struct PlaneLayout {
    int n;                 // slots taken
    int im, pez, pey, pex, phz, phy, phx;     // ordinals (valid only when present)
};
__device__ __forceinline__ PlaneLayout plane_layout(bool prolog, bool doB, bool has_mu, bool zE, bool zH, bool ys, bool xs, int xslots)
{
    PlaneLayout L;
    int o = 3;                                  // HX, HY, HZ always
    L.im = L.pez = L.pey = L.pex = L.phz = L.phy = L.phx = 0;
    if (!prolog) {
        o = 7;                                  // + EX, EY, EZ, IE
        if (zE) { L.pez = o; o += 2; }
        if (ys) { L.pey = o; o += 2; }
        if (xs) { L.pex = o; o += xslots; }
    }
    if (doB) {
        if (has_mu) { L.im = o; o += 1; }
        if (zH) { L.phz = o; o += 2; }
        if (ys) { L.phy = o; o += 2; }
        if (xs) { L.phx = o; o += xslots; }
    }
    L.n = o;
    return L;
}

// additive source contribution to component `comp` at cell (i,j,k) during this step
__device__ __noinline__ float source_at(const FwdParams &P, int n, int comp, int i, int j, int k)
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
__device__ __noinline__ void detect_cell(const FwdParams &P, int n, int comp, float v, int i, int j, int k)
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

__device__ __forceinline__ float f4get(const float4 &v, int q) { return q == 0 ? v.x : (q == 1 ? v.y : (q == 2 ? v.z : v.w)); }
__device__ __forceinline__ void f4add(float4 &v, int q, float a) { if (q == 0) v.x += a; else if (q == 1) v.y += a; else if (q == 2) v.z += a; else v.w += a; }

// psi recursion + bracket correction for one psi array:   p = b*psi + a*d ;  t += sgn*((ik-1)*d + p)
__device__ __forceinline__ float4 psi_fix(float4 &t, float sgn, float4 b, float4 a, float4 ikm1, float4 psi, float4 d)
{
    float4 p;
    p.x = fmaf(b.x, psi.x, a.x * d.x); p.y = fmaf(b.y, psi.y, a.y * d.y);
    p.z = fmaf(b.z, psi.z, a.z * d.z); p.w = fmaf(b.w, psi.w, a.w * d.w);
    t.x += sgn * fmaf(ikm1.x, d.x, p.x); t.y += sgn * fmaf(ikm1.y, d.y, p.y);
    t.z += sgn * fmaf(ikm1.z, d.z, p.z); t.w += sgn * fmaf(ikm1.w, d.w, p.w);
    return p;
}
__device__ __forceinline__ float psi_fix1(float &t, float sgn, float b, float a, float ikm1, float psi, float d)
{
    const float p = fmaf(b, psi, a * d);
    t += sgn * fmaf(ikm1, d, p);
    return p;
}

// ================================================================================================
template <class C>
__global__ void __launch_bounds__(C::THREADS, 1) k_fused_forward(const __grid_constant__ FwdParams P)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const Dims &G = P.G;
    const uint32_t slots_base = smem_u32(smem);
    const uint32_t ring_base = slots_base + (uint32_t)P.nslots * C::SLOT;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)P.nslots * C::SLOT + C::RING_BYTES);
    uint64_t *empty = full + NBAR;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = *P.step;
    const int par = n & 1;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NBAR; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], C::NCW); }
        fence_mbar_init();
    }
    __syncthreads();

    const int rot = n % P.n_rot;
    const int *sb = P.seg_begin + rot * (P.n_cta + 1);
    const Segment *segs = P.segs + (size_t)rot * P.seg_stride;
    const int seg_lo = sb[blockIdx.x], seg_hi = sb[blockIdx.x + 1];
    const bool has_mu = P.has_mu != 0;

    // ============================================================================== producer
    if (warp == C::NCW) {
        if (lane != 0) return;
        const CUtensorMap *M = P.maps;
        int ld = 0;                 // plane-loads issued
        int head = 0;               // next free slot
        int tail_ld = 0;            // oldest plane-load not yet known to be released
        int start[NBAR];            // first slot of each in-flight plane-load
        int tail_pos = 0;
        for (int sg = seg_lo; sg < seg_hi; ++sg) {
            const Segment S = segs[sg];
            const int x = S.i0 - 4, y = S.j0 - 1;
            const bool xs = (S.flags & (SEG_X_LO | SEG_X_HI)) != 0, ys = (S.flags & (SEG_Y_LO | SEG_Y_HI)) != 0;
            const int xhi = (S.flags & SEG_X_HI) ? 1 : 0, yhi = (S.flags & SEG_Y_HI) ? 1 : 0;
            const int xv = (xhi ? S.xbase - (G.nx - G.dpx) : S.xbase) - 4;     // x-psi box start in view coordinates
            const int yv = yhi ? y - (G.ny - G.d) : y;                          // y-psi box start in view coordinates
            for (int kk = S.k0 - 1; kk <= S.k1; ++kk, ++ld) {
                const bool prolog = kk == S.k0 - 1;
                const bool doB = kk >= S.k0 + 1;
                const bool zE = !prolog && in_zslab(G, kk), zH = doB && in_zslab(G, kk - 1);
                const PlaneLayout L = plane_layout(prolog, doB, has_mu, zE, zH, ys, xs, P.xslots);
                // ---- allocate L.n contiguous slots (never wrapping inside a plane-load)
                int base = head + L.n > P.nslots ? 0 : head;
                for (;;) {
                    const int inflight = ld - tail_ld;
                    bool fits;
                    if (inflight == 0) fits = true;
                    else if (inflight >= NBAR) fits = false;
                    else if (head > tail_pos) fits = (base == head) ? true : (L.n <= tail_pos);      // free: [head,N) U [0,tail)
                    else if (head < tail_pos) fits = (base == head) && (head + L.n <= tail_pos);     // free: [head,tail)
                    else fits = false;                                                                // ring full
                    if (fits) break;
                    mbar_wait(&empty[tail_ld % NBAR], (tail_ld / NBAR) & 1);
                    ++tail_ld;
                    tail_pos = (tail_ld < ld) ? start[tail_ld % NBAR] : base;
                }
                if (ld - tail_ld == 0) tail_pos = base;
                start[ld % NBAR] = base;
                head = base + L.n;
                const int bi = ld % NBAR;
                uint64_t *fb = &full[bi];
                uint8_t *st = smem + (size_t)base * C::SLOT;
                uint32_t bytes = 3 * C::BOX_BYTES;
                if (!prolog) bytes += 4 * C::BOX_BYTES + (zE ? 2 * C::BOX_BYTES : 0) + (ys ? 2 * C::BOX_BYTES : 0) + (xs ? 2 * P.small_bytes : 0);
                if (doB) bytes += (has_mu ? C::BOX_BYTES : 0) + (zH ? 2 * C::BOX_BYTES : 0) + (ys ? 2 * C::BOX_BYTES : 0) + (xs ? 2 * P.small_bytes : 0);
                mbar_expect_tx(fb, bytes);
                for (int c = 0; c < 3; ++c) tma_load_3d(st + c * C::SLOT, M + TM_FIELD + par * 6 + 3 + c, x, y, kk, fb);
                if (!prolog) {
                    for (int c = 0; c < 3; ++c) tma_load_3d(st + (3 + c) * C::SLOT, M + TM_FIELD + par * 6 + c, x, y, kk, fb);
                    tma_load_3d(st + 6 * C::SLOT, M + TM_IE, x, y, kk, fb);
                    if (zE) {
                        const int kz = zslab_index(G, kk);
                        tma_load_3d(st + L.pez * C::SLOT, M + tm_psi(par, 0, 8), x, y, kz, fb);
                        tma_load_3d(st + (L.pez + 1) * C::SLOT, M + tm_psi(par, 0, 9), x, y, kz, fb);
                    }
                    if (ys) {
                        tma_load_3d(st + L.pey * C::SLOT, M + tm_psi(par, 0, 4 + 2 * yhi), x, yv, kk, fb);
                        tma_load_3d(st + (L.pey + 1) * C::SLOT, M + tm_psi(par, 0, 5 + 2 * yhi), x, yv, kk, fb);
                    }
                    if (xs) {
                        tma_load_3d(st + L.pex * C::SLOT, M + tm_psi(par, 0, 0 + 2 * xhi), xv, y, kk, fb);
                        tma_load_3d(st + L.pex * C::SLOT + P.small_off, M + tm_psi(par, 0, 1 + 2 * xhi), xv, y, kk, fb);
                    }
                }
                if (doB) {
                    if (has_mu) tma_load_3d(st + L.im * C::SLOT, M + TM_IM, x, y, kk - 1, fb);
                    if (zH) {
                        const int kz = zslab_index(G, kk - 1);
                        tma_load_3d(st + L.phz * C::SLOT, M + tm_psi(par, 1, 8), x, y, kz, fb);
                        tma_load_3d(st + (L.phz + 1) * C::SLOT, M + tm_psi(par, 1, 9), x, y, kz, fb);
                    }
                    if (ys) {
                        tma_load_3d(st + L.phy * C::SLOT, M + tm_psi(par, 1, 4 + 2 * yhi), x, yv, kk - 1, fb);
                        tma_load_3d(st + (L.phy + 1) * C::SLOT, M + tm_psi(par, 1, 5 + 2 * yhi), x, yv, kk - 1, fb);
                    }
                    if (xs) {
                        tma_load_3d(st + L.phx * C::SLOT, M + tm_psi(par, 1, 0 + 2 * xhi), xv, y, kk - 1, fb);
                        tma_load_3d(st + L.phx * C::SLOT + P.small_off, M + tm_psi(par, 1, 1 + 2 * xhi), xv, y, kk - 1, fb);
                    }
                }
            }
        }
        return;
    }

    // ============================================================================== consumers
    const int t = threadIdx.x;
    const bool vec = t < C::NT;                                   // float4 thread
    const bool hcol = t >= C::NT && t < C::NT + C::TY;            // +x halo column thread (one scalar cell per row)
    const int ty = vec ? t / C::TX4 : (hcol ? t - C::NT : 0);
    const int tx = vec ? t - ty * C::TX4 : C::TX4;                // halo column sits at float4 index TX4
    const bool halo_row = vec && ty == C::TY;
    // byte offset of my first cell inside a big box / a narrow box / the E' ring
    const uint32_t o_own = ((1 + ty) * C::PW + 4 + 4 * tx) * 4;
    const uint32_t r_own = (ty * C::RP + 4 * tx) * 4;
    float *dst = P.buf[par ^ 1];
    const PsiSet &pE = P.psiE[par ^ 1], &pH = P.psiH[par ^ 1];
    const float S = G.S;
    const long long nc = G.nc;
    const long long plane = (long long)G.ny * G.nx;

    int ld = 0, head = 0;
    for (int sg = seg_lo; sg < seg_hi; ++sg) {
        const Segment Sg = segs[sg];
        const int i = Sg.i0 + 4 * tx, j = Sg.j0 + ty;
        const bool in_x = i < G.nx, in_y = j < G.ny;
        const bool own_ok = vec && !halo_row && in_x && in_y;
        const bool xs = (Sg.flags & (SEG_X_LO | SEG_X_HI)) != 0, ys = (Sg.flags & (SEG_Y_LO | SEG_Y_HI)) != 0;
        const bool ypml = G.d > 0 && in_y && (j < G.d || j >= G.ny - G.d);
        const bool xpml = G.d > 0 && in_x && (i < G.dpx || i >= G.nx - G.dpx);
        const bool warp_x = xs && __any_sync(0xffffffffu, xpml), warp_y = ys && __any_sync(0xffffffffu, ypml);
        const uint32_t o_x = xpml ? ((1 + ty) * P.XW + (i - Sg.xbase + 4)) * 4 : 0;   // my cells inside a narrow x-psi box
        const int sy = j < G.d ? j : j - (G.ny - 2 * G.d);
        const int sx = i < G.dpx ? i : i - (G.nx - 2 * G.dpx);
        const long long own_xy = (long long)j * G.nx + i;

        float4 hxk = splat(0.f), hyk = hxk, hzk = hxk;      // H(kk-1) at my cells   (halo column thread: .x only)
        float4 e1x = hxk, e1y = hxk, e1z = hxk;             // E'(kk-1) at my cells

        for (int kk = Sg.k0 - 1; kk <= Sg.k1; ++kk, ++ld) {
            const bool prolog = kk == Sg.k0 - 1;
            const bool doB = kk >= Sg.k0 + 1;
            const bool zE = !prolog && in_zslab(G, kk), zH = doB && in_zslab(G, kk - 1);
            const PlaneLayout L = plane_layout(prolog, doB, has_mu, zE, zH, ys, xs, P.xslots);
            const int base = head + L.n > P.nslots ? 0 : head;
            head = base + L.n;
            const int bi = ld % NBAR;
            mbar_wait(&full[bi], (ld / NBAR) & 1);
            const uint32_t sb0 = slots_base + (uint32_t)base * C::SLOT;     // first slot of this plane-load
            const uint32_t so = sb0 + o_own;
            if (prolog) {
                if (vec) { hxk = lds4(so); hyk = lds4(so + C::SLOT); hzk = lds4(so + 2 * C::SLOT); }
                else if (hcol) hxk.x = lds1(so);
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[bi]);
                continue;
            }
            const bool storeE = kk < Sg.k1;
            const uint32_t rgA = ring_base + (kk & 1) * (C::RING_SLOT * 4) + r_own;
            const bool src_plane = P.n_src && any_source_plane(P, 0, kk);
            float4 hx = splat(0.f), hy = hx, hz = hx, e2x = hx, e2y = hx, e2z = hx;
            if (vec) {
                // ------------------------------------------------------------ phase A: E'(kk), 4 cells
                hx = lds4(so); hy = lds4(so + C::SLOT); hz = lds4(so + 2 * C::SLOT);
                const float4 hx_my = lds4(so - C::PW * 4), hz_my = lds4(so + 2 * C::SLOT - C::PW * 4);
                const float hy_mx = lds1(so + C::SLOT - 4), hz_mx = lds1(so + 2 * C::SLOT - 4);
                const float4 dHz_dy = hz - hz_my, dHx_dy = hx - hx_my;
                const float4 dHy_dz = hy - hyk, dHx_dz = hx - hxk;
                const float4 dHy_dx = dminus_x(hy, hy_mx), dHz_dx = dminus_x(hz, hz_mx);
                float4 tEx = dHz_dy - dHy_dz, tEy = dHx_dz - dHz_dx, tEz = dHy_dx - dHx_dy;
                const bool wr = own_ok && storeE;                  // I own these cells: write E' and psi_E
                if (zE) {       // z axis: psiE_y0 (d = dHx_dz, +), psiE_x1 (d = dHy_dz, -)
                    const float4 b = splat(__ldg(P.T.b[0][2] + kk)), a = splat(__ldg(P.T.a[0][2] + kk)), km = splat(__ldg(P.T.ik[0][2] + kk) - 1.f);
                    const long long iz = ((long long)zslab_index(G, kk) * G.ny + j) * G.nx + i;
                    const float4 p0 = psi_fix(tEy, 1.f, b, a, km, lds4(so + L.pez * C::SLOT), dHx_dz);
                    const float4 p1 = psi_fix(tEx, -1.f, b, a, km, lds4(so + (L.pez + 1) * C::SLOT), dHy_dz);
                    if (wr) { stg4(pE.p[1][0] + iz, p0); stg4(pE.p[0][1] + iz, p1); }
                }
                if (warp_y) {   // y axis: psiE_x0 (d = dHz_dy, +), psiE_z1 (d = dHx_dy, -)
                    float b = 1.f, a = 0.f, km = 0.f;
                    if (ypml) { b = __ldg(P.T.b[0][1] + j); a = __ldg(P.T.a[0][1] + j); km = __ldg(P.T.ik[0][1] + j) - 1.f; }
                    const long long iy = ((long long)kk * (2 * G.d) + sy) * G.nx + i;
                    const float4 p0 = psi_fix(tEx, 1.f, splat(b), splat(a), splat(km), lds4(so + L.pey * C::SLOT), dHz_dy);
                    const float4 p1 = psi_fix(tEz, -1.f, splat(b), splat(a), splat(km), lds4(so + (L.pey + 1) * C::SLOT), dHx_dy);
                    if (wr && ypml) { stg4(pE.p[0][0] + iy, p0); stg4(pE.p[2][1] + iy, p1); }
                }
                if (warp_x) {   // x axis: psiE_z0 (d = dHy_dx, +), psiE_y1 (d = dHz_dx, -)
                    float4 b = splat(1.f), a = splat(0.f), km = splat(0.f), q0 = a, q1 = a;
                    if (xpml) {
                        b = ldg4(P.T.b[0][0] + i); a = ldg4(P.T.a[0][0] + i); km = ldg4(P.T.ik[0][0] + i) - splat(1.f);
                        q0 = lds4(sb0 + L.pex * C::SLOT + o_x); q1 = lds4(sb0 + L.pex * C::SLOT + P.small_off + o_x);
                    }
                    const long long ix = ((long long)kk * G.ny + j) * (2 * G.dpx) + sx;
                    const float4 p0 = psi_fix(tEz, 1.f, b, a, km, q0, dHy_dx);
                    const float4 p1 = psi_fix(tEy, -1.f, b, a, km, q1, dHz_dx);
                    if (wr && xpml) { stg4(pE.p[2][0] + ix, p0); stg4(pE.p[1][1] + ix, p1); }
                }
                const float4 sie = S * lds4(so + 6 * C::SLOT);
                e2x = lds4(so + 3 * C::SLOT) + sie * tEx;
                e2y = lds4(so + 4 * C::SLOT) + sie * tEy;
                e2z = lds4(so + 5 * C::SLOT) + sie * tEz;
                if (src_plane) {
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        f4add(e2x, q, source_at(P, n, 0, i + q, j, kk));
                        f4add(e2y, q, source_at(P, n, 1, i + q, j, kk));
                        f4add(e2z, q, source_at(P, n, 2, i + q, j, kk));
                    }
                }
                sts4(rgA, e2x); sts4(rgA + C::RING_COMP * 4, e2y); sts4(rgA + 2 * C::RING_COMP * 4, e2z);
                if (wr) {
                    float *o = dst + (long long)kk * plane + own_xy;
                    stg4(o, e2x); stg4(o + nc, e2y); stg4(o + 2 * nc, e2z);
                    if (P.n_det && any_detector_plane(P, 0, kk)) {
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            detect_cell(P, n, 0, f4get(e2x, q), i + q, j, kk);
                            detect_cell(P, n, 1, f4get(e2y, q), i + q, j, kk);
                            detect_cell(P, n, 2, f4get(e2z, q), i + q, j, kk);
                        }
                    }
                }
            } else if (hcol) {
                // ------------------------------------------------------------ phase A, +x halo column: E'_y, E'_z of one cell
                const float hx_h = lds1(so), hy_h = lds1(so + C::SLOT), hz_h = lds1(so + 2 * C::SLOT);
                const float dHx_dz = hx_h - hxk.x, dHz_dx = hz_h - lds1(so + 2 * C::SLOT - 4), dHy_dx = hy_h - lds1(so + C::SLOT - 4);
                const float dHx_dy = hx_h - lds1(so - C::PW * 4);
                float tEy = dHx_dz - dHz_dx, tEz = dHy_dx - dHx_dy;
                if (zE) psi_fix1(tEy, 1.f, __ldg(P.T.b[0][2] + kk), __ldg(P.T.a[0][2] + kk), __ldg(P.T.ik[0][2] + kk) - 1.f,
                                 lds1(so + L.pez * C::SLOT), dHx_dz);
                if (ypml) psi_fix1(tEz, -1.f, __ldg(P.T.b[0][1] + j), __ldg(P.T.a[0][1] + j), __ldg(P.T.ik[0][1] + j) - 1.f,
                                   lds1(so + (L.pey + 1) * C::SLOT), dHx_dy);
                if (xpml) {
                    const float b = __ldg(P.T.b[0][0] + i), a = __ldg(P.T.a[0][0] + i), km = __ldg(P.T.ik[0][0] + i) - 1.f;
                    psi_fix1(tEz, 1.f, b, a, km, lds1(sb0 + L.pex * C::SLOT + o_x), dHy_dx);
                    psi_fix1(tEy, -1.f, b, a, km, lds1(sb0 + L.pex * C::SLOT + P.small_off + o_x), dHz_dx);
                }
                const float sie = S * lds1(so + 6 * C::SLOT);
                float ey_h = lds1(so + 4 * C::SLOT) + sie * tEy, ez_h = lds1(so + 5 * C::SLOT) + sie * tEz;
                if (src_plane) { ey_h += source_at(P, n, 1, i, j, kk); ez_h += source_at(P, n, 2, i, j, kk); }
                sts1(rgA + C::RING_COMP * 4, ey_h);
                sts1(rgA + 2 * C::RING_COMP * 4, ez_h);
                hx.x = hx_h;
            }
            // ---------------------------------------------------------------- phase B: H'(kk-1), 4 cells
            if (vec && doB && !halo_row) {
                const int km1 = kk - 1;
                const uint32_t rgB = ring_base + (km1 & 1) * (C::RING_SLOT * 4) + r_own;
                const float4 ex_py = lds4(rgB + C::RP * 4), ez_py = lds4(rgB + (2 * C::RING_COMP + C::RP) * 4);
                const float ey_px = lds1(rgB + (C::RING_COMP + 4) * 4), ez_px = lds1(rgB + (2 * C::RING_COMP + 4) * 4);
                const float4 dEz_dy = ez_py - e1z, dEx_dy = ex_py - e1x;
                const float4 dEy_dz = e2y - e1y, dEx_dz = e2x - e1x;
                const float4 dEz_dx = dplus_x(e1z, ez_px), dEy_dx = dplus_x(e1y, ey_px);
                float4 tHx = dEz_dy - dEy_dz, tHy = dEx_dz - dEz_dx, tHz = dEy_dx - dEx_dy;
                const bool wr = own_ok;
                if (zH) {       // z axis: psiH_y0 (d = dEx_dz, +), psiH_x1 (d = dEy_dz, -)
                    const float4 b = splat(__ldg(P.T.b[1][2] + km1)), a = splat(__ldg(P.T.a[1][2] + km1)), km = splat(__ldg(P.T.ik[1][2] + km1) - 1.f);
                    const long long iz = ((long long)zslab_index(G, km1) * G.ny + j) * G.nx + i;
                    const float4 p0 = psi_fix(tHy, 1.f, b, a, km, lds4(so + L.phz * C::SLOT), dEx_dz);
                    const float4 p1 = psi_fix(tHx, -1.f, b, a, km, lds4(so + (L.phz + 1) * C::SLOT), dEy_dz);
                    if (wr) { stg4(pH.p[1][0] + iz, p0); stg4(pH.p[0][1] + iz, p1); }
                }
                if (warp_y) {   // y axis: psiH_x0 (d = dEz_dy, +), psiH_z1 (d = dEx_dy, -)
                    float b = 1.f, a = 0.f, km = 0.f;
                    if (ypml) { b = __ldg(P.T.b[1][1] + j); a = __ldg(P.T.a[1][1] + j); km = __ldg(P.T.ik[1][1] + j) - 1.f; }
                    const long long iy = ((long long)km1 * (2 * G.d) + sy) * G.nx + i;
                    const float4 p0 = psi_fix(tHx, 1.f, splat(b), splat(a), splat(km), lds4(so + L.phy * C::SLOT), dEz_dy);
                    const float4 p1 = psi_fix(tHz, -1.f, splat(b), splat(a), splat(km), lds4(so + (L.phy + 1) * C::SLOT), dEx_dy);
                    if (wr && ypml) { stg4(pH.p[0][0] + iy, p0); stg4(pH.p[2][1] + iy, p1); }
                }
                if (warp_x) {   // x axis: psiH_z0 (d = dEy_dx, +), psiH_y1 (d = dEz_dx, -)
                    float4 b = splat(1.f), a = splat(0.f), km = splat(0.f), q0 = a, q1 = a;
                    if (xpml) {
                        b = ldg4(P.T.b[1][0] + i); a = ldg4(P.T.a[1][0] + i); km = ldg4(P.T.ik[1][0] + i) - splat(1.f);
                        q0 = lds4(sb0 + L.phx * C::SLOT + o_x); q1 = lds4(sb0 + L.phx * C::SLOT + P.small_off + o_x);
                    }
                    const long long ix = ((long long)km1 * G.ny + j) * (2 * G.dpx) + sx;
                    const float4 p0 = psi_fix(tHz, 1.f, b, a, km, q0, dEy_dx);
                    const float4 p1 = psi_fix(tHy, -1.f, b, a, km, q1, dEz_dx);
                    if (wr && xpml) { stg4(pH.p[2][0] + ix, p0); stg4(pH.p[1][1] + ix, p1); }
                }
                const float4 sim = has_mu ? S * lds4(so + L.im * C::SLOT) : splat(S);
                float4 h2x = hxk - sim * tHx, h2y = hyk - sim * tHy, h2z = hzk - sim * tHz;
                if (wr) {
                    if (P.n_src && any_source_plane(P, 1, km1)) {
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            f4add(h2x, q, source_at(P, n, 3, i + q, j, km1));
                            f4add(h2y, q, source_at(P, n, 4, i + q, j, km1));
                            f4add(h2z, q, source_at(P, n, 5, i + q, j, km1));
                        }
                    }
                    float *o = dst + 3 * nc + (long long)km1 * plane + own_xy;
                    stg4(o, h2x); stg4(o + nc, h2y); stg4(o + 2 * nc, h2z);
                    if (P.n_det && any_detector_plane(P, 1, km1)) {
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            detect_cell(P, n, 3, f4get(h2x, q), i + q, j, km1);
                            detect_cell(P, n, 4, f4get(h2y, q), i + q, j, km1);
                            detect_cell(P, n, 5, f4get(h2z, q), i + q, j, km1);
                        }
                    }
                }
            }
            e1x = e2x; e1y = e2y; e1z = e2z;
            hxk = hx; hyk = hy; hzk = hz;
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[bi]);
            named_bar_sync(1, C::NCW * 32);      // E' ring slot (kk-1)&1 may be overwritten in the next iteration
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

// ---- the compiled tile shapes ----------------------------------------------------------------------
struct TileImpl {
    int TX, TY, threads, slot, ring_bytes;
    void (*launch)(const FwdParams &, int n_cta, size_t smem, cudaStream_t);
    cudaError_t (*set_smem)(size_t);
};
template <class C> void launch_impl(const FwdParams &P, int n_cta, size_t smem, cudaStream_t st)
{
    k_fused_forward<C><<<n_cta, C::THREADS, smem, st>>>(P);
}
template <class C> cudaError_t set_smem_impl(size_t smem)
{
    return cudaFuncSetAttribute(k_fused_forward<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}
#define TILE(TX4, TY) { 4 * TX4, TY, Cfg<TX4, TY>::THREADS, Cfg<TX4, TY>::SLOT, Cfg<TX4, TY>::RING_BYTES, launch_impl<Cfg<TX4, TY>>, set_smem_impl<Cfg<TX4, TY>> }
const TileImpl kTiles[] = {
    TILE(2, 2), TILE(4, 4), TILE(8, 8), TILE(16, 8), TILE(16, 16), TILE(25, 10), TILE(25, 16), TILE(32, 8), TILE(32, 12),
};
constexpr int kNumTiles = sizeof(kTiles) / sizeof(kTiles[0]);

}  // namespace

struct FusedState {
    const TileImpl *tile = nullptr;
    int TX = 0, TY = 0, nslots = 0, n_cta = 0, n_rot = 1;
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

// cuts the flattened (tile, plane) sequence, rotated by `rot` planes, into n_cta equal runs
void make_segments(const Dims &G, int TX, int TY, int n_cta, long long rot, std::vector<Segment> &segs, std::vector<int> &seg_begin)
{
    const int ntx = (G.nx + TX - 1) / TX, nty = (G.ny + TY - 1) / TY;
    const long long total = (long long)ntx * nty * G.nz;
    segs.clear();
    seg_begin.assign(n_cta + 1, 0);
    rot = ((rot % total) + total) % total;
    for (int cta = 0; cta < n_cta; ++cta) {
        seg_begin[cta] = (int)segs.size();
        long long a = total * cta / n_cta, b = total * (cta + 1) / n_cta;      // positions in the rotated sequence
        while (a < b) {
            const long long pos = (a + rot) % total;                            // position in the canonical sequence
            const long long tile = pos / G.nz;
            const int k = (int)(pos % G.nz);
            const int len = (int)std::min<long long>(b - a, G.nz - k);
            const int txi = (int)(tile / nty), tyi = (int)(tile % nty);
            Segment s{};
            s.i0 = txi * TX; s.j0 = tyi * TY; s.k0 = k; s.k1 = k + len;
            if (G.d > 0) {
                if (s.i0 < G.dpx) s.flags |= SEG_X_LO;
                if (s.i0 + TX >= G.nx - G.dpx) s.flags |= SEG_X_HI;
                if (s.j0 < G.d) s.flags |= SEG_Y_LO;
                if (s.j0 + TY >= G.ny - G.d) s.flags |= SEG_Y_HI;
            }
            s.xbase = (s.flags & SEG_X_HI) ? std::max(s.i0, G.nx - G.dpx) : s.i0;
            segs.push_back(s);
            a += len;
        }
    }
    seg_begin[n_cta] = (int)segs.size();
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

    // ---- tile choice among the compiled shapes --------------------------------------------------------------------
    // A tile (with its +x halo column / +y halo row) may touch at most one CPML slab per axis, and the two narrow
    // x-psi boxes must fit into one slot.
    const int base_slots_per_plane = 7 + 1 + (G.d > 0 ? 8 : 0);
    int fTX = 0, fTY = 0;
    if (const char *e = getenv("FDTD_TILE")) sscanf(e, "%d,%d", &fTX, &fTY);
    const TileImpl *best = nullptr;
    double best_score = -1;
    int best_slots = 0;
    for (int q = 0; q < kNumTiles; ++q) {
        const TileImpl &t = kTiles[q];
        if (fTX && (t.TX != fTX || t.TY != fTY)) continue;
        if (G.d > 0) {
            if (t.TX >= G.nx - 2 * G.dpx || t.TY + 1 >= G.ny - 2 * G.d) continue;
        }
        const int xsl = G.d > 0 ? (2 * align_up((G.dpx + 8) * (t.TY + 2) * 4, 128) + t.slot - 1) / t.slot : 0;
        const int max_slots_per_plane = base_slots_per_plane + 2 * xsl;
        const int nslots = std::min(4096, (smem_cap - t.ring_bytes - 2 * NBAR * 8 - 1024) / t.slot);
        if (nslots < max_slots_per_plane + 3) continue;              // at least one plane of lookahead even in a corner
        const double eff_x = (double)G.nx / (((G.nx + t.TX - 1) / t.TX) * t.TX);
        const double eff_y = (double)G.ny / (((G.ny + t.TY - 1) / t.TY) * t.TY);
        const double halo = (double)(t.TX + 8) * (t.TY + 2) / ((double)t.TX * t.TY);
        const int NT = (t.TX / 4) * (t.TY + 1);
        const double thr = (double)NT / (t.threads - 32);
        const long long n_tiles = (long long)((G.nx + t.TX - 1) / t.TX) * ((G.ny + t.TY - 1) / t.TY);
        const double fill = std::min(1.0, (double)n_tiles * G.nz / (8.0 * n_sm));   // enough planes per CTA to amortise prologues
        const double score = eff_x * eff_y * thr * fill / (28.0 * halo + 24.0);
        if (score > best_score) { best_score = score; best = &t; best_slots = nslots; }
    }
    if (!best) { g->fused_why_not = "no compiled tile shape fits this grid (too small for its PML)"; return FDTD_OK; }

    FusedState *F = new FusedState();
    g->fused = F;
    F->tile = best; F->TX = best->TX; F->TY = best->TY; F->nslots = best_slots;
    F->smem = (size_t)best_slots * best->slot + best->ring_bytes + 2 * NBAR * 8;
    int rc;
    if ((rc = g->alloc((void **)&F->bufB, (size_t)G.nc * 6 * sizeof(float)))) return rc;
    if ((rc = g->alloc_psi(g->psiE[1])) || (rc = g->alloc_psi(g->psiH[1]))) return rc;
    if ((rc = g->alloc((void **)&F->d_maps, sizeof(CUtensorMap) * TM_COUNT))) return rc;
    if (cudaMallocHost((void **)&F->h_maps, sizeof(CUtensorMap) * TM_COUNT) != cudaSuccess ||
        cudaEventCreateWithFlags(&F->maps_done, cudaEventDisableTiming) != cudaSuccess) {
        (void)cudaGetLastError();
        return fdtd_fail(FDTD_ENOMEM, "pinned tensor-map staging allocation failed");
    }

    // ---- segments ---------------------------------------------------------------------------------------------------
    const int ntx = (G.nx + F->TX - 1) / F->TX, nty = (G.ny + F->TY - 1) / F->TY;
    const long long total = (long long)ntx * nty * G.nz;
    int n_cta = (int)std::min<long long>(n_sm, std::max<long long>(1, total / 6));
    if (const char *e = getenv("FDTD_NCTA")) n_cta = std::max(1, atoi(e));
    // rotation of the work sequence between steps (L2 reuse: a CTA starts where the data written last step is
    // still cached); n_rot tables, step n uses table n % n_rot
    int n_rot = 1;
    if (const char *e = getenv("FDTD_NROT")) n_rot = std::max(1, std::min(16, atoi(e)));
    F->n_cta = n_cta; F->n_rot = n_rot;
    std::vector<Segment> all;
    std::vector<int> begins;
    std::vector<std::vector<Segment>> per(n_rot);
    std::vector<std::vector<int>> per_b(n_rot);
    size_t stride = 0;
    for (int r = 0; r < n_rot; ++r) {
        const long long per_cta = total / n_cta;
        make_segments(G, F->TX, F->TY, n_cta, -(long long)r * (per_cta / n_rot), per[r], per_b[r]);
        stride = std::max(stride, per[r].size());
    }
    all.resize(stride * n_rot);
    for (int r = 0; r < n_rot; ++r) {
        std::copy(per[r].begin(), per[r].end(), all.begin() + r * stride);
        begins.insert(begins.end(), per_b[r].begin(), per_b[r].end());
    }
    if ((rc = g->alloc((void **)&F->d_segs, all.size() * sizeof(Segment)))) return rc;
    if ((rc = g->alloc((void **)&F->d_seg_begin, begins.size() * sizeof(int)))) return rc;
    if (cudaMemcpy(F->d_segs, all.data(), all.size() * sizeof(Segment), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(F->d_seg_begin, begins.data(), begins.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
        (void)cudaGetLastError();
        return fdtd_fail(FDTD_ECUDA, "upload of the segment table failed");
    }

    // ---- kernel parameters that do not depend on the call -----------------------------------------------------------
    FwdParams &P = F->fp;
    P.G = G; P.T = g->T; P.maps = F->d_maps; P.segs = F->d_segs; P.seg_begin = F->d_seg_begin;
    P.n_rot = n_rot; P.seg_stride = (int)stride; P.n_cta = n_cta;
    P.step = g->d_step;
    P.nslots = F->nslots;
    P.XW = G.dpx + 8;
    P.small_bytes = P.XW * (F->TY + 2) * 4;
    P.small_off = align_up(P.small_bytes, 128);       // the second narrow box stays 128-byte aligned
    P.xslots = G.d > 0 ? (2 * P.small_off + best->slot - 1) / best->slot : 0;
    if (best->set_smem(F->smem) != cudaSuccess) {
        (void)cudaGetLastError();
        g->fused_why_not = "cannot reserve shared memory";
        return FDTD_OK;
    }
    g->path = FDTD_PATH_FUSED;
    g->tile_x = F->TX; g->tile_y = F->TY;
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
    cudaError_t e = cudaMemcpyAsync(F->d_maps, F->h_maps, sizeof(CUtensorMap) * TM_COUNT, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaEventRecord(F->maps_done, st);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, std::string("tensor map upload: ") + cudaGetErrorString(e)); }
    F->maps_fields = fields; F->maps_ie = ie; F->maps_im = im;
    return FDTD_OK;
}

}  // namespace

// run_steps lives in fdtd_api.cu; reached through a small trampoline
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
      F->tile->launch(c->P, F->n_cta, F->smem, cs); }
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
