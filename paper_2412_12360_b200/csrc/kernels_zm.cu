// kernels_zm.cu -- fused z-marching kernels of the hot path (DESIGN.md sections 7-8):
//
//   k_zm_step<C, false>  forward step  : E update + H update + CPML psi + sources + detectors (F1-F7)
//   k_zm_step<C, true>   adjoint step  : transpose of the H update, then of the E update, adjoint CPML (B2+B5)
//   k_zm_inverse<C>      inverse step  : H = H' + S im curl+ E', q = curl- H, g += S lamE'.q, E = E' - S ie q (B3+B4)
//
// PAPER.md: Eq. 1-2 (L64-66) for the curl updates, L72 for the CPML, L78-84 for the VJP and the inverse step.
//
// Common design
//   * ping-pong volumes: a launch reads buffer `par` and writes buffer `par^1`, so tiles are independent;
//   * the xy plane is cut into TX x TY tiles, a tile's z column into segments; a persistent CTA (one per SM)
//     marches its segments plane by plane (2.5-D blocking), carrying the previous plane in registers;
//   * one producer thread streams each plane's boxes (fields, inv_eps, psi slabs; one-cell halo, 16-byte
//     aligned in x) global -> shared with TMA (cp.async.bulk.tensor; the zero fill outside the grid IS the
//     zero-pad wall convention R7) into a ring of equally sized slots; a plane takes as many slots as it has
//     arrays, so interior planes are prefetched several deep; mbarrier full/empty per plane;
//   * consumer threads own a float4 of cells.  Plane kk, phase A: the E-type update of plane kk on the tile
//     plus a +x halo column and a +y halo row (recomputed, not exchanged between CTAs), result to global and
//     to a shared ring; phase B: the H-type update of plane kk-1 from the phase-A results of planes kk-1
//     (registers + shared ring) and kk (registers);
//   * CPML: every difference D gets the correction of the time-recursive filter  p' = b p + a x,
//     c = (ik-1) x + p'  only on planes / warps that touch a slab.  Forward: x = D (filter after the
//     difference).  Adjoint: the filter acts on the operands before the difference (its tables depend on
//     the position along the difference axis), with the rescaled state theta = (a/b) * lambda_psi, which
//     obeys the same recursion as the forward psi.
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

struct StepParams {
    Dims G;
    Tables T;
    const CUtensorMap *maps;       // tensor maps of this kernel's volumes (layout: fused_common.cuh)
    const Segment *segs;           // [n_rot][seg_stride]
    const int *seg_begin;          // [n_rot][n_cta + 1]
    int n_rot, seg_stride, n_cta;
    float *buf[2];                 // ping-pong volumes, [6][nc] each
    PsiSet psiE[2], psiH[2];       // CPML states of the E-type / H-type update, ping-pong
    const int *step;
    int nslots;                    // slots in the shared-memory ring
    int XW, small_bytes;           // narrow x-psi box: width (floats) and exact byte size (TMA transaction bytes)
    int small_off, xslots;         // a pair of narrow boxes sits at offsets 0 / small_off of `xslots` consecutive slots
    int TW;                        // CPML table window: entries [0,TW) and [N-TW+4, N+4) of every axis table live in smem
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
    static constexpr int ROWB = PW * 4;                                  // box row pitch in bytes
    static constexpr int BOX_BYTES = PW * ROWS * 4;                    // TMA transaction bytes of a big box
    static constexpr int SLOT = (BOX_BYTES + 127) / 128 * 128;          // slot pitch
    static constexpr int CW = TX4 + 1;                                  // float4 threads per row (incl. the +x halo column)
    static constexpr int RP = 4 * CW;                                   // phase-A result ring: row pitch (floats)
    static constexpr int RING_COMP = (TY + 1) * RP, RING_SLOT = 3 * RING_COMP;
    static constexpr int RING_BYTES = (2 * RING_SLOT * 4 + 127) / 128 * 128;
    static constexpr int NT = CW * (TY + 1);                            // float4 threads (incl. halo row and column)
    static constexpr int NCW = (NT + 31) / 32;                          // consumer warps
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
__device__ __forceinline__ float4 ldg4(const float *p) { return __ldg(reinterpret_cast<const float4 *>(p)); }
__device__ __forceinline__ void stg4(float *p, float4 v) { *reinterpret_cast<float4 *>(p) = v; }
__device__ __forceinline__ float4 fma4(float4 a, float4 b, float4 c)
{
    return make_float4(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y), fmaf(a.z, b.z, c.z), fmaf(a.w, b.w, c.w));
}
__device__ __forceinline__ float4 fma4(float a, float4 b, float4 c)
{
    return make_float4(fmaf(a, b.x, c.x), fmaf(a, b.y, c.y), fmaf(a, b.z, c.z), fmaf(a, b.w, c.w));
}

__device__ __forceinline__ bool in_zslab(const Dims &G, int k) { return G.d > 0 && k >= 0 && k < G.nz && (k < G.d || k >= G.nz - G.d); }
__device__ __forceinline__ int zslab_index(const Dims &G, int k) { return k < G.d ? k : k - (G.nz - 2 * G.d); }

// CPML recursive filter at one point: p' = b p + a x; returns the correction c = (ik - 1) x + p'
__device__ __forceinline__ float4 cpml4(float4 b, float4 a, float4 km, float4 p, float4 x, float4 &pn)
{
    pn = fma4(b, p, a * x);
    return fma4(km, x, pn);
}
__device__ __forceinline__ float4 cpml4(float b, float a, float km, float4 p, float4 x, float4 &pn)
{
    pn = fma4(b, p, a * x);
    return fma4(km, x, pn);
}
__device__ __forceinline__ float cpml1(float b, float a, float km, float p, float x) { return fmaf(km, x, fmaf(b, p, a * x)); }

// Slot ordinals of the arrays every non-prologue plane of a segment carries.  Shared by producer and consumers.
//   0-2 H-type fields, 3-5 E-type fields, 6 inv_eps, [inv_mu], [y-slab: E-state pair, H-state pair],
//   [x-slab: E-state narrow pair, H-state narrow pair], then per plane [z-slab phase-A pair] [z-slab phase-B pair]
struct SegLayout { int im, ey, hy, ex, hx, nconst; };
__device__ __forceinline__ SegLayout seg_layout(bool has_mu, bool ys, bool xs, int xslots)
{
    SegLayout L;
    int o = 7;
    L.im = L.ey = L.hy = L.ex = L.hx = 0;
    if (has_mu) { L.im = o; o += 1; }
    if (ys) { L.ey = o; o += 2; L.hy = o; o += 2; }
    if (xs) { L.ex = o; o += xslots; L.hx = o; o += xslots; }
    L.nconst = o;
    return L;
}

// additive source contribution to component `comp` at cell (i,j,k) during this step
__device__ __noinline__ float source_at(const StepParams &P, int n, int comp, int i, int j, int k)
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

// running DFT of component `comp` (value v) at cell (i,j,k): P_f += v (cos - i sin)
__device__ __noinline__ void detect_cell(const StepParams &P, int n, int comp, float v, int i, int j, int k)
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

__device__ __forceinline__ float f4get(const float4 &v, int q) { return q == 0 ? v.x : (q == 1 ? v.y : (q == 2 ? v.z : v.w)); }
__device__ __forceinline__ void f4add(float4 &v, int q, float a) { if (q == 0) v.x += a; else if (q == 1) v.y += a; else if (q == 2) v.z += a; else v.w += a; }

// adds the sources of `family` (0 = E, 1 = H) to the three float4s of cell group (i..i+3, j, k); rare planes only
#define ADD_SOURCES4(P, n, family, vx, vy, vz, i, j, k)                                                   \
    do {                                                                                                  \
        vx.x += source_at(P, n, 3 * (family) + 0, (i) + 0, j, k); vx.y += source_at(P, n, 3 * (family) + 0, (i) + 1, j, k); \
        vx.z += source_at(P, n, 3 * (family) + 0, (i) + 2, j, k); vx.w += source_at(P, n, 3 * (family) + 0, (i) + 3, j, k); \
        vy.x += source_at(P, n, 3 * (family) + 1, (i) + 0, j, k); vy.y += source_at(P, n, 3 * (family) + 1, (i) + 1, j, k); \
        vy.z += source_at(P, n, 3 * (family) + 1, (i) + 2, j, k); vy.w += source_at(P, n, 3 * (family) + 1, (i) + 3, j, k); \
        vz.x += source_at(P, n, 3 * (family) + 2, (i) + 0, j, k); vz.y += source_at(P, n, 3 * (family) + 2, (i) + 1, j, k); \
        vz.z += source_at(P, n, 3 * (family) + 2, (i) + 2, j, k); vz.w += source_at(P, n, 3 * (family) + 2, (i) + 3, j, k); \
    } while (0)
__device__ __noinline__ void detect4(const StepParams &P, int n, int family, float4 vx, float4 vy, float4 vz, int i, int j, int k)
{
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        detect_cell(P, n, 3 * family + 0, f4get(vx, q), i + q, j, k);
        detect_cell(P, n, 3 * family + 1, f4get(vy, q), i + q, j, k);
        detect_cell(P, n, 3 * family + 2, f4get(vz, q), i + q, j, k);
    }
}

// ================================================================================================
// The step kernel.  Names follow the forward step: "F" is the H-type source of phase A, "e" the
// E-type target, "v" the phase-A result that phase B differences, "h" the H-type target.
//   forward : e' = e + S ie curl-(F = H)            v = e'            h' = h - S im curl+(v)
//   adjoint : e' = e - S curl-(F = lamH)   (im = 1) v = S ie e'       h' = h + curl+(v)
// curl with CPML: t_x = Dy_z - Dz_y, t_y = Dz_x - Dx_z, t_z = Dx_y - Dy_x, where D<a>_<c> is the
// (filtered) difference of component c along axis a; its state array is
//   Dy_z p[0][0]   Dz_y p[0][1]   Dz_x p[1][0]   Dx_z p[1][1]   Dx_y p[2][0]   Dy_x p[2][1].
// ================================================================================================
template <class C, bool ADJ>
__global__ void __launch_bounds__(C::THREADS, 1) k_zm_step(const __grid_constant__ StepParams P)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const Dims &G = P.G;
    const uint32_t slots_base = smem_u32(smem);
    const uint32_t ring_base = slots_base + (uint32_t)P.nslots * C::SLOT;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)P.nslots * C::SLOT + C::RING_BYTES);
    uint64_t *empty = full + NBAR;
    int *start = reinterpret_cast<int *>(empty + NBAR);      // producer: first slot of each in-flight plane-load
    float *tabs = reinterpret_cast<float *>(start + NBAR);   // CPML table windows [family][axis][b, a, ik-1][2*TW]
    const uint32_t tab_base = smem_u32(tabs);
    const int TW = P.TW;
    const uint32_t tw8 = 2u * TW * 4u;                       // bytes of one table (both windows)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = *P.step;
    const int par = (n + (ADJ ? 1 : 0)) & 1;       // forward step n reads buffer n&1; reverse step n reads (n+1)&1
    constexpr int FA = ADJ ? 1 : 0, FB = ADJ ? 0 : 1;   // CPML family (tables, states) of phase A / phase B

    if (threadIdx.x == 0) {
        for (int s = 0; s < NBAR; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], C::NCW); }
        fence_mbar_init();
    }
    if (G.d > 0) {
        // window entry q of axis a: position q (q < TW) or N_a - 2*TW + 4 + q (the first cell outside the grid included)
        for (int e = threadIdx.x; e < 18 * 2 * TW; e += blockDim.x) {
            const int tb = e / (2 * TW), q = e - tb * (2 * TW);
            const int fam = tb / 9, ax = (tb / 3) % 3, kind = tb % 3;
            const int N = ax == 0 ? G.nx : (ax == 1 ? G.ny : G.nz);
            int pos = q < TW ? q : N - 2 * TW + 4 + q;
            pos = min(max(pos, 0), N + 3);                    // tables are padded to N + 4 entries (b = 1, a = 0, ik = 1)
            const float *src = kind == 0 ? P.T.b[fam][ax] : (kind == 1 ? P.T.a[fam][ax] : P.T.ik[fam][ax]);
            tabs[e] = __ldg(src + pos) - (kind == 2 ? 1.f : 0.f);
        }
    }
    __syncthreads();

    const int rot = n % P.n_rot;
    const int *sb = P.seg_begin + rot * (P.n_cta + 1);
    const Segment *segs = P.segs + (size_t)rot * P.seg_stride;
    const int seg_lo = sb[blockIdx.x], seg_hi = sb[blockIdx.x + 1];
    const bool has_mu = !ADJ && P.has_mu != 0;

    // ============================================================================== producer
    if (warp == C::NCW) {
        if (lane != 0) return;
        const CUtensorMap *M = P.maps;
        int ld = 0;                 // plane-loads issued
        int head = 0;               // next free slot
        int tail_ld = 0;            // oldest plane-load not yet known to be released
        int tail_pos = 0;
        for (int sg = seg_lo; sg < seg_hi; ++sg) {
            const Segment S = segs[sg];
            const int x = S.i0 - 4, y = S.j0 - 1;
            const bool xs = (S.flags & (SEG_X_LO | SEG_X_HI)) != 0, ys = (S.flags & (SEG_Y_LO | SEG_Y_HI)) != 0;
            const int xhi = (S.flags & SEG_X_HI) ? 1 : 0, yhi = (S.flags & SEG_Y_HI) ? 1 : 0;
            const int xv = (xhi ? S.xbase - (G.nx - G.dpx) : S.xbase) - 4;     // x-psi box start in view coordinates
            const int yv = yhi ? y - (G.ny - G.d) : y;                          // y-psi box start in view coordinates
            const SegLayout L = seg_layout(has_mu, ys, xs, P.xslots);
            for (int kk = S.k0 - 1; kk <= S.k1; ++kk, ++ld) {
                const bool prolog = kk == S.k0 - 1;
                const bool zk = in_zslab(G, kk);
                bool zA, zB;
                int nsl, n_big, n_small;
                if (prolog) { zA = ADJ && zk; zB = false; nsl = 3 + (zA ? 2 : 0); n_big = nsl; n_small = 0; }
                else {
                    zA = zk;
                    zB = ADJ ? zk : (kk >= S.k0 + 1 && in_zslab(G, kk - 1));
                    nsl = L.nconst + (zA ? 2 : 0) + (zB ? 2 : 0);
                    n_small = xs ? 4 : 0;
                    n_big = nsl - (xs ? 2 * P.xslots : 0);
                }
                // ---- allocate nsl contiguous slots (never wrapping inside a plane-load)
                int base = head + nsl > P.nslots ? 0 : head;
                for (;;) {
                    const int inflight = ld - tail_ld;
                    bool fits;
                    if (inflight == 0) fits = true;
                    else if (inflight >= NBAR) fits = false;
                    else if (head > tail_pos) fits = (base == head) ? true : (nsl <= tail_pos);      // free: [head,N) U [0,tail)
                    else if (head < tail_pos) fits = (base == head) && (head + nsl <= tail_pos);     // free: [head,tail)
                    else fits = false;                                                                // ring full
                    if (fits) break;
                    mbar_wait(&empty[tail_ld % NBAR], (tail_ld / NBAR) & 1);
                    ++tail_ld;
                    tail_pos = (tail_ld < ld) ? start[tail_ld % NBAR] : base;
                }
                if (ld - tail_ld == 0) tail_pos = base;
                start[ld % NBAR] = base;
                head = base + nsl;
                uint64_t *fb = &full[ld % NBAR];
                uint8_t *st = smem + (size_t)base * C::SLOT;
                mbar_expect_tx(fb, (uint32_t)n_big * C::BOX_BYTES + (uint32_t)n_small * P.small_bytes);
                for (int c = 0; c < 3; ++c) tma_load_3d(st + c * C::SLOT, M + TM_FIELD + par * 6 + 3 + c, x, y, kk, fb);
                if (prolog) {
                    if (zA) {
                        const int kz = zslab_index(G, kk);
                        tma_load_3d(st + 3 * C::SLOT, M + tm_psi(par, FA, 8), x, y, kz, fb);
                        tma_load_3d(st + 4 * C::SLOT, M + tm_psi(par, FA, 9), x, y, kz, fb);
                    }
                    continue;
                }
                for (int c = 0; c < 3; ++c) tma_load_3d(st + (3 + c) * C::SLOT, M + TM_FIELD + par * 6 + c, x, y, kk, fb);
                tma_load_3d(st + 6 * C::SLOT, M + TM_IE, x, y, kk, fb);
                if (has_mu) tma_load_3d(st + L.im * C::SLOT, M + TM_IM, x, y, kk - 1, fb);
                const int oA_y = ADJ ? L.hy : L.ey, oB_y = ADJ ? L.ey : L.hy;
                const int oA_x = ADJ ? L.hx : L.ex, oB_x = ADJ ? L.ex : L.hx;
                if (ys) {
                    tma_load_3d(st + oA_y * C::SLOT, M + tm_psi(par, FA, 4 + 2 * yhi), x, yv, kk, fb);
                    tma_load_3d(st + (oA_y + 1) * C::SLOT, M + tm_psi(par, FA, 5 + 2 * yhi), x, yv, kk, fb);
                    tma_load_3d(st + oB_y * C::SLOT, M + tm_psi(par, FB, 4 + 2 * yhi), x, yv, kk - 1, fb);
                    tma_load_3d(st + (oB_y + 1) * C::SLOT, M + tm_psi(par, FB, 5 + 2 * yhi), x, yv, kk - 1, fb);
                }
                if (xs) {
                    tma_load_3d(st + oA_x * C::SLOT, M + tm_psi(par, FA, 0 + 2 * xhi), xv, y, kk, fb);
                    tma_load_3d(st + oA_x * C::SLOT + P.small_off, M + tm_psi(par, FA, 1 + 2 * xhi), xv, y, kk, fb);
                    tma_load_3d(st + oB_x * C::SLOT, M + tm_psi(par, FB, 0 + 2 * xhi), xv, y, kk - 1, fb);
                    tma_load_3d(st + oB_x * C::SLOT + P.small_off, M + tm_psi(par, FB, 1 + 2 * xhi), xv, y, kk - 1, fb);
                }
                int o = L.nconst;
                if (zA) {
                    const int kz = zslab_index(G, kk);
                    tma_load_3d(st + o * C::SLOT, M + tm_psi(par, FA, 8), x, y, kz, fb);
                    tma_load_3d(st + (o + 1) * C::SLOT, M + tm_psi(par, FA, 9), x, y, kz, fb);
                    o += 2;
                }
                if (zB) {
                    const int kz = zslab_index(G, ADJ ? kk : kk - 1);
                    tma_load_3d(st + o * C::SLOT, M + tm_psi(par, FB, 8), x, y, kz, fb);
                    tma_load_3d(st + (o + 1) * C::SLOT, M + tm_psi(par, FB, 9), x, y, kz, fb);
                }
            }
        }
        return;
    }

    // ============================================================================== consumers
    const int t = threadIdx.x;
    const bool act = t < C::NT;                                   // thread has a float4 of cells
    const int ty = act ? t / C::CW : 0;
    const int tx = act ? t - ty * C::CW : 0;
    const bool inner = act && ty < C::TY && tx < C::TX4;          // not a halo thread
    const uint32_t o_own = ((1 + ty) * C::PW + 4 + 4 * tx) * 4;   // my first cell inside a big box (bytes)
    const uint32_t r_own = (ty * C::RP + 4 * tx) * 4;             // ... inside the phase-A result ring
    float *dst = P.buf[par ^ 1];
    const PsiSet &pA = ADJ ? P.psiH[par ^ 1] : P.psiE[par ^ 1];   // states written by phase A / phase B
    const PsiSet &pB = ADJ ? P.psiE[par ^ 1] : P.psiH[par ^ 1];
    const float S = G.S;
    const long long nc = G.nc;
    const long long plane = (long long)G.ny * G.nx;
    // smem addresses of the table windows: family F, axis a, kind (0 b, 1 a, 2 ik-1)
#define TAB(F, a, kind) (tab_base + (uint32_t)(((F) * 3 + (a)) * 3 + (kind)) * tw8)
    const int hs_x = G.nx - 2 * TW + 4, hs_y = G.ny - 2 * TW + 4, hs_z = G.nz - 2 * TW + 4;   // window entry q >= TW holds position hs + q

    // k ranges of the planes that hold sources / detectors (forward only)
    int sEl = 1 << 30, sEh = -1, sHl = 1 << 30, sHh = -1, dEl = 1 << 30, dEh = -1, dHl = 1 << 30, dHh = -1;
    if (!ADJ) {
        for (int s = 0; s < P.n_src; ++s) {
            if (P.src[s].comp < 3) { sEl = min(sEl, P.src[s].lo[2]); sEh = max(sEh, P.src[s].hi[2]); }
            else { sHl = min(sHl, P.src[s].lo[2]); sHh = max(sHh, P.src[s].hi[2]); }
        }
        for (int s = 0; s < P.n_det; ++s) {
            if (P.det[s].mask & 7) { dEl = min(dEl, P.det[s].lo[2]); dEh = max(dEh, P.det[s].hi[2]); }
            if (P.det[s].mask >> 3) { dHl = min(dHl, P.det[s].lo[2]); dHh = max(dHh, P.det[s].hi[2]); }
        }
    }

    int ld = 0, head = 0;
    for (int sg = seg_lo; sg < seg_hi; ++sg) {
        const Segment Sg = segs[sg];
        const int i = Sg.i0 + 4 * tx, j = Sg.j0 + ty;
        const bool in_x = act && i < G.nx, in_y = act && j < G.ny;
        const bool own_ok = inner && in_x && in_y;
        const bool xs = (Sg.flags & (SEG_X_LO | SEG_X_HI)) != 0, ys = (Sg.flags & (SEG_Y_LO | SEG_Y_HI)) != 0;
        const SegLayout L = seg_layout(has_mu, ys, xs, P.xslots);
        const int oA_y = ADJ ? L.hy : L.ey, oB_y = ADJ ? L.ey : L.hy;
        const int oA_x = ADJ ? L.hx : L.ex, oB_x = ADJ ? L.ex : L.hx;
        // cells whose own CPML state exists (store predicate) and cells that run the slab code of each phase
        const bool ypml = G.d > 0 && in_y && (j < G.d || j >= G.ny - G.d);
        const bool xpml = G.d > 0 && in_x && (i < G.dpx || i >= G.nx - G.dpx);
        const bool yA = ys && (ADJ ? (G.d > 0 && in_y && (j <= G.d || j >= G.ny - G.d)) : ypml);
        const bool yB = ys && (ADJ ? (G.d > 0 && in_y && (j < G.d || j >= G.ny - G.d - 1)) : ypml);
        const bool xA = xs && (ADJ ? (G.d > 0 && in_x && (i <= G.dpx || i >= G.nx - G.dpx)) : xpml);
        const bool xB = xs && (ADJ ? (G.d > 0 && in_x && (i < G.dpx || i >= G.nx - G.dpx - 4)) : xpml);
        const bool warp_yA = __any_sync(0xffffffffu, yA), warp_yB = __any_sync(0xffffffffu, yB && inner);
        const bool warp_xA = __any_sync(0xffffffffu, xA), warp_xB = __any_sync(0xffffffffu, xB && inner);
        const uint32_t o_x = (xA || xB) ? ((1 + ty) * P.XW + (i - Sg.xbase + 4)) * 4 : 0;   // my cells inside a narrow x-psi box
        const int sy = j < G.d ? j : j - (G.ny - 2 * G.d);
        const int sx = i < G.dpx ? i : i - (G.nx - 2 * G.dpx);
        const long long own_xy = (long long)j * G.nx + i;
        // byte offsets of my position inside the table windows (valid whenever the slab code of that axis runs)
        const uint32_t txo = (uint32_t)(i < TW ? i : i - hs_x) * 4u, txo_m = i > 0 ? txo - 4u : txo;
        const uint32_t tyo = (uint32_t)(j < TW ? j : j - hs_y) * 4u, tyo_m = j > 0 ? tyo - 4u : tyo;

        float4 hxk = splat(0.f), hyk = hxk, hzk = hxk;      // H-type target of plane kk-1 at my cells (raw)
        float4 fxk = hxk, fyk = hxk;                        // z operands of phase A from plane kk-1 (adjoint: filtered)
        float4 v1x = hxk, v1y = hxk, v1z = hxk;             // phase-A result of plane kk-1 at my cells
        float4 g1x = hxk, g1y = hxk;                        // z operands of phase B from plane kk-1 (adjoint: filtered)

        for (int kk = Sg.k0 - 1; kk <= Sg.k1; ++kk, ++ld) {
            const bool prolog = kk == Sg.k0 - 1;
            const bool doB = kk >= Sg.k0 + 1;
            const bool zk = in_zslab(G, kk);
            bool zA, zB;
            int nsl;
            if (prolog) { zA = ADJ && zk; zB = false; nsl = 3 + (zA ? 2 : 0); }
            else {
                zA = zk;
                zB = ADJ ? zk : (doB && in_zslab(G, kk - 1));
                nsl = L.nconst + (zA ? 2 : 0) + (zB ? 2 : 0);
            }
            const int base = head + nsl > P.nslots ? 0 : head;
            head = base + nsl;
            const int bi = ld % NBAR;
            mbar_wait(&full[bi], (ld / NBAR) & 1);
            const uint32_t sb0 = slots_base + (uint32_t)base * C::SLOT;     // first slot of this plane-load
            const uint32_t so = sb0 + o_own;
            const int oAz = prolog ? 3 : L.nconst, oBz = L.nconst + (zA ? 2 : 0);
            const uint32_t tz = (uint32_t)(kk < TW ? kk : kk - hs_z) * 4u;                  // used on z-slab planes only
            const uint32_t tzm = (uint32_t)(kk - 1 < TW ? kk - 1 : kk - 1 - hs_z) * 4u;
            if (prolog) {
                if (act) {
                    hxk = lds4(so); hyk = lds4(so + C::SLOT); hzk = lds4(so + 2 * C::SLOT);
                    fxk = hxk; fyk = hyk;
                    if (ADJ && zA) {
                        const float b = lds1(TAB(FA, 2, 0) + tz), a = lds1(TAB(FA, 2, 1) + tz), km = lds1(TAB(FA, 2, 2) + tz);
                        float4 pn;
                        fxk = hxk + cpml4(b, a, km, lds4(so + oAz * C::SLOT), hxk, pn);
                        fyk = hyk + cpml4(b, a, km, lds4(so + (oAz + 1) * C::SLOT), hyk, pn);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[bi]);
                continue;
            }
            const bool storeE = kk < Sg.k1;
            const uint32_t rgA = ring_base + (kk & 1) * (C::RING_SLOT * 4) + r_own;
            float4 fx = splat(0.f), fy = fx, fz = fx, gx = fx, gy = fx, v2x = fx, v2y = fx, v2z = fx, g2x = fx, g2y = fx;
            if (act) {
                // ------------------------------------------------------------ phase A: E-type update of plane kk
                fx = lds4(so); fy = lds4(so + C::SLOT); fz = lds4(so + 2 * C::SLOT);
                const float4 fx_my = lds4(so - C::ROWB), fz_my = lds4(so + 2 * C::SLOT - C::ROWB);
                const float fy_mx = lds1(so + C::SLOT - 4), fz_mx = lds1(so + 2 * C::SLOT - 4);
                float4 Dy_z = fz - fz_my, Dy_x = fx - fx_my;
                float4 Dx_y = dminus_x(fy, fy_mx), Dx_z = dminus_x(fz, fz_mx);
                float4 Dz_x, Dz_y;
                const bool wr = own_ok && storeE;                  // I own these cells: write the result and the phase-A states
                gx = fx; gy = fy;
                if (ADJ) {
                    if (zA) {
                        const float b = lds1(TAB(FA, 2, 0) + tz), a = lds1(TAB(FA, 2, 1) + tz), km = lds1(TAB(FA, 2, 2) + tz);
                        float4 p0, p1;
                        gx = fx + cpml4(b, a, km, lds4(so + oAz * C::SLOT), fx, p0);
                        gy = fy + cpml4(b, a, km, lds4(so + (oAz + 1) * C::SLOT), fy, p1);
                        if (wr) {
                            const long long iz = ((long long)zslab_index(G, kk) * G.ny + j) * G.nx + i;
                            stg4(pA.p[1][0] + iz, p0); stg4(pA.p[0][1] + iz, p1);
                        }
                    }
                    Dz_x = gx - fxk; Dz_y = gy - fyk;
                } else {
                    Dz_x = fx - fxk; Dz_y = fy - fyk;
                    if (zA) {
                        const float b = lds1(TAB(FA, 2, 0) + tz), a = lds1(TAB(FA, 2, 1) + tz), km = lds1(TAB(FA, 2, 2) + tz);
                        float4 p0, p1;
                        Dz_x = Dz_x + cpml4(b, a, km, lds4(so + oAz * C::SLOT), Dz_x, p0);
                        Dz_y = Dz_y + cpml4(b, a, km, lds4(so + (oAz + 1) * C::SLOT), Dz_y, p1);
                        if (wr) {
                            const long long iz = ((long long)zslab_index(G, kk) * G.ny + j) * G.nx + i;
                            stg4(pA.p[1][0] + iz, p0); stg4(pA.p[0][1] + iz, p1);
                        }
                    }
                }
                if (warp_yA) {
                    if (yA) {
                        const float b = lds1(TAB(FA, 1, 0) + tyo), a = lds1(TAB(FA, 1, 1) + tyo), km = lds1(TAB(FA, 1, 2) + tyo);
                        const float4 s0 = lds4(so + oA_y * C::SLOT), s1 = lds4(so + (oA_y + 1) * C::SLOT);
                        float4 p0, p1;
                        if (ADJ) {
                            const float bm = lds1(TAB(FA, 1, 0) + tyo_m), am = lds1(TAB(FA, 1, 1) + tyo_m), kmm = lds1(TAB(FA, 1, 2) + tyo_m);
                            float4 q0, q1;
                            Dy_z = Dy_z + (cpml4(b, a, km, s0, fz, p0) - cpml4(bm, am, kmm, lds4(so + oA_y * C::SLOT - C::ROWB), fz_my, q0));
                            Dy_x = Dy_x + (cpml4(b, a, km, s1, fx, p1) - cpml4(bm, am, kmm, lds4(so + (oA_y + 1) * C::SLOT - C::ROWB), fx_my, q1));
                        } else {
                            Dy_z = Dy_z + cpml4(b, a, km, s0, Dy_z, p0);
                            Dy_x = Dy_x + cpml4(b, a, km, s1, Dy_x, p1);
                        }
                        if (wr && ypml) {
                            const long long iy = ((long long)kk * (2 * G.d) + sy) * G.nx + i;
                            stg4(pA.p[0][0] + iy, p0); stg4(pA.p[2][1] + iy, p1);
                        }
                    }
                }
                if (warp_xA) {
                    if (xA) {
                        const float4 b = lds4(TAB(FA, 0, 0) + txo), a = lds4(TAB(FA, 0, 1) + txo), km = lds4(TAB(FA, 0, 2) + txo);
                        const uint32_t sx0 = sb0 + oA_x * C::SLOT + o_x, sx1 = sx0 + P.small_off;
                        const float4 s0 = lds4(sx0), s1 = lds4(sx1);
                        float4 p0, p1;
                        if (ADJ) {
                            const float bm = lds1(TAB(FA, 0, 0) + txo_m), am = lds1(TAB(FA, 0, 1) + txo_m), kmm = lds1(TAB(FA, 0, 2) + txo_m);
                            Dx_y = Dx_y + dminus_x(cpml4(b, a, km, s0, fy, p0), cpml1(bm, am, kmm, lds1(sx0 - 4), fy_mx));
                            Dx_z = Dx_z + dminus_x(cpml4(b, a, km, s1, fz, p1), cpml1(bm, am, kmm, lds1(sx1 - 4), fz_mx));
                        } else {
                            Dx_y = Dx_y + cpml4(b, a, km, s0, Dx_y, p0);
                            Dx_z = Dx_z + cpml4(b, a, km, s1, Dx_z, p1);
                        }
                        if (wr && xpml) {
                            const long long ix = ((long long)kk * G.ny + j) * (2 * G.dpx) + sx;
                            stg4(pA.p[2][0] + ix, p0); stg4(pA.p[1][1] + ix, p1);
                        }
                    }
                }
                const float4 tEx = Dy_z - Dz_y, tEy = Dz_x - Dx_z, tEz = Dx_y - Dy_x;
                const float4 sie = S * lds4(so + 6 * C::SLOT);
                float4 e2x, e2y, e2z;
                if (ADJ) {
                    e2x = fma4(-S, tEx, lds4(so + 3 * C::SLOT));
                    e2y = fma4(-S, tEy, lds4(so + 4 * C::SLOT));
                    e2z = fma4(-S, tEz, lds4(so + 5 * C::SLOT));
                    v2x = sie * e2x; v2y = sie * e2y; v2z = sie * e2z;
                } else {
                    e2x = fma4(sie, tEx, lds4(so + 3 * C::SLOT));
                    e2y = fma4(sie, tEy, lds4(so + 4 * C::SLOT));
                    e2z = fma4(sie, tEz, lds4(so + 5 * C::SLOT));
                    if (kk >= sEl && kk < sEh) ADD_SOURCES4(P, n, 0, e2x, e2y, e2z, i, j, kk);
                    v2x = e2x; v2y = e2y; v2z = e2z;
                }
                sts4(rgA, v2x); sts4(rgA + C::RING_COMP * 4, v2y); sts4(rgA + 2 * C::RING_COMP * 4, v2z);
                if (wr) {
                    float *o = dst + (long long)kk * plane + own_xy;
                    stg4(o, e2x); stg4(o + nc, e2y); stg4(o + 2 * nc, e2z);
                    if (!ADJ && kk >= dEl && kk < dEh) detect4(P, n, 0, e2x, e2y, e2z, i, j, kk);
                }
                g2x = v2x; g2y = v2y;
                if (ADJ && zB) {       // z operands of phase B, filtered at plane kk
                    const float b = lds1(TAB(FB, 2, 0) + tz), a = lds1(TAB(FB, 2, 1) + tz), km = lds1(TAB(FB, 2, 2) + tz);
                    float4 p0, p1;
                    g2x = v2x + cpml4(b, a, km, lds4(so + oBz * C::SLOT), v2x, p0);
                    g2y = v2y + cpml4(b, a, km, lds4(so + (oBz + 1) * C::SLOT), v2y, p1);
                    if (wr) {
                        const long long iz = ((long long)zslab_index(G, kk) * G.ny + j) * G.nx + i;
                        stg4(pB.p[1][0] + iz, p0); stg4(pB.p[0][1] + iz, p1);
                    }
                }
            }
            // ---------------------------------------------------------------- phase B: H-type update of plane kk-1
            if (inner && doB) {
                const int km1 = kk - 1;
                const uint32_t rgB = ring_base + (km1 & 1) * (C::RING_SLOT * 4) + r_own;
                const float4 vx_py = lds4(rgB + C::RP * 4), vz_py = lds4(rgB + (2 * C::RING_COMP + C::RP) * 4);
                const float vy_px = lds1(rgB + (C::RING_COMP + 4) * 4), vz_px = lds1(rgB + (2 * C::RING_COMP + 4) * 4);
                float4 Dy_z = vz_py - v1z, Dy_x = vx_py - v1x;
                float4 Dz_y = g2y - g1y, Dz_x = g2x - g1x;
                float4 Dx_z = dplus_x(v1z, vz_px), Dx_y = dplus_x(v1y, vy_px);
                const bool wr = own_ok;
                if (!ADJ && zB) {
                    const float b = lds1(TAB(FB, 2, 0) + tzm), a = lds1(TAB(FB, 2, 1) + tzm), km = lds1(TAB(FB, 2, 2) + tzm);
                    float4 p0, p1;
                    Dz_x = Dz_x + cpml4(b, a, km, lds4(so + oBz * C::SLOT), Dz_x, p0);
                    Dz_y = Dz_y + cpml4(b, a, km, lds4(so + (oBz + 1) * C::SLOT), Dz_y, p1);
                    if (wr) {
                        const long long iz = ((long long)zslab_index(G, km1) * G.ny + j) * G.nx + i;
                        stg4(pB.p[1][0] + iz, p0); stg4(pB.p[0][1] + iz, p1);
                    }
                }
                if (warp_yB) {
                    if (yB) {
                        const float b = lds1(TAB(FB, 1, 0) + tyo), a = lds1(TAB(FB, 1, 1) + tyo), km = lds1(TAB(FB, 1, 2) + tyo);
                        const float4 s0 = lds4(so + oB_y * C::SLOT), s1 = lds4(so + (oB_y + 1) * C::SLOT);
                        float4 p0, p1;
                        if (ADJ) {
                            const float bp = lds1(TAB(FB, 1, 0) + tyo + 4), ap = lds1(TAB(FB, 1, 1) + tyo + 4), kmp = lds1(TAB(FB, 1, 2) + tyo + 4);
                            float4 q0, q1;
                            Dy_z = Dy_z + (cpml4(bp, ap, kmp, lds4(so + oB_y * C::SLOT + C::ROWB), vz_py, q0) - cpml4(b, a, km, s0, v1z, p0));
                            Dy_x = Dy_x + (cpml4(bp, ap, kmp, lds4(so + (oB_y + 1) * C::SLOT + C::ROWB), vx_py, q1) - cpml4(b, a, km, s1, v1x, p1));
                        } else {
                            Dy_z = Dy_z + cpml4(b, a, km, s0, Dy_z, p0);
                            Dy_x = Dy_x + cpml4(b, a, km, s1, Dy_x, p1);
                        }
                        if (wr && ypml) {
                            const long long iy = ((long long)km1 * (2 * G.d) + sy) * G.nx + i;
                            stg4(pB.p[0][0] + iy, p0); stg4(pB.p[2][1] + iy, p1);
                        }
                    }
                }
                if (warp_xB) {
                    if (xB) {
                        const float4 b = lds4(TAB(FB, 0, 0) + txo), a = lds4(TAB(FB, 0, 1) + txo), km = lds4(TAB(FB, 0, 2) + txo);
                        const uint32_t sx0 = sb0 + oB_x * C::SLOT + o_x, sx1 = sx0 + P.small_off;
                        const float4 s0 = lds4(sx0), s1 = lds4(sx1);
                        float4 p0, p1;
                        if (ADJ) {
                            const float bp = lds1(TAB(FB, 0, 0) + txo + 16), ap = lds1(TAB(FB, 0, 1) + txo + 16), kmp = lds1(TAB(FB, 0, 2) + txo + 16);
                            Dx_y = Dx_y + dplus_x(cpml4(b, a, km, s0, v1y, p0), cpml1(bp, ap, kmp, lds1(sx0 + 16), vy_px));
                            Dx_z = Dx_z + dplus_x(cpml4(b, a, km, s1, v1z, p1), cpml1(bp, ap, kmp, lds1(sx1 + 16), vz_px));
                        } else {
                            Dx_y = Dx_y + cpml4(b, a, km, s0, Dx_y, p0);
                            Dx_z = Dx_z + cpml4(b, a, km, s1, Dx_z, p1);
                        }
                        if (wr && xpml) {
                            const long long ix = ((long long)km1 * G.ny + j) * (2 * G.dpx) + sx;
                            stg4(pB.p[2][0] + ix, p0); stg4(pB.p[1][1] + ix, p1);
                        }
                    }
                }
                const float4 tHx = Dy_z - Dz_y, tHy = Dz_x - Dx_z, tHz = Dx_y - Dy_x;
                float4 h2x, h2y, h2z;
                if (ADJ) {
                    h2x = hxk + tHx; h2y = hyk + tHy; h2z = hzk + tHz;
                } else {
                    const float4 sim = has_mu ? S * lds4(so + L.im * C::SLOT) : splat(S);
                    h2x = hxk - sim * tHx; h2y = hyk - sim * tHy; h2z = hzk - sim * tHz;
                }
                if (wr) {
                    if (!ADJ && km1 >= sHl && km1 < sHh) ADD_SOURCES4(P, n, 1, h2x, h2y, h2z, i, j, km1);
                    float *o = dst + 3 * nc + (long long)km1 * plane + own_xy;
                    stg4(o, h2x); stg4(o + nc, h2y); stg4(o + 2 * nc, h2z);
                    if (!ADJ && km1 >= dHl && km1 < dHh) detect4(P, n, 1, h2x, h2y, h2z, i, j, km1);
                }
            }
            v1x = v2x; v1y = v2y; v1z = v2z;
            g1x = g2x; g1y = g2y;
            hxk = fx; hyk = fy; hzk = fz;
            fxk = gx; fyk = gy;
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[bi]);
            named_bar_sync(1, C::NCW * 32);      // ring slot (kk-1)&1 may be overwritten in the next iteration
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
    void (*launch_fwd)(const StepParams &, int n_cta, size_t smem, cudaStream_t);
    void (*launch_adj)(const StepParams &, int n_cta, size_t smem, cudaStream_t);
    cudaError_t (*set_smem)(size_t);
};
template <class C> void launch_fwd_impl(const StepParams &P, int n_cta, size_t smem, cudaStream_t st)
{
    k_zm_step<C, false><<<n_cta, C::THREADS, smem, st>>>(P);
}
template <class C> void launch_adj_impl(const StepParams &P, int n_cta, size_t smem, cudaStream_t st)
{
    k_zm_step<C, true><<<n_cta, C::THREADS, smem, st>>>(P);
}
template <class C> cudaError_t set_smem_impl(size_t smem)
{
    cudaError_t e = cudaFuncSetAttribute(k_zm_step<C, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_zm_step<C, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    return e;
}
#define TILE(TX4, TY) { 4 * TX4, TY, Cfg<TX4, TY>::THREADS, Cfg<TX4, TY>::SLOT, Cfg<TX4, TY>::RING_BYTES, \
                        launch_fwd_impl<Cfg<TX4, TY>>, launch_adj_impl<Cfg<TX4, TY>>, set_smem_impl<Cfg<TX4, TY>> }
const TileImpl kTiles[] = {
    TILE(2, 2), TILE(4, 4), TILE(8, 8), TILE(16, 8), TILE(16, 16), TILE(25, 10), TILE(25, 16), TILE(32, 8), TILE(32, 14), TILE(50, 8),
};
constexpr int kNumTiles = sizeof(kTiles) / sizeof(kTiles[0]);

}  // namespace

struct FusedState {
    const TileImpl *tile = nullptr;
    int TX = 0, TY = 0, nslots = 0, n_cta = 0, n_rot = 1;
    size_t smem = 0;
    StepParams sp{};
    float *bufB = nullptr;                 // second primal field buffer
    float *lamB = nullptr;                 // second cotangent buffer
    // tensor-map tables: [0] primal (fields / bufB, psi), [1] cotangents (lam / lamB, psi cotangents)
    CUtensorMap *d_maps[2] = { nullptr, nullptr };
    CUtensorMap *h_maps[2] = { nullptr, nullptr };   // pinned staging
    cudaEvent_t maps_done = nullptr;
    Segment *d_segs = nullptr;
    int *d_seg_begin = nullptr;
    const float *maps_key[2][3] = { { nullptr, nullptr, nullptr }, { nullptr, nullptr, nullptr } };   // pointers the maps were built for
};

namespace {

// Work sequence: z is cut into n_chunk chunks; the sequence is (chunk, tile [y fastest], plane in chunk); it is
// rotated by `rot` positions and cut into n_cta equal runs.  With chunk length ~ run length, CTAs that hold
// y-adjacent tiles march through the same planes at about the same time, so halo rows hit L2.
void make_segments(const Dims &G, int TX, int TY, int n_cta, int n_chunk, long long rot, std::vector<Segment> &segs,
                   std::vector<int> &seg_begin)
{
    const int ntx = (G.nx + TX - 1) / TX, nty = (G.ny + TY - 1) / TY;
    const long long n_tiles = (long long)ntx * nty;
    const long long total = n_tiles * G.nz;
    std::vector<int> cb(n_chunk + 1);
    for (int c = 0; c <= n_chunk; ++c) cb[c] = (int)((long long)G.nz * c / n_chunk);
    std::vector<long long> cstart(n_chunk + 1, 0);       // sequence position where each chunk begins
    for (int c = 0; c < n_chunk; ++c) cstart[c + 1] = cstart[c] + n_tiles * (cb[c + 1] - cb[c]);
    segs.clear();
    seg_begin.assign(n_cta + 1, 0);
    rot = ((rot % total) + total) % total;
    for (int cta = 0; cta < n_cta; ++cta) {
        seg_begin[cta] = (int)segs.size();
        long long a = total * cta / n_cta, b = total * (cta + 1) / n_cta;      // positions in the rotated sequence
        while (a < b) {
            const long long pos = (a + rot) % total;                            // position in the canonical sequence
            int c = (int)(std::upper_bound(cstart.begin(), cstart.end(), pos) - cstart.begin()) - 1;
            const int clen = cb[c + 1] - cb[c];
            const long long in_chunk = pos - cstart[c];
            const long long tile = in_chunk / clen;
            const int k = cb[c] + (int)(in_chunk % clen);
            const int len = (int)std::min<long long>(std::min<long long>(b - a, total - pos), cb[c + 1] - k);
            const int txi = (int)(tile / nty), tyi = (int)(tile % nty);
            Segment s{};
            s.i0 = txi * TX; s.j0 = tyi * TY; s.k0 = k; s.k1 = k + len;
            if (G.d > 0) {
                // a tile "touches" a slab if one of its threads (halo column / row included) runs slab code
                // in either kernel: own cells in the slab, or (adjoint) a difference neighbour in it
                if (s.i0 <= G.dpx) s.flags |= SEG_X_LO;
                if (s.i0 + TX >= G.nx - G.dpx) s.flags |= SEG_X_HI;
                if (s.j0 <= G.d) s.flags |= SEG_Y_LO;
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
    // A tile (with its halo column / row and the adjoint's difference neighbours) may touch at most one CPML slab
    // per axis, and the two narrow x-psi boxes must fit into whole slots.
    const int base_slots_per_plane = 7 + 1 + (G.d > 0 ? 8 : 0);       // fields, ie, im, y and z state pairs of both phases
    int fTX = 0, fTY = 0;
    if (const char *e = getenv("FDTD_TILE")) sscanf(e, "%d,%d", &fTX, &fTY);
    const int TW = G.d > 0 ? G.dpx + 8 : 0;                                  // CPML table window (entries per side)
    const int tail_bytes = 2 * NBAR * 8 + NBAR * 4 + 18 * 2 * TW * 4;        // mbarriers, producer bookkeeping, table windows
    const TileImpl *best = nullptr;
    double best_score = -1;
    int best_slots = 0;
    for (int q = 0; q < kNumTiles; ++q) {
        const TileImpl &t = kTiles[q];
        if (fTX && (t.TX != fTX || t.TY != fTY)) continue;
        if (G.d > 0) {
            if (t.TX + 8 > G.nx - 2 * G.dpx || t.TY + 3 > G.ny - 2 * G.d) continue;
        }
        const int xsl = G.d > 0 ? (2 * align_up((G.dpx + 8) * (t.TY + 2) * 4, 128) + t.slot - 1) / t.slot : 0;
        const int max_slots_per_plane = base_slots_per_plane + 2 * xsl;
        const int nslots = std::min(4096, (smem_cap - t.ring_bytes - tail_bytes - 1024) / t.slot);
        if (nslots < max_slots_per_plane + 3) continue;              // at least one plane of lookahead even in a corner
        const double eff_x = (double)G.nx / (((G.nx + t.TX - 1) / t.TX) * t.TX);
        const double eff_y = (double)G.ny / (((G.ny + t.TY - 1) / t.TY) * t.TY);
        const double halo = (double)(t.TX + 8) * (t.TY + 2) / ((double)t.TX * t.TY);
        const double thr = (double)(t.TX / 4) * t.TY / (t.threads - 32);
        const long long n_tiles = (long long)((G.nx + t.TX - 1) / t.TX) * ((G.ny + t.TY - 1) / t.TY);
        const double fill = std::min(1.0, (double)n_tiles * G.nz / (8.0 * n_sm));   // enough planes per CTA to amortise prologues
        const double warps = std::min(1.0, (t.threads - 32) / 384.0);               // enough warps to hide latency
        const double score = eff_x * eff_y * thr * fill * warps / (28.0 * halo + 24.0);
        if (score > best_score) { best_score = score; best = &t; best_slots = nslots; }
    }
    if (!best) { g->fused_why_not = "no compiled tile shape fits this grid (too small for its PML)"; return FDTD_OK; }

    FusedState *F = new FusedState();
    g->fused = F;
    F->tile = best; F->TX = best->TX; F->TY = best->TY; F->nslots = best_slots;
    F->smem = (size_t)best_slots * best->slot + best->ring_bytes + tail_bytes;
    int rc;
    if ((rc = g->alloc((void **)&F->bufB, (size_t)G.nc * 6 * sizeof(float)))) return rc;
    if ((rc = g->alloc_psi(g->psiE[1])) || (rc = g->alloc_psi(g->psiH[1]))) return rc;
    for (int q = 0; q < 2; ++q) {
        if ((rc = g->alloc((void **)&F->d_maps[q], sizeof(CUtensorMap) * TM_COUNT))) return rc;
        if (cudaMallocHost((void **)&F->h_maps[q], sizeof(CUtensorMap) * TM_COUNT) != cudaSuccess) {
            (void)cudaGetLastError();
            return fdtd_fail(FDTD_ENOMEM, "pinned tensor-map staging allocation failed");
        }
    }
    if (cudaEventCreateWithFlags(&F->maps_done, cudaEventDisableTiming) != cudaSuccess) {
        (void)cudaGetLastError();
        return fdtd_fail(FDTD_ENOMEM, "event creation failed");
    }

    // ---- segments ---------------------------------------------------------------------------------------------------
    const int ntx = (G.nx + F->TX - 1) / F->TX, nty = (G.ny + F->TY - 1) / F->TY;
    const long long total = (long long)ntx * nty * G.nz;
    int n_cta = (int)std::min<long long>(n_sm, std::max<long long>(1, total / 6));
    if (const char *e = getenv("FDTD_NCTA")) n_cta = std::max(1, atoi(e));
    const double run = (double)total / n_cta;                         // planes per CTA
    int n_chunk = std::max(1, (int)(G.nz / run + 0.5));
    if (const char *e = getenv("FDTD_NCHUNK")) n_chunk = std::max(1, std::min(G.nz, atoi(e)));
    // rotation of the work sequence between steps (n_rot tables, step n uses table n % n_rot)
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
        make_segments(G, F->TX, F->TY, n_cta, n_chunk, -(long long)r * (per_cta / n_rot), per[r], per_b[r]);
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
    StepParams &P = F->sp;
    P.G = G; P.T = g->T; P.segs = F->d_segs; P.seg_begin = F->d_seg_begin;
    P.n_rot = n_rot; P.seg_stride = (int)stride; P.n_cta = n_cta;
    P.step = g->d_step;
    P.nslots = F->nslots;
    P.XW = G.dpx + 8;
    P.TW = TW;
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
        for (int q = 0; q < 2; ++q) if (g->fused->h_maps[q]) cudaFreeHost(g->fused->h_maps[q]);
        if (g->fused->maps_done) cudaEventDestroy(g->fused->maps_done);
    }
    delete g->fused;
    g->fused = nullptr;
}

namespace {

// (re)builds one tensor-map table when the pointers it was built for changed.
//   which = 0: volumes A/B = fields / bufB, states = psiE/psiH;  which = 1: lam / lamB, lpsiE/lpsiH
int build_maps(fdtd_grid *g, int which, float *volA, float *volB, const float *ie, const float *im, cudaStream_t st)
{
    FusedState *F = g->fused;
    const Dims &G = g->G;
    const float **key = F->maps_key[which];
    if (key[0] == volA && key[1] == ie && key[2] == im) return FDTD_OK;
    const int PW = F->TX + 8, ROWS = F->TY + 2, XW = F->sp.XW;
    if (cudaEventSynchronize(F->maps_done) != cudaSuccess) { (void)cudaGetLastError(); }   // earlier upload finished
    CUtensorMap *H = F->h_maps[which];
    bool ok = true;
    float *bufs[2] = { volA, volB };
    for (int set = 0; set < 2; ++set)
        for (int c = 0; c < 6; ++c)
            ok &= encode3d(&H[TM_FIELD + set * 6 + c], bufs[set] + (long long)c * G.nc, G.nx, G.ny, G.nz, G.nx,
                           (long long)G.nx * G.ny, PW, ROWS);
    ok &= encode3d(&H[TM_IE], ie, G.nx, G.ny, G.nz, G.nx, (long long)G.nx * G.ny, PW, ROWS);
    ok &= encode3d(&H[TM_IM], im ? im : ie, G.nx, G.ny, G.nz, G.nx, (long long)G.nx * G.ny, PW, ROWS);
    if (G.d > 0) {
        for (int set = 0; set < 2; ++set)
            for (int fam = 0; fam < 2; ++fam) {
                const PsiSet &ps = which ? (fam ? g->lpsiH[set] : g->lpsiE[set]) : (fam ? g->psiH[set] : g->psiE[set]);
                // x axis arrays: (c=z,s=0) and (c=y,s=1); layout [nz][ny][2*dpx]
                const float *xa[2] = { ps.p[2][0], ps.p[1][1] };
                for (int q = 0; q < 2; ++q)
                    for (int view = 0; view < 2; ++view)
                        ok &= encode3d(&H[tm_psi(set, fam, q + 2 * view)], xa[q] + view * G.dpx, G.dpx, G.ny, G.nz,
                                       2 * G.dpx, (long long)2 * G.dpx * G.ny, XW, ROWS);
                // y axis arrays: (c=x,s=0) and (c=z,s=1); layout [nz][2*d][nx]
                const float *ya[2] = { ps.p[0][0], ps.p[2][1] };
                for (int q = 0; q < 2; ++q)
                    for (int view = 0; view < 2; ++view)
                        ok &= encode3d(&H[tm_psi(set, fam, 4 + q + 2 * view)], ya[q] + (long long)view * G.d * G.nx, G.nx,
                                       G.d, G.nz, G.nx, (long long)2 * G.d * G.nx, PW, ROWS);
                // z axis arrays: (c=y,s=0) and (c=x,s=1); layout [2*d][ny][nx]
                const float *za[2] = { ps.p[1][0], ps.p[0][1] };
                for (int q = 0; q < 2; ++q)
                    ok &= encode3d(&H[tm_psi(set, fam, 8 + q)], za[q], G.nx, G.ny, 2 * G.d, G.nx, (long long)G.nx * G.ny, PW, ROWS);
            }
    }
    if (!ok) return fdtd_fail(FDTD_ECUDA, "cuTensorMapEncodeTiled failed");
    cudaError_t e = cudaMemcpyAsync(F->d_maps[which], H, sizeof(CUtensorMap) * TM_COUNT, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaEventRecord(F->maps_done, st);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, std::string("tensor map upload: ") + cudaGetErrorString(e)); }
    key[0] = volA; key[1] = ie; key[2] = im;
    return FDTD_OK;
}

}  // namespace

// run_steps lives in fdtd_api.cu; reached through small trampolines
int fdtd_run_steps_fwd(fdtd_grid *g, const std::string &key, int n_steps, int launches_per_step, cudaStream_t st,
                       void (*enqueue)(void *, cudaStream_t), void *ctx);
int fdtd_run_steps_bwd(fdtd_grid *g, const std::string &key, int n_steps, int launches_per_step, cudaStream_t st,
                       void (*enqueue)(void *, cudaStream_t), void *ctx);

namespace {
struct FwdCtx {
    fdtd_grid *g; StepParams P; bool recording; float *A; float *B;
};
void enqueue_fwd(void *vctx, cudaStream_t cs)
{
    FwdCtx *c = (FwdCtx *)vctx;
    fdtd_grid *g = c->g;
    FusedState *F = g->fused;
    { ProfScope p(g, fdtd_grid::PC_FUSED_FWD, cs);
      F->tile->launch_fwd(c->P, F->n_cta, F->smem, cs); }
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
    int rc = build_maps(g, 0, fields, F->bufB, inv_eps, inv_mu, st);
    if (rc) return rc;
    for (int q = 0; q < 2; ++q)
        if ((rc = g->zero_psi(g->psiE[q], st)) || (rc = g->zero_psi(g->psiH[q], st))) return rc;
    FwdCtx ctx{ g, F->sp, recording, fields, F->bufB };
    StepParams &P = ctx.P;
    P.maps = F->d_maps[0];
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
