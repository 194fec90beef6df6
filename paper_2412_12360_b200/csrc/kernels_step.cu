// kernels_step.cu -- fused z-marching step kernels of the hot path (DESIGN.md sections 7-8):
//
//   k_step<C, false, N4>  forward step : E update + H update + CPML psi + sources + detectors   (F1-F7)
//   k_step<C, true, N4>   adjoint step : transpose of the H update, then of the E update, adjoint CPML (B2+B5)
//   (N4 = true: the instance with the operands beyond the contract's path -- inv_mu, three inv_eps volumes, a conductivity)
//
// PAPER.md: Eq. 1-2 (L64-66) for the curl updates, L72 for the CPML, L78-84 for the VJP.
//
// Design
//   * ping-pong volumes: a launch reads buffer `par` and writes buffer `par^1`, so tiles are independent;
//   * the xy plane is cut into TX x TY tiles, a tile's z column into segments; a persistent CTA marches its
//     segments plane by plane (2.5-D blocking); the previous plane stays in its stage / in the ring;
//   * only the three arrays that are differenced in phase A (the H-type operand F) need neighbours: one
//     producer thread streams their boxes (one-cell halo, 16-byte aligned in x) global -> shared with TMA
//     (cp.async.bulk.tensor; the zero fill outside the grid IS the zero-pad wall convention R7) through a
//     ring of NST stages with full/empty mbarriers (a stage is released when its own plane is done: what the next
//     plane needs of it -- F at a thread's own cells -- travels in registers).  The E-type target, inv_eps and the x-slab CPML states
//     travel in the same stage (seven boxes plus four narrow ones); only the y / z slab CPML states (and inv_mu)
//     are read straight from global memory as float4 at a thread's own cells;
//   * consumer warps are 8 x 4 patches of float4 threads (128 B contiguous per patch row), so CPML slab
//     code is executed by the few warps that touch a slab.  Plane kk, phase A: the E-type update of plane
//     kk on the tile plus a +x halo column and a +y halo row (recomputed, not exchanged between CTAs),
//     result to global and to a shared ring; phase B: the H-type update of plane kk-1 from the phase-A
//     results of planes kk-1 (registers + ring) and kk (registers); one named barrier per plane;
//   * CPML: the time-recursive filter  p' = b p + a x,  c = (ik-1) x + p'  adds c to a difference.
//     Forward: x = the difference.  Adjoint: the filter acts on the operands before the difference (its
//     tables depend on the position along the difference axis) with the rescaled state
//     theta = (a/b) * lambda_psi, which obeys the same recursion; phase-B operands are filtered by the
//     thread that produces them in phase A and travel through the ring already filtered.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <utility>
#include <vector>

#include "fdtd_grid.h"
#include "fused_common.cuh"

using namespace fdtd;

namespace {

constexpr int MAX_SRC = FDTD_FUSED_MAX_SRC, MAX_DET = FDTD_FUSED_MAX_DET;
// timing experiments (wrong results): build with -DFDTD_TIMING_EXPERIMENTS and set FDTD_DBG to a bit mask:
// 1 no global stores, 2 no phase B, 4 no barrier, 8 load pipeline only, 16 no CPML, 32/64/128 no x/y/z slab code
#ifdef FDTD_TIMING_EXPERIMENTS
#define DBG(bit) (P.dbg & (bit))
#else
#define DBG(bit) 0
#endif
constexpr int MAX_ST = 8;               // upper bound of pipeline stages

struct StepParams {
    Dims G;
    Tables T;
    const CUtensorMap *maps;       // [set][6]: components of buffer `set`; [12]: inv_eps; [13 + set*4 + family*2 + a]: x-slab states
    const Segment *segs;           // [n_rot][seg_stride]
    const int *seg_begin;          // [n_rot][n_cta + 1]
    int n_rot, seg_stride, n_cta;
    float *buf[2];                 // ping-pong volumes, [6][nc] each
    const float *ie, *im;
    const float *sigma;            // N4 (reading R29): normalised conductivity volume or NULL.  With G.aniso (R30) `ie` is [3][nc]
    float *e2_out;                 // lossy adjoint step in the checkpointed sweep: lamE' before its scaling by Ca, [3][nc], or NULL
    PsiSet psiE[2], psiH[2];       // CPML states of the E-type / H-type update, ping-pong
    const int *step;               // the slot of the two-slot step counter this step reads
    int *step_next;                // the other slot: block 0 writes n + step_delta for the next step (or NULL)
    int step_delta;
    int nst;                       // pipeline stages
    int hold;                      // 1: a stage is released one plane late (the consumers stay one plane closer to the loads)
    int stage;                     // bytes of one stage: 7 boxes + 4 x-slab state boxes
    int xs_bytes, xs_pitch;        // x-slab state box [ROWS][2*dpx]: exact bytes (TMA transaction) and 128-byte aligned pitch
    unsigned long long *dbg_t;     // timing experiments only (FDTD_DBG_TIMES): per-CTA start / end globaltimer
    int dbg;                       // timing experiments only (FDTD_DBG): 1 no global stores, 2 no phase B, 4 no barrier
    int n_src, n_det, total_freq;
    int sEl, sEh, sHl, sHh, dEl, dEh, dHl, dHh;   // k ranges of the planes that hold E/H sources and E/H detectors
    SourceDev src[MAX_SRC];
    DetectorDev det[MAX_DET];
    const float *cs;
    // N3, peer stores (fdtd_halo_attach): the H-type result of my lowest / highest owned plane also goes straight into the
    // ghost plane of the neighbouring slab's volume, and my own ghost planes on attached sides are left to the neighbour
    int peer_on;                   // bit 0: a neighbour below is attached, bit 1: above
    int own_lo, own_hi;            // lowest / highest owned plane (local index)
    float *peer[2][2];             // [side][volume]: component 3 of the neighbour's ghost plane in its volume 0 / 1
    long long peer_nc[2];          // the neighbour's component stride
};

template <int TX4_, int TY_>
struct Cfg {
    static constexpr int TX4 = TX4_, TY = TY_, TX = 4 * TX4_;
    static constexpr int CW = TX4 + 1, RW = TY + 1;                     // float4 lanes per row / rows, halo included
    static constexpr int PCX = (CW + 7) / 8, PCY = (RW + 3) / 4;        // 8 x 4 thread patches
    static constexpr int NCW = PCX * PCY;                               // consumer warps
    static constexpr int THREADS = NCW * 32 + 32;
    static constexpr int PW = TX + 8, ROWS = TY + 2;
    static constexpr int ROWB = PW * 4;                                 // box row pitch in bytes
    static constexpr int BOX_BYTES = PW * ROWS * 4;                     // TMA transaction bytes of one box
    static constexpr int BOXE_BYTES = PW * (ROWS - 1) * 4;              // ... of an own-cell array of the step kernel (e, inv_eps): no row below the tile
    static constexpr int SLOT = (BOX_BYTES + 127) / 128 * 128;
    static constexpr int STAGE = 7 * SLOT;                               // F x3, e x3, inv_eps
    static constexpr int RP = 4 * CW;                                   // ring row pitch (floats)
    static constexpr int RING_ARR = RW * RP;                            // floats of one ring array
    static constexpr int RING_SLOT = 4 * RING_ARR;                      // Yx, Yz, Xy, Xz
    static constexpr int RING_BYTES = (2 * RING_SLOT * 4 + 127) / 128 * 128;
    // inverse step kernel: three box shapes per stage (see k_inverse)
    static constexpr int BW = TX + 4, BROWS = TY + 1;                  // H' and E'(kk+1): my cells, minus-side halo threads included
    static constexpr int BOXB_BYTES = BW * BROWS * 4, SLOTB = (BOXB_BYTES + 127) / 128 * 128;
    static constexpr int BOXC_BYTES = TX * TY * 4, SLOTC = (BOXC_BYTES + 127) / 128 * 128;     // inv_eps, lamE': owned cells only
    static constexpr int ISTAGE = 3 * SLOT + 5 * SLOTB + 4 * SLOTC;
    static constexpr int IRING_BYTES = (2 * 3 * RING_ARR * 4 + 127) / 128 * 128;              // H_x, H_y, H_z, two planes
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
__device__ __forceinline__ float4 ld4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ void stg4(float *p, float4 v) { *reinterpret_cast<float4 *>(p) = v; }
// 1 / a to one unit in the last place (MUFU.RCP; the IEEE division's slow-path calls cost the step kernel its registers)
__device__ __forceinline__ float rcp1(float a) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ float4 rcp4(float4 a) { return make_float4(rcp1(a.x), rcp1(a.y), rcp1(a.z), rcp1(a.w)); }
__device__ __forceinline__ float4 fma4(float4 a, float4 b, float4 c)
{
    return make_float4(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y), fmaf(a.z, b.z, c.z), fmaf(a.w, b.w, c.w));
}
__device__ __forceinline__ float4 fma4(float a, float4 b, float4 c)
{
    return make_float4(fmaf(a, b.x, c.x), fmaf(a, b.y, c.y), fmaf(a, b.z, c.z), fmaf(a, b.w, c.w));
}

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

// slab-compact coordinate along an axis of length n with slab storage width w per side, or -1
__device__ __forceinline__ int slab_pos(int p, int n, int w) { return p < 0 || p >= n ? -1 : (p < w ? p : (p >= n - w ? p - (n - 2 * w) : -1)); }

// additive source contribution to component `comp` at cell (i,j,k) during this step
template <class PT>
__device__ __noinline__ float source_at(const PT &P, int n, int comp, int i, int j, int k)
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

// adjoint of the running DFT (B1) at the cells (i..i+3, j, k) of component `comp`: v += sum_f Gr cos - Gi sin, with the
// caller's phasor cotangents in det[].phasor (NULL: no cotangent for that detector)
__device__ __noinline__ float4 det_adjoint4(const StepParams &P, int n, int comp, float4 v, int i, int j, int k)
{
    for (int s = 0; s < P.n_det; ++s) {
        const DetectorDev &q = P.det[s];
        if (!q.phasor || !((q.mask >> comp) & 1)) continue;
        if (j < q.lo[1] || j >= q.hi[1] || k < q.lo[2] || k >= q.hi[2] || i + 3 < q.lo[0] || i >= q.hi[0]) continue;
        const int bx = q.hi[0] - q.lo[0], by = q.hi[1] - q.lo[1], bz = q.hi[2] - q.lo[2];
        const long long bc = (long long)bx * by * bz;
        const long long cell = ((long long)(k - q.lo[2]) * by + (j - q.lo[1])) * bx + (i - q.lo[0]);
        int ci = 0;
        for (int c = 0; c < comp; ++c) ci += (q.mask >> c) & 1;
        const float *csn = P.cs + ((long long)n * P.total_freq + q.cs_off) * 2;
        const bool whole = i >= q.lo[0] && i + 3 < q.hi[0];
        for (int f = 0; f < q.n_freq; ++f) {
            const float c = __ldg(csn + 2 * f), sn = __ldg(csn + 2 * f + 1);
            const float2 *ph = reinterpret_cast<const float2 *>(q.phasor) + ((long long)f * q.ncomp + ci) * bc + cell;
            if (whole && (reinterpret_cast<unsigned long long>(ph) & 15ull) == 0) {
                const float4 a = ldg4(reinterpret_cast<const float *>(ph)), b = ldg4(reinterpret_cast<const float *>(ph + 2));
                v.x += a.x * c - a.y * sn; v.y += a.z * c - a.w * sn;
                v.z += b.x * c - b.y * sn; v.w += b.z * c - b.w * sn;
            } else {
                float add[4] = { 0.f, 0.f, 0.f, 0.f };
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    if (i + e < q.lo[0] || i + e >= q.hi[0]) continue;
                    const float2 Gq = __ldg(ph + e);
                    add[e] = Gq.x * c - Gq.y * sn;
                }
                v.x += add[0]; v.y += add[1]; v.z += add[2]; v.w += add[3];
            }
        }
    }
    return v;
}

// exact per-plane tests behind the coarse k ranges of the parameters (sEl..dHh span all sources / detectors of a
// family: with two detector planes far apart every plane in between would otherwise pay for the box tests per cell)
template <class PT>
__device__ __forceinline__ int src_mask(const PT &P, int k)      // bit c: some source of component c has cells on plane k
{
    int m = 0;
    for (int s = 0; s < P.n_src; ++s) if (k >= P.src[s].lo[2] && k < P.src[s].hi[2]) m |= 1 << P.src[s].comp;
    return m;
}
__device__ __forceinline__ int det_mask(const StepParams &P, int k, bool need_cotangent)   // bit c: a detector of component c on plane k
{
    int m = 0;
    for (int s = 0; s < P.n_det; ++s)
        if (k >= P.det[s].lo[2] && k < P.det[s].hi[2] && (!need_cotangent || P.det[s].phasor != nullptr)) m |= P.det[s].mask;
    return m;
}

__device__ __forceinline__ float f4get(const float4 &v, int q) { return q == 0 ? v.x : (q == 1 ? v.y : (q == 2 ? v.z : v.w)); }

// adds the sources of component `comp` to the float4 of cells (i..i+3, j, k); rare planes only
template <class PT>
__device__ __noinline__ float4 add_sources4(const PT &P, int n, int comp, float4 v, int i, int j, int k)
{
    v.x += source_at(P, n, comp, i + 0, j, k);
    v.y += source_at(P, n, comp, i + 1, j, k);
    v.z += source_at(P, n, comp, i + 2, j, k);
    v.w += source_at(P, n, comp, i + 3, j, k);
    return v;
}
// running DFT of component `comp` at the cells (i..i+3, j, k): two float4 read-modify-writes per frequency when the
// four cells are inside the box and their phasors 16-byte aligned, cell by cell otherwise
__device__ __noinline__ void detect_comp4(const StepParams &P, int n, int comp, float4 v, int i, int j, int k)
{
    for (int s = 0; s < P.n_det; ++s) {
        const DetectorDev &q = P.det[s];
        if (!((q.mask >> comp) & 1)) continue;
        if (j < q.lo[1] || j >= q.hi[1] || k < q.lo[2] || k >= q.hi[2] || i + 3 < q.lo[0] || i >= q.hi[0]) continue;
        const int bx = q.hi[0] - q.lo[0], by = q.hi[1] - q.lo[1], bz = q.hi[2] - q.lo[2];
        const long long bc = (long long)bx * by * bz;
        const long long cell = ((long long)(k - q.lo[2]) * by + (j - q.lo[1])) * bx + (i - q.lo[0]);
        int ci = 0;
        for (int c = 0; c < comp; ++c) ci += (q.mask >> c) & 1;
        const float *csn = P.cs + ((long long)n * P.total_freq + q.cs_off) * 2;
        const bool whole = i >= q.lo[0] && i + 3 < q.hi[0];
        for (int f = 0; f < q.n_freq; ++f) {
            const float c = __ldg(csn + 2 * f), sn = __ldg(csn + 2 * f + 1);
            float2 *ph = reinterpret_cast<float2 *>(q.phasor) + ((long long)f * q.ncomp + ci) * bc + cell;
            if (whole && (reinterpret_cast<unsigned long long>(ph) & 15ull) == 0) {
                float4 a = ld4(reinterpret_cast<const float *>(ph)), b = ld4(reinterpret_cast<const float *>(ph + 2));
                a.x += v.x * c; a.y -= v.x * sn; a.z += v.y * c; a.w -= v.y * sn;
                b.x += v.z * c; b.y -= v.z * sn; b.z += v.w * c; b.w -= v.w * sn;
                stg4(reinterpret_cast<float *>(ph), a); stg4(reinterpret_cast<float *>(ph + 2), b);
            } else {
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    if (i + e < q.lo[0] || i + e >= q.hi[0]) continue;
                    float2 acc = ph[e];
                    const float x = f4get(v, e);
                    acc.x += x * c; acc.y -= x * sn;
                    ph[e] = acc;
                }
            }
        }
    }
}
__device__ __forceinline__ void detect4(const StepParams &P, int n, int family, int dm, float4 vx, float4 vy, float4 vz, int i, int j, int k)
{
    if ((dm >> (3 * family)) & 1) detect_comp4(P, n, 3 * family + 0, vx, i, j, k);
    if ((dm >> (3 * family)) & 2) detect_comp4(P, n, 3 * family + 1, vy, i, j, k);
    if ((dm >> (3 * family)) & 4) detect_comp4(P, n, 3 * family + 2, vz, i, j, k);
}

// ================================================================================================
// The step kernel.  Names follow the forward step: "F" is the H-type operand of phase A, "e" the
// E-type target, "v" the phase-A result that phase B differences, "h" the H-type target.
//   forward : e' = e + S ie curl-(F = H)            v = e'            h' = h - S im curl+(v)
//   adjoint : e' = e - S curl-(F = im lamH)         v = S ie e'       h' = h + im curl+(v)     (h = im lamH)
// curl with CPML: t_x = Dy_z - Dz_y, t_y = Dz_x - Dx_z, t_z = Dx_y - Dy_x, where D<a>_<c> is the
// (filtered) difference of component c along axis a; its state array is
//   Dy_z p[0][0]   Dz_y p[0][1]   Dz_x p[1][0]   Dx_z p[1][1]   Dx_y p[2][0]   Dy_x p[2][1].
// ================================================================================================
#ifndef FDTD_PF_MODE
#define FDTD_PF_MODE 2
#endif
__device__ __forceinline__ void pf_l2(const float *p)
{
#if FDTD_PF_MODE == 2
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
#elif FDTD_PF_MODE == 1
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
#endif
}
__device__ __forceinline__ void pf_l1(const float *p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
#ifndef FDTD_PF_DIST
#define FDTD_PF_DIST 1
#endif

// N4 = true: the instance that takes the operands beyond the contract's path, read by LDG at a thread's own cells: an inv_mu
// volume (P.im), three inv_eps volumes (G.aniso), a conductivity (P.sigma).  The contract's path runs N4 = false.
template <class C, bool ADJ, bool N4>
__global__ void __launch_bounds__(C::THREADS, 1) k_step(const __grid_constant__ StepParams P)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const Dims &G = P.G;
    const uint32_t stage_base = smem_u32(smem);
    const uint32_t ring_base = stage_base + (uint32_t)P.nst * P.stage;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)P.nst * P.stage + C::RING_BYTES);
    uint64_t *empty = full + MAX_ST;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int FA = ADJ ? 1 : 0, FB = ADJ ? 0 : 1;   // CPML family (tables, states) of phase A / phase B
    const int nst = P.nst;
    // programmatic dependent launch: the next step kernel may be placed on an SM as soon as this CTA has left it;
    // its prologue (tables, barriers) touches nothing a step writes and it waits below before it reads the counter
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    // CPML tables of the slab cells in shared memory, indexed by slab-compact coordinate:
    // [family][b, a, 1/kappa - 1][x: 2 dpx | y: 2 d | z: 2 d]
    float *tabs = reinterpret_cast<float *>(empty + MAX_ST);
    const uint32_t tab_base = smem_u32(tabs);
    const int YO = 2 * G.dpx, ZO = 2 * G.dpx + 2 * G.d, TL = 2 * G.dpx + 4 * G.d;
#define TB1(F, kind, off) lds1(tab_base + (uint32_t)((((F) * 3 + (kind)) * TL + (off)) * 4))
#define TB4(F, kind, off) lds4(tab_base + (uint32_t)((((F) * 3 + (kind)) * TL + (off)) * 4))
    for (int e = threadIdx.x; e < 6 * TL; e += blockDim.x) {
        const int fk = e / TL, q = e - fk * TL, fam = fk / 3, kind = fk - 3 * fam;
        const int ax = q < YO ? 0 : (q < ZO ? 1 : 2);
        const int sc = q - (ax == 0 ? 0 : (ax == 1 ? YO : ZO));
        const int w = ax == 0 ? G.dpx : G.d, N = ax == 0 ? G.nx : (ax == 1 ? G.ny : G.nz);
        // (on a z-slab sub-grid the entries between the zl low and the zh high planes are never read: clamp)
        const int pos = min(max(sc < w ? sc : N - 2 * w + sc, 0), N - 1);
        const float *src = kind == 0 ? P.T.b[fam][ax] : (kind == 1 ? P.T.a[fam][ax] : P.T.ik[fam][ax]);
        tabs[e] = __ldg(src + pos) - (kind == 2 ? 1.f : 0.f);
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < nst; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], C::NCW); }
        fence_mbar_init();
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");   // everything the previous launches wrote is visible from here on
    const int n = *P.step;
    const int par = (n + (ADJ ? 1 : 0)) & 1;       // forward step n reads buffer n&1; reverse step n reads (n+1)&1
    if (threadIdx.x == 0) {
        if (blockIdx.x == 0 && P.step_next) *P.step_next = n + P.step_delta;
        if (P.dbg_t) { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); P.dbg_t[2 * blockIdx.x] = t; }
    }
    __syncthreads();

    const int rot = n % P.n_rot;
    const int *sb = P.seg_begin + rot * (P.n_cta + 1);
    const Segment *segs = P.segs + (size_t)rot * P.seg_stride;
    const int seg_lo = sb[blockIdx.x], seg_hi = sb[blockIdx.x + 1];

    // ============================================================================== producer
    if (warp == C::NCW) {
        if (lane != 0) return;
        const CUtensorMap *M = P.maps + par * 6;
        const CUtensorMap *Mie = P.maps + 12;
        int s = 0, use = 0;
        for (int sg = seg_lo; sg < seg_hi; ++sg) {
            const Segment S = segs[sg];
            const int x = S.i0 - 4, y = S.j0 - 1;
            for (int kk = S.k0 - 1; kk <= S.k1; ++kk) {
                if (use > 0) mbar_wait(&empty[s], (use - 1) & 1);
                uint64_t *fb = &full[s];
                uint8_t *st = smem + (size_t)s * P.stage;
                const bool prolog = kk == S.k0 - 1;
                const bool xs = G.d > 0 && !prolog;
                mbar_expect_tx(fb, 3u * C::BOX_BYTES + (prolog ? 0u : 4u * C::BOXE_BYTES) + (xs ? 4u * P.xs_bytes : 0u));
                tma_load_3d(st, M + 3, x, y, kk, fb);
                tma_load_3d(st + C::SLOT, M + 4, x, y, kk, fb);
                tma_load_3d(st + 2 * C::SLOT, M + 5, x, y, kk, fb);
                if (!prolog) {
                    // e and inv_eps are read at a thread's own cells only (rows j0 .. j0 + TY): their boxes start one row later
                    tma_load_3d(st + 3 * C::SLOT, M + 0, x, y + 1, kk, fb);
                    tma_load_3d(st + 4 * C::SLOT, M + 1, x, y + 1, kk, fb);
                    tma_load_3d(st + 5 * C::SLOT, M + 2, x, y + 1, kk, fb);
                    tma_load_3d(st + 6 * C::SLOT, Mie, x, y + 1, kk, fb);
                }
                if (xs) {      // phase A states of plane kk; phase B states of plane kk-1 (forward) / kk (adjoint)
                    const CUtensorMap *MA = P.maps + 13 + par * 4 + FA * 2, *MB = P.maps + 13 + par * 4 + FB * 2;
                    uint8_t *sx0 = st + 7 * C::SLOT;
                    const int kb = ADJ ? kk : kk - 1;
                    tma_load_3d(sx0, MA, 0, y, kk, fb);
                    tma_load_3d(sx0 + P.xs_pitch, MA + 1, 0, y, kk, fb);
                    tma_load_3d(sx0 + 2 * P.xs_pitch, MB, 0, y, kb, fb);
                    tma_load_3d(sx0 + 3 * P.xs_pitch, MB + 1, 0, y, kb, fb);
                }
                if (++s == nst) { s = 0; ++use; }
            }
        }
        return;
    }

    // ============================================================================== consumers
    // 8 x 4 patches of float4 threads; threads beyond the tile duplicate the last column / row (they never store)
    const int tx0 = (warp % C::PCX) * 8 + (lane & 7), ty0 = (warp / C::PCX) * 4 + (lane >> 3);
    const bool dup = tx0 >= C::CW || ty0 >= C::RW;
    const int tx = min(tx0, C::CW - 1), ty = min(ty0, C::RW - 1);
    const bool inner = !dup && ty < C::TY && tx < C::TX4;         // not a halo thread
    const uint32_t o_own = ((1 + ty) * C::PW + 4 + 4 * tx) * 4;   // my first cell inside a box (bytes)
    const uint32_t r_own = (ty * C::RP + 4 * tx) * 4;             // ... inside a ring array
    float *dst = P.buf[par ^ 1];
    const PsiSet &qAi = ADJ ? P.psiH[par] : P.psiE[par], &qAo = ADJ ? P.psiH[par ^ 1] : P.psiE[par ^ 1];
    const PsiSet &qBi = ADJ ? P.psiE[par] : P.psiH[par], &qBo = ADJ ? P.psiE[par ^ 1] : P.psiH[par ^ 1];
    const float S = G.S;
    const long long nc = G.nc;
    const int plane = G.ny * G.nx;
    const bool pml = G.d > 0 && !DBG(16);
    const bool has_mu = N4 && P.im != nullptr;      // (the N4 = false instance is launched without inv_mu)
    const int pz = plane, py = 2 * G.d * G.nx, px = G.ny * 2 * G.dpx;      // plane pitch of the z / y / x state arrays

    const float4 Z4 = splat(0.f);

    int st_i = 0;                 // pipeline stage of the next plane
    uint32_t st_ph = 0;           // its full-barrier parity
    uint32_t st_off = 0;          // st_i * STAGE
    float4 cgx = Z4, cgy = Z4, cZx = Z4, cZy = Z4;   // adjoint: z-filtered operands of the previous plane at my cells
    // forward: F of the previous plane at my cells (= the H-type target of phase B) travels in registers, so a stage is
    // released as soon as its own plane is done and the ring of NST stages keeps one more plane in flight
    float4 pFx = Z4, pFy = Z4, pFz = Z4;
    int pv_i = 0;                 // P.hold: the stage of the previous plane
    for (int sg = seg_lo; sg < seg_hi; ++sg) {
        const Segment Sg = segs[sg];
        const int i = Sg.i0 + 4 * tx, j = Sg.j0 + ty;
        const bool ing = i < G.nx && j < G.ny;                      // my cells are inside the grid
        const bool own_ok = inner && ing;
        const int own_xy = j * G.nx + i;
        // slab-compact coordinates of my cells and (adjoint) of my -x / -y neighbours; -1: not in a slab
        const int sx = (pml && ing && !DBG(32)) ? slab_pos(i, G.nx, G.dpx) : -1;
        const int sy = (pml && ing && !DBG(64)) ? slab_pos(j, G.ny, G.d) : -1;
        const int sxm = (ADJ && pml && ing && !DBG(32)) ? slab_pos(i - 1, G.nx, G.dpx) : -1;
        const int sym = (ADJ && pml && ing && !DBG(64)) ? slab_pos(j - 1, G.ny, G.d) : -1;
        const bool slab_xy = __any_sync(0xffffffffu, (sx & sy & sxm & sym) >= 0);   // this warp runs x / y slab code
        const int oy = sy * G.nx + i, oym = sym * G.nx + i;                          // + k * py
        const int ox = j * (2 * G.dpx) + sx, oxm = j * (2 * G.dpx) + sxm;           // + k * px
        const uint32_t xo = ((1 + ty) * 2 * G.dpx + sx) * 4, xom = ((1 + ty) * 2 * G.dpx + sxm) * 4;   // inside an x-slab state box
        const int k1 = Sg.k1;

        // ---------------------------------------------------------------- one plane (phase A of kk, phase B of kk-1)
        auto plane_step = [&](const int kk, const bool doB) {
            const int zs = (pml && !DBG(128)) ? zslab_pos(G, kk) : -1;
            if (N4 && ing && kk < G.nz) {      // the operands that come by LDG at my cells: on their way while the stage lands
                const float *q = P.ie + (kk * (G.ny * G.nx) + own_xy);
                if (G.aniso) { pf_l1(q + G.nc); pf_l1(q + 2 * G.nc); }
                if (P.sigma) pf_l1(P.sigma + (kk * (G.ny * G.nx) + own_xy));
            }
            if (has_mu && own_ok && doB) pf_l1(P.im + ((kk - 1) * (G.ny * G.nx) + own_xy));     // phase B's inv_mu, likewise
            mbar_wait(&full[st_i], st_ph);
            const uint32_t so = stage_base + st_off + o_own;
            if (ADJ && kk >= P.dEl && kk < P.dEh && !dup) {
                // B1 for E-component detectors: the cotangents are added to lamE in the stage, at my cells, before
                // anything is live in registers (lamE is only ever read at a thread's own cells)
                const int dm = det_mask(P, kk, true);
                for (int c = 0; c < 3; ++c) {
                    if (!((dm >> c) & 1)) continue;
                    const uint32_t se = so - C::ROWB + (3 + c) * C::SLOT;
                    sts4(se, det_adjoint4(P, n, c, lds4(se), i, j, kk));
                }
                if (dm & 7) fence_proxy_async();
            }
            const uint32_t xs0 = stage_base + st_off + 7 * C::SLOT; // x-slab state boxes of this stage
            const float4 fx = lds4(so), fy = lds4(so + C::SLOT), fz = lds4(so + 2 * C::SLOT);
            const float4 fx_my = lds4(so - C::ROWB), fz_my = lds4(so + 2 * C::SLOT - C::ROWB);
            const float fy_mx = lds1(so + C::SLOT - 4), fz_mx = lds1(so + 2 * C::SLOT - 4);

            const bool wr = own_ok && kk < k1 && !DBG(1);                 // I own these cells: write the result and the phase-A states
            const int off = kk * plane + own_xy;
            const int oz = zs * pz + own_xy;
            const uint32_t rgA = ring_base + (uint32_t)(kk & 1) * (C::RING_SLOT * 4) + r_own;
            // plane nz (the zero wall behind the last plane) has no CPML states: all its inputs are zero
            const bool kin = kk < G.nz;
            const bool pf = kk + FDTD_PF_DIST < G.nz;                     // L2 prefetch of the states two planes ahead stays inside the arrays
            const int sxk = kin ? sx : -1, syk = kin ? sy : -1, sxmk = kin ? sxm : -1, symk = kin ? sym : -1;
            // ------------------------------------------------------------ phase A: E-type update of plane kk
            float4 Dy_z = fz - fz_my, Dy_x = fx - fx_my;
            float4 Dx_y = dminus_x(fy, fy_mx), Dx_z = dminus_x(fz, fz_mx);
            float4 Dz_x, Dz_y;
            if (pml && ing) {
                const int zs2 = zslab_pos(G, kk + FDTD_PF_DIST);
                if (zs2 >= 0) {
                    const int q = zs2 * pz + own_xy;
                    pf_l2(qAi.p[1][0] + q); pf_l2(qAi.p[0][1] + q); pf_l2(qBi.p[1][0] + q); pf_l2(qBi.p[0][1] + q);
                }
            }
            if (!ADJ) {
                Dz_x = fx - pFx; Dz_y = fy - pFy;
                if (slab_xy || zs >= 0) {
                    if (zs >= 0 && ing) {
                        const float b = TB1(FA, 0, ZO + zs), a = TB1(FA, 1, ZO + zs), km = TB1(FA, 2, ZO + zs);
                        float4 p0, p1;
                        Dz_x = Dz_x + cpml4(b, a, km, ldg4(qAi.p[1][0] + oz), Dz_x, p0);
                        Dz_y = Dz_y + cpml4(b, a, km, ldg4(qAi.p[0][1] + oz), Dz_y, p1);
                        if (wr) { stg4(qAo.p[1][0] + oz, p0); stg4(qAo.p[0][1] + oz, p1); }
                    }
                    if (syk >= 0) {
                        const float b = TB1(FA, 0, YO + sy), a = TB1(FA, 1, YO + sy), km = TB1(FA, 2, YO + sy);
                        const int q = kk * py + oy;
                        float4 p0, p1;
                        Dy_z = Dy_z + cpml4(b, a, km, ldg4(qAi.p[0][0] + q), Dy_z, p0);
                        Dy_x = Dy_x + cpml4(b, a, km, ldg4(qAi.p[2][1] + q), Dy_x, p1);
                        if (pf) { pf_l2(qAi.p[0][0] + q + FDTD_PF_DIST * py); pf_l2(qAi.p[2][1] + q + FDTD_PF_DIST * py); }
                        if (wr) { stg4(qAo.p[0][0] + q, p0); stg4(qAo.p[2][1] + q, p1); }
                    }
                    if (sxk >= 0) {
                        const float4 b = TB4(FA, 0, sx), a = TB4(FA, 1, sx), km = TB4(FA, 2, sx);
                        const int q = kk * px + ox;
                        float4 p0, p1;
                        Dx_y = Dx_y + cpml4(b, a, km, lds4(xs0 + xo), Dx_y, p0);
                        Dx_z = Dx_z + cpml4(b, a, km, lds4(xs0 + P.xs_pitch + xo), Dx_z, p1);
                        if (wr) { stg4(qAo.p[2][0] + q, p0); stg4(qAo.p[1][1] + q, p1); }
                    }
                }
            } else {
                float4 gx = fx, gy = fy;                       // z operands at plane kk, filtered
                if (slab_xy || zs >= 0) {
                    if (zs >= 0 && ing) {
                        const float b = TB1(FA, 0, ZO + zs), a = TB1(FA, 1, ZO + zs), km = TB1(FA, 2, ZO + zs);
                        float4 p0, p1;
                        gx = fx + cpml4(b, a, km, ldg4(qAi.p[1][0] + oz), fx, p0);
                        gy = fy + cpml4(b, a, km, ldg4(qAi.p[0][1] + oz), fy, p1);
                        if (wr) { stg4(qAo.p[1][0] + oz, p0); stg4(qAo.p[0][1] + oz, p1); }
                    }
                    if (syk >= 0) {
                        const float b = TB1(FA, 0, YO + sy), a = TB1(FA, 1, YO + sy), km = TB1(FA, 2, YO + sy);
                        const int q = kk * py + oy;
                        float4 p0, p1;
                        Dy_z = Dy_z + cpml4(b, a, km, ldg4(qAi.p[0][0] + q), fz, p0);
                        Dy_x = Dy_x + cpml4(b, a, km, ldg4(qAi.p[2][1] + q), fx, p1);
                        if (pf) { pf_l2(qAi.p[0][0] + q + FDTD_PF_DIST * py); pf_l2(qAi.p[2][1] + q + FDTD_PF_DIST * py); }
                        if (wr) { stg4(qAo.p[0][0] + q, p0); stg4(qAo.p[2][1] + q, p1); }
                    }
                    if (symk >= 0) {
                        const float b = TB1(FA, 0, YO + sym), a = TB1(FA, 1, YO + sym), km = TB1(FA, 2, YO + sym);
                        const int q = kk * py + oym;
                        float4 p0, p1;
                        Dy_z = Dy_z - cpml4(b, a, km, ldg4(qAi.p[0][0] + q), fz_my, p0);
                        Dy_x = Dy_x - cpml4(b, a, km, ldg4(qAi.p[2][1] + q), fx_my, p1);
                        if (pf && syk < 0) { pf_l2(qAi.p[0][0] + q + FDTD_PF_DIST * py); pf_l2(qAi.p[2][1] + q + FDTD_PF_DIST * py); }
                    }
                    if (sxk >= 0 || sxmk >= 0) {
                        float4 cy = Z4, cz = Z4;
                        float ly = 0.f, lz = 0.f;
                        if (sxk >= 0) {
                            const float4 b = TB4(FA, 0, sx), a = TB4(FA, 1, sx), km = TB4(FA, 2, sx);
                            const int q = kk * px + ox;
                            float4 p0, p1;
                            cy = cpml4(b, a, km, lds4(xs0 + xo), fy, p0);
                            cz = cpml4(b, a, km, lds4(xs0 + P.xs_pitch + xo), fz, p1);
                            if (wr) { stg4(qAo.p[2][0] + q, p0); stg4(qAo.p[1][1] + q, p1); }
                        }
                        if (sxmk >= 0) {
                            const float b = TB1(FA, 0, sxm), a = TB1(FA, 1, sxm), km = TB1(FA, 2, sxm);
                            const int q = kk * px + oxm;
                            ly = cpml1(b, a, km, lds1(xs0 + xom), fy_mx);
                            lz = cpml1(b, a, km, lds1(xs0 + P.xs_pitch + xom), fz_mx);
                        }
                        Dx_y = Dx_y + dminus_x(cy, ly);
                        Dx_z = Dx_z + dminus_x(cz, lz);
                    }
                }
                Dz_x = gx - cgx; Dz_y = gy - cgy;
                cgx = gx; cgy = gy;
            }
            const float4 tEx = Dy_z - Dz_y, tEy = Dz_x - Dx_z, tEz = Dx_y - Dy_x;
            const uint32_t soe = so - C::ROWB;           // my cells inside a box of e / inv_eps (no row below the tile)
            const float4 ex = lds4(soe + 3 * C::SLOT), ey = lds4(soe + 4 * C::SLOT), ez = lds4(soe + 5 * C::SLOT);
            const float4 sie = S * lds4(soe + 6 * C::SLOT);
            // N4: one inv_eps volume per component (R30: the stage holds component x, y and z come by LDG at my cells) and / or
            // a conductivity (R29: E' = Ca E + Cb S ie bracket, beta = sigma S ie / 2, Ca = (1 - beta) / (1 + beta), Cb = 1 / (1 + beta))
            const bool n4 = N4 && (G.aniso || P.sigma != nullptr);
            float4 siy = sie, siz = sie, six = sie, cax = splat(1.f), cay = cax, caz = cax;
            if (n4) {
                const bool ld_ok = ing && kin;
                if (G.aniso && ld_ok) { siy = S * ldg4(P.ie + nc + off); siz = S * ldg4(P.ie + 2 * nc + off); }
                if (N4 && P.sigma) {
                    const float4 hs = ld_ok ? 0.5f * ldg4(P.sigma + off) : Z4;
                    const float4 bx = hs * six, by = hs * siy, bz = hs * siz;
                    const float4 cbx = rcp4(splat(1.f) + bx), cby = rcp4(splat(1.f) + by), cbz = rcp4(splat(1.f) + bz);
                    cax = (splat(1.f) - bx) * cbx; cay = (splat(1.f) - by) * cby; caz = (splat(1.f) - bz) * cbz;
                    six = six * cbx; siy = siy * cby; siz = siz * cbz;
                }
            }
            float4 e2x, e2y, e2z, v2x, v2y, v2z;
            if (ADJ) {
                e2x = fma4(-S, tEx, ex); e2y = fma4(-S, tEy, ey); e2z = fma4(-S, tEz, ez);
                if (n4) { v2x = six * e2x; v2y = siy * e2y; v2z = siz * e2z; }
                else { v2x = sie * e2x; v2y = sie * e2y; v2z = sie * e2z; }
            } else {
                if (n4) { e2x = fma4(cax, ex, six * tEx); e2y = fma4(cay, ey, siy * tEy); e2z = fma4(caz, ez, siz * tEz); }
                else { e2x = fma4(sie, tEx, ex); e2y = fma4(sie, tEy, ey); e2z = fma4(sie, tEz, ez); }
                if (kk >= P.sEl && kk < P.sEh) {
                    const int sm = src_mask(P, kk);
                    if (sm & 1) e2x = add_sources4(P, n, 0, e2x, i, j, kk);
                    if (sm & 2) e2y = add_sources4(P, n, 1, e2y, i, j, kk);
                    if (sm & 4) e2z = add_sources4(P, n, 2, e2z, i, j, kk);
                }
                v2x = e2x; v2y = e2y; v2z = e2z;
            }
            if (wr) {
                float *o = dst + off;
                if (ADJ && N4 && P.sigma) {    // lamE of the earlier step is Ca lamE'; the checkpointed sweep's gradient wants lamE' itself
                    if (P.e2_out) { float *q = P.e2_out + off; stg4(q, e2x); stg4(q + nc, e2y); stg4(q + 2 * nc, e2z); }
                    stg4(o, cax * e2x); stg4(o + nc, cay * e2y); stg4(o + 2 * nc, caz * e2z);
                } else {
                    stg4(o, e2x); stg4(o + nc, e2y); stg4(o + 2 * nc, e2z);
                }
                if (!ADJ && kk >= P.dEl && kk < P.dEh) detect4(P, n, 0, det_mask(P, kk, false), e2x, e2y, e2z, i, j, kk);
            }
            float4 Yx = v2x, Yz = v2z, Xy = v2y, Xz = v2z, Zx = v2x, Zy = v2y;
            if (ADJ && (slab_xy || zs >= 0)) {       // phase-B operands are filtered where they are produced
                if (zs >= 0 && ing) {
                    const float b = TB1(FB, 0, ZO + zs), a = TB1(FB, 1, ZO + zs), km = TB1(FB, 2, ZO + zs);
                    float4 p0, p1;
                    Zx = v2x + cpml4(b, a, km, ldg4(qBi.p[1][0] + oz), v2x, p0);
                    Zy = v2y + cpml4(b, a, km, ldg4(qBi.p[0][1] + oz), v2y, p1);
                    if (wr) { stg4(qBo.p[1][0] + oz, p0); stg4(qBo.p[0][1] + oz, p1); }
                }
                if (syk >= 0) {
                    const float b = TB1(FB, 0, YO + sy), a = TB1(FB, 1, YO + sy), km = TB1(FB, 2, YO + sy);
                    const int q = kk * py + oy;
                    float4 p0, p1;
                    Yz = v2z + cpml4(b, a, km, ldg4(qBi.p[0][0] + q), v2z, p0);
                    Yx = v2x + cpml4(b, a, km, ldg4(qBi.p[2][1] + q), v2x, p1);
                    if (pf) { pf_l2(qBi.p[0][0] + q + FDTD_PF_DIST * py); pf_l2(qBi.p[2][1] + q + FDTD_PF_DIST * py); }
                    if (wr) { stg4(qBo.p[0][0] + q, p0); stg4(qBo.p[2][1] + q, p1); }
                }
                if (sxk >= 0) {
                    const float4 b = TB4(FB, 0, sx), a = TB4(FB, 1, sx), km = TB4(FB, 2, sx);
                    const int q = kk * px + ox;
                    float4 p0, p1;
                    Xy = v2y + cpml4(b, a, km, lds4(xs0 + 2 * P.xs_pitch + xo), v2y, p0);
                    Xz = v2z + cpml4(b, a, km, lds4(xs0 + 3 * P.xs_pitch + xo), v2z, p1);
                    if (wr) { stg4(qBo.p[2][0] + q, p0); stg4(qBo.p[1][1] + q, p1); }
                }
            }
            sts4(rgA, Yx); sts4(rgA + C::RING_ARR * 4, Yz); sts4(rgA + 2 * C::RING_ARR * 4, Xy);
            if (ADJ) sts4(rgA + 3 * C::RING_ARR * 4, Xz);
            // ---------------------------------------------------------------- phase B: H-type update of plane kk-1
            if (own_ok && doB && !DBG(2)) {
                const int km1 = kk - 1;
                const uint32_t rgB = ring_base + (uint32_t)(km1 & 1) * (C::RING_SLOT * 4) + r_own;
                const float4 Yx_py = lds4(rgB + C::RP * 4), Yz_py = lds4(rgB + (C::RING_ARR + C::RP) * 4);
                const float Xy_px = lds1(rgB + (2 * C::RING_ARR + 4) * 4);
                const float Xz_px = lds1(rgB + ((ADJ ? 3 : 1) * C::RING_ARR + 4) * 4);
                const float4 oYx = lds4(rgB), oYz = lds4(rgB + C::RING_ARR * 4), oXy = lds4(rgB + 2 * C::RING_ARR * 4);
                const float4 oXz = ADJ ? lds4(rgB + 3 * C::RING_ARR * 4) : oYz;
                float4 Dy_z = Yz_py - oYz, Dy_x = Yx_py - oYx;
                float4 Dz_y = Zy - (ADJ ? cZy : oXy), Dz_x = Zx - (ADJ ? cZx : oYx);
                float4 Dx_z = dplus_x(oXz, Xz_px), Dx_y = dplus_x(oXy, Xy_px);
                const int offm = off - plane;
                const int zsm = (!ADJ && pml && !DBG(128)) ? zslab_pos(G, km1) : -1;
                if (!ADJ && (slab_xy || zsm >= 0)) {
                    if (zsm >= 0) {
                        const float b = TB1(FB, 0, ZO + zsm), a = TB1(FB, 1, ZO + zsm), km = TB1(FB, 2, ZO + zsm);
                        const int q = zsm * pz + own_xy;
                        float4 p0, p1;
                        Dz_x = Dz_x + cpml4(b, a, km, ldg4(qBi.p[1][0] + q), Dz_x, p0);
                        Dz_y = Dz_y + cpml4(b, a, km, ldg4(qBi.p[0][1] + q), Dz_y, p1);
                        stg4(qBo.p[1][0] + q, p0); stg4(qBo.p[0][1] + q, p1);
                    }
                    if (sy >= 0) {
                        const float b = TB1(FB, 0, YO + sy), a = TB1(FB, 1, YO + sy), km = TB1(FB, 2, YO + sy);
                        const int q = km1 * py + oy;
                        float4 p0, p1;
                        Dy_z = Dy_z + cpml4(b, a, km, ldg4(qBi.p[0][0] + q), Dy_z, p0);
                        Dy_x = Dy_x + cpml4(b, a, km, ldg4(qBi.p[2][1] + q), Dy_x, p1);
                        if (pf) { pf_l2(qBi.p[0][0] + q + FDTD_PF_DIST * py); pf_l2(qBi.p[2][1] + q + FDTD_PF_DIST * py); }
                        stg4(qBo.p[0][0] + q, p0); stg4(qBo.p[2][1] + q, p1);
                    }
                    if (sx >= 0) {
                        const float4 b = TB4(FB, 0, sx), a = TB4(FB, 1, sx), km = TB4(FB, 2, sx);
                        const int q = km1 * px + ox;
                        float4 p0, p1;
                        Dx_y = Dx_y + cpml4(b, a, km, lds4(xs0 + 2 * P.xs_pitch + xo), Dx_y, p0);
                        Dx_z = Dx_z + cpml4(b, a, km, lds4(xs0 + 3 * P.xs_pitch + xo), Dx_z, p1);
                        stg4(qBo.p[2][0] + q, p0); stg4(qBo.p[1][1] + q, p1);
                    }
                }
                const float4 tHx = Dy_z - Dz_y, tHy = Dz_x - Dx_z, tHz = Dx_y - Dy_x;
                const float4 hx = pFx, hy = pFy, hz = pFz;
                float4 h2x, h2y, h2z;
                if (ADJ) {
                    // with inv_mu the H part of the cotangent volumes holds Lambda_H = im lamH (fused_backward): phase A
                    // differences it as it is, and the transpose of the E update lands in it scaled by im at my cells
                    if (has_mu) { const float4 m = ldg4(P.im + offm); h2x = fma4(m, tHx, hx); h2y = fma4(m, tHy, hy); h2z = fma4(m, tHz, hz); }
                    else { h2x = hx + tHx; h2y = hy + tHy; h2z = hz + tHz; }
                } else {
                    const float4 sim = has_mu ? S * ldg4(P.im + offm) : splat(S);
                    h2x = hx - sim * tHx; h2y = hy - sim * tHy; h2z = hz - sim * tHz;
                    if (km1 >= P.sHl && km1 < P.sHh) {
                        const int sm = src_mask(P, km1);
                        if (sm & 8) h2x = add_sources4(P, n, 3, h2x, i, j, km1);
                        if (sm & 16) h2y = add_sources4(P, n, 4, h2y, i, j, km1);
                        if (sm & 32) h2z = add_sources4(P, n, 5, h2z, i, j, km1);
                    }
                }
                float *o = dst + 3 * nc + offm;
                if (!P.peer_on) {
                    stg4(o, h2x); stg4(o + nc, h2y); stg4(o + 2 * nc, h2z);
                } else {
                    // N3 with attached neighbours: a ghost plane's H-type components are written by the neighbour's kernel
                    // (nothing of mine may land on them in the same step); my boundary planes go to the neighbour as well
                    const bool ghost = ((P.peer_on & 1) && km1 == 0) || ((P.peer_on & 2) && km1 == G.nz - 1);
                    if (!ghost) { stg4(o, h2x); stg4(o + nc, h2y); stg4(o + 2 * nc, h2z); }
                    for (int sd = 0; sd < 2; ++sd) {
                        if (!((P.peer_on >> sd) & 1) || km1 != (sd ? P.own_hi : P.own_lo)) continue;
                        float *q = P.peer[sd][par ^ 1] + own_xy;
                        stg4(q, h2x); stg4(q + P.peer_nc[sd], h2y); stg4(q + 2 * P.peer_nc[sd], h2z);
                    }
                }
                if (!ADJ && km1 >= P.dHl && km1 < P.dHh) detect4(P, n, 1, det_mask(P, km1, false), h2x, h2y, h2z, i, j, km1);
            }
            if (ADJ) { cZx = Zx; cZy = Zy; }
            pFx = fx; pFy = fy; pFz = fz;
            // nothing of plane kk is read from its stage again; with P.hold the stage of plane kk-1 goes instead
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[P.hold ? pv_i : st_i]);
            pv_i = st_i;
            st_off += P.stage;
            if (++st_i == nst) { st_i = 0; st_off = 0; st_ph ^= 1; }
            if (!DBG(4)) named_bar_sync(1, C::NCW * 32);      // ring slot (kk-1)&1 may be overwritten in the next iteration
        };

        // ---------------------------------------------------------------- prologue: plane k0-1 (F only) becomes the held stage
        {
            const int kk = Sg.k0 - 1;
            mbar_wait(&full[st_i], st_ph);
            if (ADJ) {
                const uint32_t so = stage_base + st_off + o_own;
                cgx = lds4(so); cgy = lds4(so + C::SLOT);
                if (pml) {
                    const int zs = zslab_pos(G, kk);
                    if (zs >= 0 && ing) {
                        const float b = TB1(FA, 0, ZO + zs), a = TB1(FA, 1, ZO + zs), km = TB1(FA, 2, ZO + zs);
                        const int oz = zs * pz + own_xy;
                        float4 pn;
                        cgx = cgx + cpml4(b, a, km, ldg4(qAi.p[1][0] + oz), cgx, pn);
                        cgy = cgy + cpml4(b, a, km, ldg4(qAi.p[0][1] + oz), cgy, pn);
                    }
                }
            }
            {
                const uint32_t so = stage_base + st_off + o_own;
                pFx = lds4(so); pFy = lds4(so + C::SLOT); pFz = lds4(so + 2 * C::SLOT);
                __syncwarp();
                if (lane == 0 && !P.hold) mbar_arrive(&empty[st_i]);
            }
            pv_i = st_i;
            st_off += P.stage;
            if (++st_i == nst) { st_i = 0; st_off = 0; st_ph ^= 1; }
        }
        plane_step(Sg.k0, false);
        for (int kk = Sg.k0 + 1; kk <= k1; ++kk) plane_step(kk, true);
        if (P.hold) {
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[pv_i]);      // the stage of plane k1
        }
    }
    if (P.dbg_t && threadIdx.x == 0) { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); P.dbg_t[2 * blockIdx.x + 1] = t; }
}

// ================================================================================================
// The inverse step kernel (B3 + B4): on the interior box I
//   H  = H' - srcH + S curl+(E')                 (E' at index hi comes from the record, injected before the launch)
//   q  = curl-(H)                                (H at index lo-1 is the recorded pre-step H, injected likewise)
//   g += S sum_c lamE'_c q_c   on the gradient box;      E = E' - srcE - S ie q
// Reads primal volume (n+1)&1 and cotangent volume n&1 (lamE' as the adjoint step left it), writes primal
// volume n&1.  Same tiling as k_step with the halo on the minus side: thread column 0 / row 0 recompute H on
// the cells left of / below the tile; cells outside I keep their (recorded or stale) values.
// A stage holds everything plane kk needs, in three box shapes (round 2: the stage of plane kk+1 used to be read for
// E'_x, E'_y at my cells, so two stages had to be resident and only one load was in flight; ncu showed the consumers
// waiting for data, long_scoreboard 5.5 per issue):
//   slots 0-2  E'_x,y,z(kk)          [TY+2][TX+8]   (+x / +y neighbours)
//   slots 3-5  H'_x,y,z(kk)          [TY+1][TX+4]   (my cells, halo threads included)
//   slots 6-7  E'_x, E'_y(kk+1)      [TY+1][TX+4]
//   slots 8-11 inv_eps, lamE'_x,y,z  [TY][TX]       (owned cells)
// ================================================================================================
struct InvParams {
    Dims G;
    const CUtensorMap *maps;       // [set][3] E' (shape A); [6 + set*5 + q] H'_x,y,z, E'_x, E'_y (shape B); [16] inv_eps, [17 + set*3 + c] lamE' (shape C)
    const Segment *segs;
    const int *seg_begin;          // [n_cta + 1]
    float *buf[2];                 // primal ping-pong volumes
    float *grad;                   // dL/d inv_eps, accumulated ([3][nc] with G.aniso)
    const float *im;               // inv_mu or NULL (= 1)
    const float *ie;               // inv_eps (G.aniso: [3][nc]; components y, z come by LDG at my cells)
    float *gmu;                    // N4: dL/d inv_mu, accumulated (g_mu -= S sum_c lamH'_c (curl+ E')_c), or NULL
    const float *lamH[2];          // ... the H part of the cotangent volumes: lamH' of step n is in volume (n+1)&1 (im lamH' with inv_mu)
    const int *step;
    int bias, n_steps;             // this launch inverts step n = *step + bias; nothing to do if n >= n_steps (see enqueue_bwd)
    int nst, stage;
    int n_src;
    int sEl, sEh, sHl, sHh;
    SourceDev src[MAX_SRC];
};

__device__ __forceinline__ float4 sel4(bool m0, bool m1, bool m2, bool m3, float4 a, float4 b)
{
    return make_float4(m0 ? a.x : b.x, m1 ? a.y : b.y, m2 ? a.z : b.z, m3 ? a.w : b.w);
}
__device__ __forceinline__ void st_masked(float *p, float4 v, bool all, bool m0, bool m1, bool m2, bool m3)
{
    if (all) { stg4(p, v); return; }
    if (m0) p[0] = v.x;
    if (m1) p[1] = v.y;
    if (m2) p[2] = v.z;
    if (m3) p[3] = v.w;
}

template <class C>
__global__ void __launch_bounds__(C::THREADS, 1) k_inverse(const __grid_constant__ InvParams P)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const Dims &G = P.G;
    const uint32_t stage_base = smem_u32(smem);
    const uint32_t ring_base = stage_base + (uint32_t)P.nst * P.stage;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)P.nst * P.stage + C::IRING_BYTES);
    uint64_t *empty = full + MAX_ST;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = *P.step + P.bias;
    if (n >= P.n_steps) return;
    const int rd = (n + 1) & 1, wv = n & 1;
    const int nst = P.nst;
    constexpr uint32_t OB = 3 * C::SLOT, OD = OB + 3 * C::SLOTB, OC = OB + 5 * C::SLOTB;   // slot groups inside a stage

    if (threadIdx.x == 0) {
        for (int s = 0; s < nst; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], C::NCW); }
        fence_mbar_init();
    }
    __syncthreads();
    const int seg_lo = P.seg_begin[blockIdx.x], seg_hi = P.seg_begin[blockIdx.x + 1];

    // ============================================================================== producer
    if (warp == C::NCW) {
        if (lane != 0) return;
        const CUtensorMap *MA = P.maps + rd * 3, *MB = P.maps + 6 + rd * 5, *Mie = P.maps + 16, *ML = P.maps + 17 + wv * 3;
        int s = 0, use = 0;
        for (int sg = seg_lo; sg < seg_hi; ++sg) {
            const Segment S = P.segs[sg];
            const int x = S.i0 - 4, y = S.j0 - 1;
            for (int kk = S.k0 - 1; kk < S.k1; ++kk) {
                if (use > 0) mbar_wait(&empty[s], (use - 1) & 1);
                uint64_t *fb = &full[s];
                uint8_t *st = smem + (size_t)s * P.stage;
                const bool first = kk == S.k0 - 1;       // only H of this plane is wanted: no inv_eps, no lamE'
                // lamE' only enters the gradient: planes and tiles outside the gradient box do not load it
                const bool lam = !first && kk >= G.glo[2] && kk < G.ghi[2] && S.i0 < G.ghi[0] && S.i0 + C::TX > G.glo[0] &&
                                 S.j0 < G.ghi[1] && S.j0 + C::TY > G.glo[1];
                mbar_expect_tx(fb, 3u * C::BOX_BYTES + 5u * C::BOXB_BYTES + (first ? 0u : (lam ? 4u : 1u) * C::BOXC_BYTES));
                for (int c = 0; c < 3; ++c) tma_load_3d(st + c * C::SLOT, MA + c, x, y, kk, fb);
                for (int c = 0; c < 3; ++c) tma_load_3d(st + OB + c * C::SLOTB, MB + c, x, y, kk, fb);
                for (int c = 0; c < 2; ++c) tma_load_3d(st + OD + c * C::SLOTB, MB + 3 + c, x, y, kk + 1, fb);
                if (!first) {
                    tma_load_3d(st + OC, Mie, S.i0, S.j0, kk, fb);
                    if (lam) for (int c = 0; c < 3; ++c) tma_load_3d(st + OC + (1 + c) * C::SLOTC, ML + c, S.i0, S.j0, kk, fb);
                }
                if (++s == nst) { s = 0; ++use; }
            }
        }
        return;
    }

    // ============================================================================== consumers
    const int tx0 = (warp % C::PCX) * 8 + (lane & 7), ty0 = (warp / C::PCX) * 4 + (lane >> 3);
    const bool dup = tx0 >= C::CW || ty0 >= C::RW;
    const int tx = min(tx0, C::CW - 1), ty = min(ty0, C::RW - 1);
    const bool inner = !dup && tx >= 1 && ty >= 1;                 // column 0 / row 0 are the halo threads
    const uint32_t oA = (ty * C::PW + 4 * tx) * 4;                 // my first cell inside a box of each shape
    const uint32_t oB = (ty * C::BW + 4 * tx) * 4;
    const uint32_t oC = (max(ty - 1, 0) * C::TX + 4 * max(tx - 1, 0)) * 4;
    const uint32_t r_own = (ty * C::RP + 4 * tx) * 4;
    float *dst = P.buf[wv];
    const float S = G.S;
    const long long nc = G.nc;
    const int plane = G.ny * G.nx;

    int st_i = 0;
    uint32_t st_ph = 0, st_off = 0;
    for (int sg = seg_lo; sg < seg_hi; ++sg) {
        const Segment Sg = P.segs[sg];
        const int i = Sg.i0 - 4 + 4 * tx, j = Sg.j0 - 1 + ty;
        const bool iny = j >= G.lo[1] && j < G.hi[1];
        const bool m0 = iny && i + 0 >= G.lo[0] && i + 0 < G.hi[0], m1 = iny && i + 1 >= G.lo[0] && i + 1 < G.hi[0];
        const bool m2 = iny && i + 2 >= G.lo[0] && i + 2 < G.hi[0], m3 = iny && i + 3 >= G.lo[0] && i + 3 < G.hi[0];
        const bool mall = m0 && m1 && m2 && m3, many = m0 || m1 || m2 || m3;
        const bool gy = j >= G.glo[1] && j < G.ghi[1];
        const bool g0 = gy && i + 0 >= G.glo[0] && i + 0 < G.ghi[0], g1 = gy && i + 1 >= G.glo[0] && i + 1 < G.ghi[0];
        const bool g2 = gy && i + 2 >= G.glo[0] && i + 2 < G.ghi[0], g3 = gy && i + 3 >= G.glo[0] && i + 3 < G.ghi[0];
        const bool gall = g0 && g1 && g2 && g3, gany = g0 || g1 || g2 || g3;
        const bool own_ok = inner && many;
        const int own_xy = j * G.nx + i;
        float4 cHx = splat(0.f), cHy = cHx;      // H_x, H_y of plane kk-1 at my cells

        for (int kk = Sg.k0 - 1; kk < Sg.k1; ++kk) {
            const bool prolog = kk == Sg.k0 - 1;
            const bool inz = kk >= G.lo[2] && kk < G.hi[2];
            mbar_wait(&full[st_i], st_ph);
            const uint32_t sb = stage_base + st_off;
            const uint32_t sA = sb + oA, sB = sb + OB + oB, sD = sb + OD + oB, sC = sb + OC + oC;
            // ------------------------------------------------------------ H of plane kk
            const float4 Ex = lds4(sA), Ey = lds4(sA + C::SLOT), Ez = lds4(sA + 2 * C::SLOT);
            const float4 Ex_py = lds4(sA + C::ROWB), Ez_py = lds4(sA + 2 * C::SLOT + C::ROWB);
            const float Ey_px = lds1(sA + C::SLOT + 16), Ez_px = lds1(sA + 2 * C::SLOT + 16);
            const float4 Ex_pz = lds4(sD), Ey_pz = lds4(sD + C::SLOTB);
            const float4 Hpx = lds4(sB), Hpy = lds4(sB + C::SLOTB), Hpz = lds4(sB + 2 * C::SLOTB);
            const float4 Dy_z = Ez_py - Ez, Dy_x = Ex_py - Ex;
            const float4 Dx_y = dplus_x(Ey, Ey_px), Dx_z = dplus_x(Ez, Ez_px);
            const float4 Dz_x = Ex_pz - Ex, Dz_y = Ey_pz - Ey;
            // S im at my cells (halo threads included: whatever they produce outside I is discarded below)
            const float4 sim = (P.im && many && inz) ? S * ldg4(P.im + kk * plane + own_xy) : splat(S);
            float4 Hx = fma4(sim, Dy_z - Dz_y, Hpx), Hy = fma4(sim, Dz_x - Dx_z, Hpy), Hz = fma4(sim, Dx_y - Dy_x, Hpz);
            if (kk >= P.sHl && kk < P.sHh) {
                const int sm = src_mask(P, kk);
                if (sm & 8) Hx = Hx - add_sources4(P, n, 3, splat(0.f), i, j, kk);
                if (sm & 16) Hy = Hy - add_sources4(P, n, 4, splat(0.f), i, j, kk);
                if (sm & 32) Hz = Hz - add_sources4(P, n, 5, splat(0.f), i, j, kk);
            }
            if (P.gmu && !prolog && own_ok && inz) {          // N4, dL/d inv_mu at my cells of I (sequential sweep only: see fused_backward)
                const int off = kk * plane + own_xy;
                const float *lh = P.lamH[(n + 1) & 1] + off;
                float4 a = ldg4(lh) * (Dy_z - Dz_y);
                a = fma4(ldg4(lh + nc), Dz_x - Dx_z, a);
                a = fma4(ldg4(lh + 2 * nc), Dx_y - Dy_x, a);
                if (P.im) a = a * (S * rcp4(sim));                // the volume holds im lamH': a / im = a S / (S im)
                a = S * a;
                float *gp = P.gmu + off;
                if (mall) stg4(gp, ld4(gp) - a);
                else {
                    if (m0) gp[0] -= a.x;
                    if (m1) gp[1] -= a.y;
                    if (m2) gp[2] -= a.z;
                    if (m3) gp[3] -= a.w;
                }
            }
            // outside I the volume's own value stands (the recorded pre-step H at index lo-1)
            Hx = sel4(m0 && inz, m1 && inz, m2 && inz, m3 && inz, Hx, Hpx);
            Hy = sel4(m0 && inz, m1 && inz, m2 && inz, m3 && inz, Hy, Hpy);
            Hz = sel4(m0 && inz, m1 && inz, m2 && inz, m3 && inz, Hz, Hpz);
            if (!prolog) {
                const uint32_t rg = ring_base + (uint32_t)(kk & 1) * (3 * C::RING_ARR * 4) + r_own;
                sts4(rg, Hx); sts4(rg + C::RING_ARR * 4, Hy); sts4(rg + 2 * C::RING_ARR * 4, Hz);
                const int off = kk * plane + own_xy;
                float4 gv = splat(0.f);
                const bool gz = kk >= G.glo[2] && kk < G.ghi[2];
                if (own_ok && gz && gall && !G.aniso) gv = ld4(P.grad + off);
                named_bar_sync(1, C::NCW * 32);
                // ------------------------------------------------------------ q, gradient, E of plane kk
                if (own_ok) {
                    const float4 Hx_my = lds4(rg - C::RP * 4), Hz_my = lds4(rg + 2 * C::RING_ARR * 4 - C::RP * 4);
                    const float Hy_mx = lds1(rg + C::RING_ARR * 4 - 4), Hz_mx = lds1(rg + 2 * C::RING_ARR * 4 - 4);
                    const float4 By_z = Hz - Hz_my, By_x = Hx - Hx_my;
                    const float4 Bx_y = dminus_x(Hy, Hy_mx), Bx_z = dminus_x(Hz, Hz_mx);
                    const float4 Bz_x = Hx - cHx, Bz_y = Hy - cHy;
                    const float4 qx = By_z - Bz_y, qy = Bz_x - Bx_z, qz = Bx_y - By_x;
                    const float4 sie = S * lds4(sC);
                    const float4 lx = lds4(sC + C::SLOTC), ly = lds4(sC + 2 * C::SLOTC), lz = lds4(sC + 3 * C::SLOTC);
                    float4 siy = sie, siz = sie;
                    if (G.aniso) { siy = S * ldg4(P.ie + nc + off); siz = S * ldg4(P.ie + 2 * nc + off); }
                    float4 E2x = Ex - sie * qx, E2y = Ey - siy * qy, E2z = Ez - siz * qz;
                    if (kk >= P.sEl && kk < P.sEh) {
                        const int sm = src_mask(P, kk);
                        if (sm & 1) E2x = E2x - add_sources4(P, n, 0, splat(0.f), i, j, kk);
                        if (sm & 2) E2y = E2y - add_sources4(P, n, 1, splat(0.f), i, j, kk);
                        if (sm & 4) E2z = E2z - add_sources4(P, n, 2, splat(0.f), i, j, kk);
                    }
                    float *o = dst + off;
                    st_masked(o, E2x, mall, m0, m1, m2, m3);
                    st_masked(o + nc, E2y, mall, m0, m1, m2, m3);
                    st_masked(o + 2 * nc, E2z, mall, m0, m1, m2, m3);
                    st_masked(o + 3 * nc, Hx, mall, m0, m1, m2, m3);
                    st_masked(o + 4 * nc, Hy, mall, m0, m1, m2, m3);
                    st_masked(o + 5 * nc, Hz, mall, m0, m1, m2, m3);
                    if (gz && gany && G.aniso) {               // reading R30: one gradient volume per component
                        const float4 gc[3] = { S * (lx * qx), S * (ly * qy), S * (lz * qz) };
                        for (int c = 0; c < 3; ++c) {
                            float *gp = P.grad + c * nc + off;
                            if (gall) stg4(gp, ld4(gp) + gc[c]);
                            else {
                                if (g0) gp[0] += gc[c].x;
                                if (g1) gp[1] += gc[c].y;
                                if (g2) gp[2] += gc[c].z;
                                if (g3) gp[3] += gc[c].w;
                            }
                        }
                    } else if (gz && gany) {
                        const float4 ga = S * fma4(lx, qx, fma4(ly, qy, lz * qz));
                        if (gall) stg4(P.grad + off, gv + ga);
                        else {
                            float *gp = P.grad + off;
                            if (g0) gp[0] += ga.x;
                            if (g1) gp[1] += ga.y;
                            if (g2) gp[2] += ga.z;
                            if (g3) gp[3] += ga.w;
                        }
                    }
                }
            }
            cHx = Hx; cHy = Hy;
            // nothing of this plane is read from its stage again
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st_i]);
            st_off += P.stage;
            if (++st_i == nst) { st_i = 0; st_off = 0; st_ph ^= 1; }
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

// ---- the compiled tile shapes ----------------------------------------------------------------------
struct TileImpl {
    int TX, TY, threads, ncw, stage, ring_bytes, istage, iring_bytes;
    void (*launch_fwd)(const StepParams &, int n_cta, size_t smem, cudaStream_t);
    void (*launch_adj)(const StepParams &, int n_cta, size_t smem, cudaStream_t);
    cudaError_t (*set_smem)(size_t);
    void (*launch_inv)(const InvParams &, int n_cta, size_t smem, cudaStream_t);
    cudaError_t (*set_smem_inv)(size_t);
};
template <class C> void launch_inv_impl(const InvParams &P, int n_cta, size_t smem, cudaStream_t st)
{
    k_inverse<C><<<n_cta, C::THREADS, smem, st>>>(P);
}
template <class C> cudaError_t set_smem_inv_impl(size_t smem)
{
    cudaError_t e = cudaFuncSetAttribute(k_inverse<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_inverse<C>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    return e;
}
// step kernels are launched with programmatic stream serialisation (see the top of k_step)
template <class C, bool ADJ> void launch_step_impl(const StepParams &P, int n_cta, size_t smem, cudaStream_t st)
{
    static const bool pdl = !getenv("FDTD_NO_PDL");
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(n_cta); cfg.blockDim = dim3(C::THREADS); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    if (P.G.aniso || P.sigma || P.im) cudaLaunchKernelEx(&cfg, k_step<C, ADJ, true>, P);
    else cudaLaunchKernelEx(&cfg, k_step<C, ADJ, false>, P);
}
template <class C> void launch_fwd_impl(const StepParams &P, int n_cta, size_t smem, cudaStream_t st) { launch_step_impl<C, false>(P, n_cta, smem, st); }
template <class C> void launch_adj_impl(const StepParams &P, int n_cta, size_t smem, cudaStream_t st) { launch_step_impl<C, true>(P, n_cta, smem, st); }
template <class K> cudaError_t set_smem_kernel(K kernel, size_t smem)
{
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    // the same shared-memory carve-out for every kernel of the time loop: no L1 / shared reconfiguration between launches
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    return e;
}
template <class C> cudaError_t set_smem_impl(size_t smem)
{
    cudaError_t e = set_smem_kernel(k_step<C, false, false>, smem);
    if (e == cudaSuccess) e = set_smem_kernel(k_step<C, true, false>, smem);
    if (e == cudaSuccess) e = set_smem_kernel(k_step<C, false, true>, smem);
    if (e == cudaSuccess) e = set_smem_kernel(k_step<C, true, true>, smem);
    return e;
}
#define TILE(TX4, TY) { 4 * TX4, TY, Cfg<TX4, TY>::THREADS, Cfg<TX4, TY>::NCW, Cfg<TX4, TY>::STAGE, Cfg<TX4, TY>::RING_BYTES, \
                        Cfg<TX4, TY>::ISTAGE, Cfg<TX4, TY>::IRING_BYTES, \
                        launch_fwd_impl<Cfg<TX4, TY>>, launch_adj_impl<Cfg<TX4, TY>>, set_smem_impl<Cfg<TX4, TY>>, \
                        launch_inv_impl<Cfg<TX4, TY>>, set_smem_inv_impl<Cfg<TX4, TY>> }
// shapes compiled for the inverse step only (widths that cover common interiors without a ragged second tile column)
#define ITILE(TX4, TY) { 4 * TX4, TY, Cfg<TX4, TY>::THREADS, Cfg<TX4, TY>::NCW, Cfg<TX4, TY>::STAGE, Cfg<TX4, TY>::RING_BYTES, \
                         Cfg<TX4, TY>::ISTAGE, Cfg<TX4, TY>::IRING_BYTES, nullptr, nullptr, nullptr, \
                         launch_inv_impl<Cfg<TX4, TY>>, set_smem_inv_impl<Cfg<TX4, TY>> }
const TileImpl kTiles[] = {
    TILE(2, 3), TILE(4, 3), TILE(8, 7), TILE(16, 7), TILE(16, 15), TILE(25, 7), TILE(25, 11),
    TILE(32, 7), TILE(32, 11), TILE(50, 7), TILE(50, 11), TILE(62, 7),
    ITILE(36, 7), ITILE(40, 7), ITILE(44, 7), ITILE(48, 7), ITILE(56, 7),
};
constexpr int kNumTiles = sizeof(kTiles) / sizeof(kTiles[0]);

}  // namespace

struct FusedState {
    const TileImpl *tile = nullptr;
    int TX = 0, TY = 0, nst = 0, n_cta = 0, n_rot = 1;
    // pipelined reverse sweep (enqueue_bwd): the adjoint step (n_adj CTAs) is launched together with the inverse step
    // of the step before it (n_inv_p CTAs); n_inv_p = 0: one kernel after the other (see fused_setup)
    int n_adj = 0, n_inv_p = 0;
    Segment *d_isegs_p = nullptr;
    int *d_iseg_begin_p = nullptr;
    size_t smem = 0;
    StepParams sp{};
    // inverse step kernel: its own tile shape and segment table (interior box only)
    const TileImpl *itile = nullptr;
    int inst = 0, in_cta = 0;
    size_t ismem = 0;
    InvParams ip{};
    Segment *d_isegs = nullptr;
    int *d_iseg_begin = nullptr;
    float *bufB = nullptr;                 // second primal field buffer
    float *lamB = nullptr;                 // second cotangent buffer
    // tensor-map tables: [0] primal (fields / bufB), [1] cotangents (lam / lamB); entry set*6 + c, [12] = inv_eps
    // [2]: the inverse kernel's table (its own box shape): [set][6] primal, [12] inv_eps, [13 + set*3 + c] lamE'
    CUtensorMap *d_maps[3] = { nullptr, nullptr, nullptr };
    CUtensorMap *h_maps[3] = { nullptr, nullptr, nullptr };   // pinned staging
    cudaEvent_t maps_done = nullptr;
    Segment *d_segs[2] = { nullptr, nullptr };      // work tables of the forward / adjoint step kernel
    int *d_seg_begin[2] = { nullptr, nullptr };
    size_t seg_cap = 0;
    unsigned long long *d_cta_t = nullptr;          // per-CTA start / end timestamps (calibration)
    double calibrated_us[2] = { 0.0, 0.0 };
    const float *maps_key[3][2] = { { nullptr, nullptr }, { nullptr, nullptr }, { nullptr, nullptr } };   // volume A / inv_eps the maps were built for
};

namespace {

// Work sequence: position q = column * nz + plane, column = tile (y fastest).  It is split into n_cta runs of equal
// estimated cost.  The cost model (a plane of a tile costs 1, plus wy if the tile has rows in a y slab, plus wz if
// the plane is in a z slab: their CPML states are read by every thread of the tile) is only the starting point:
// calibrate() measures the CTAs and moves the cuts.
std::vector<double> model_cost(const Dims &G, int TX, int TY, double wy, double wz)
{
    const int ntx = (G.nx + TX - 1) / TX, nty = (G.ny + TY - 1) / TY;
    const long long n_tiles = (long long)ntx * nty;
    std::vector<double> w((size_t)n_tiles * G.nz);
    for (long long t = 0; t < n_tiles; ++t) {
        const int j0 = (int)(t % nty) * TY;
        const bool ys = G.d > 0 && (j0 <= G.d || j0 + TY >= G.ny - G.d);
        for (int k = 0; k < G.nz; ++k) {
            const bool zs = G.d > 0 && (k <= G.d || k >= G.nz - G.d - 1);
            w[t * G.nz + k] = 1.0 + (ys ? wy : 0.0) + (zs ? wz : 0.0);
        }
    }
    return w;
}

// Columns that do the same work per plane (same CPML slabs, same number of valid rows and float4 columns) form a
// class; the cost profiles of a class are kept identical so that its columns get identical cuts.
std::vector<int> column_classes(const Dims &G, int TX, int TY)
{
    const int ntx = (G.nx + TX - 1) / TX, nty = (G.ny + TY - 1) / TY;
    std::vector<int> cls((size_t)ntx * nty);
    std::vector<int> keys;
    for (int t = 0; t < ntx * nty; ++t) {
        const int i0 = (t / nty) * TX, j0 = (t % nty) * TY;
        int key = 0;
        if (G.d > 0) {
            key |= (j0 <= G.d) | (j0 + TY >= G.ny - G.d) << 1;
            key |= (i0 <= G.d) << 2 | (i0 + TX >= G.nx - G.d) << 3;
        }
        key |= (j0 + TY > G.ny) << 4 | (i0 + TX > G.nx) << 5;
        size_t c = std::find(keys.begin(), keys.end(), key) - keys.begin();
        if (c == keys.size()) keys.push_back(key);
        cls[t] = (int)c;
    }
    return cls;
}

void average_classes(std::vector<double> &w, const std::vector<int> &cls, int nz)
{
    const int n_cls = cls.empty() ? 0 : *std::max_element(cls.begin(), cls.end()) + 1;
    std::vector<double> mean((size_t)n_cls * nz, 0.0);
    std::vector<int> cnt(n_cls, 0);
    for (size_t t = 0; t < cls.size(); ++t) {
        ++cnt[cls[t]];
        for (int k = 0; k < nz; ++k) mean[(size_t)cls[t] * nz + k] += w[t * nz + k];
    }
    for (size_t t = 0; t < cls.size(); ++t)
        for (int k = 0; k < nz; ++k) w[t * nz + k] = mean[(size_t)cls[t] * nz + k] / cnt[cls[t]];
}

// n_cta + 1 cut positions that split the sequence into runs of equal summed cost (every run non-empty)
std::vector<long long> equal_cost_cuts(const std::vector<double> &w, int n_cta)
{
    const long long total = (long long)w.size();
    std::vector<double> pre(total + 1, 0.0);
    for (long long q = 0; q < total; ++q) pre[q + 1] = pre[q] + w[q];
    std::vector<long long> cut(n_cta + 1, 0);
    for (int c = 1; c < n_cta; ++c) {
        const double target = pre[total] * c / n_cta;
        long long q = std::lower_bound(pre.begin(), pre.end(), target) - pre.begin();
        q = std::max(q, cut[c - 1] + 1);
        cut[c] = std::min(q, total - (n_cta - c));
    }
    cut[n_cta] = total;
    return cut;
}

// One run per CTA: ranges [a, b) of sequence positions, marched in order.
typedef std::vector<std::vector<std::pair<long long, long long>>> Runs;

// The plain split: the whole sequence cut into n_cta contiguous runs.  Neighbouring columns are then marched
// with arbitrary plane offsets, so the halo rows a tile shares with its y neighbours miss L2 (measured on C3:
// +76 MB of DRAM reads per launch, +27 % over the lock-step split below).
thread_local int t_partition_kind = FDTD_PARTITION_NONE;    // what the last make_runs() on this thread produced

Runs contiguous_runs(const std::vector<double> &w, int nz, int n_cta)
{
    t_partition_kind = FDTD_PARTITION_CONTIGUOUS;
    const std::vector<long long> cut = equal_cost_cuts(w, n_cta);
    Runs runs(n_cta);
    for (int c = 0; c < n_cta; ++c)
        for (long long a = cut[c]; a < cut[c + 1];) {
            const long long b = std::min(cut[c + 1], (a / nz + 1) * nz);
            runs[c].push_back({ a, b });
            a = b;
        }
    return runs;
}

// The lock-step split.  With L = total cost / n_cta, a column of cost Z gets floor(Z / L) full runs cut at the
// cost positions 0, L, 2L, ...; columns of one class have the same profile, hence the same cuts, and because
// every CTA starts at time 0 and costs are times, y-adjacent tiles walk through the same planes at the same
// time: a halo row is fetched from DRAM once and found in L2 by the neighbour.  What is left at the top of the
// columns (less than L each) is chained, column after column, into the remaining CTAs; they also cost L each.
Runs lockstep_runs(const std::vector<double> &w, int nz, int n_cta)
{
    const long long n_col = (long long)w.size() / nz;
    double total = 0.0;
    for (double x : w) total += x;
    const double L = total / n_cta, eps = 1e-7 * L;
    Runs runs;
    std::vector<double> left_w;
    std::vector<long long> left_q;
    std::vector<double> pre(nz + 1);
    for (long long t = 0; t < n_col; ++t) {
        pre[0] = 0.0;
        for (int k = 0; k < nz; ++k) pre[k + 1] = pre[k] + w[t * nz + k];
        const int R = (int)std::floor(pre[nz] / L + 1e-7);
        int k_prev = 0;
        for (int j = 1; j <= R; ++j) {
            const int k = (int)(std::lower_bound(pre.begin(), pre.end(), j * L - eps) - pre.begin());
            if (k <= k_prev) return contiguous_runs(w, nz, n_cta);          // L is below one plane: nothing to align
            runs.push_back({ { t * nz + k_prev, t * nz + k } });
            k_prev = k;
        }
        for (int k = k_prev; k < nz; ++k) { left_w.push_back(w[t * nz + k]); left_q.push_back(t * nz + k); }
    }
    const int n_left = n_cta - (int)runs.size();
    if (n_left < 0 || (n_left == 0 && !left_q.empty()) || (long long)left_q.size() < n_left)
        return contiguous_runs(w, nz, n_cta);
    if (n_left > 0) {
        const std::vector<long long> cut = equal_cost_cuts(left_w, n_left);
        for (int c = 0; c < n_left; ++c) {
            std::vector<std::pair<long long, long long>> run;
            for (long long p = cut[c]; p < cut[c + 1]; ++p) {
                const long long q = left_q[p];
                if (!run.empty() && run.back().second == q && q % nz != 0) ++run.back().second;
                else run.push_back({ q, q + 1 });
            }
            runs.push_back(run);
        }
    }
    t_partition_kind = FDTD_PARTITION_LOCKSTEP;
    return runs;
}

// Large grids: more columns than CTAs.  Whole columns are dealt out in waves (CTA c takes the c-th, (c + n_cta)-th,
// ... of them): every CTA starts a column at plane 0 at time 0, so the n_cta y-consecutive columns of a wave are
// marched in lock step.  Only the cheap columns (no y slab: they all cost the same, so the CTAs stay together) are
// dealt, for as long as a CTA's total stays below the mean; the last wave may be partial.  The other columns form
// a pool that is cut, in sequence order, into one chunk per CTA sized so that every CTA ends up with the same
// total cost (a CTA whose whole columns already cost the mean gets nothing from the pool).
Runs wave_runs(const std::vector<double> &w, int nz, int n_cta)
{
    const long long n_col = (long long)w.size() / nz;
    std::vector<double> colw(n_col, 0.0);
    double total = 0.0, cheapest = 1e300;
    for (long long t = 0; t < n_col; ++t) {
        for (int k = 0; k < nz; ++k) colw[t] += w[t * nz + k];
        total += colw[t];
        cheapest = std::min(cheapest, colw[t]);
    }
    std::vector<long long> order;                       // cheap columns first, each group in sequence order
    for (long long t = 0; t < n_col; ++t) if (colw[t] <= 1.2 * cheapest) order.push_back(t);
    const size_t n_cheap = order.size();
    for (long long t = 0; t < n_col; ++t) if (colw[t] > 1.2 * cheapest) order.push_back(t);
    const double mean = total / n_cta;
    Runs runs(n_cta);
    std::vector<double> used(n_cta, 0.0);
    size_t dealt = 0;
    for (; dealt < n_cheap; ++dealt) {
        const int c = (int)(dealt % n_cta);
        const long long t = order[dealt];
        if (used[c] + colw[t] > mean * (1.0 + 1e-9)) break;
        runs[c].push_back({ t * nz, (t + 1) * nz });
        used[c] += colw[t];
    }
    if (dealt < (size_t)n_cta) return lockstep_runs(w, nz, n_cta);      // not even one full wave
    t_partition_kind = FDTD_PARTITION_WAVES;
    if (dealt == order.size()) return runs;
    // the pool: positions of the columns order[dealt..], column after column
    double pool = 0.0;
    for (size_t p = dealt; p < order.size(); ++p) pool += colw[order[p]];
    // level: sum_c max(0, level - used[c]) = pool
    std::vector<double> u(used);
    std::sort(u.begin(), u.end());
    double level = u[0] + pool, below = 0.0;
    for (int m = 1; m <= n_cta; ++m) {           // the m cheapest CTAs share the pool
        below += u[m - 1];
        level = (pool + below) / m;
        if (m == n_cta || level <= u[m]) break;
    }
    int last_c = -1;
    for (int c = 0; c < n_cta; ++c) if (level - used[c] > 0.0) last_c = c;
    size_t p = dealt;
    int k = 0;                                   // next position: plane k of column order[p]
    double acc = 0.0, target = 0.0;
    for (int c = 0; c < n_cta && p < order.size(); ++c) {
        const double budget = level - used[c];
        if (budget <= 0.0) continue;
        target += budget;
        bool first = true;
        while (p < order.size()) {
            const long long t = order[p];
            const double x = w[t * nz + k];
            if (c != last_c && !first && acc + x > target * (1.0 + 1e-9)) break;
            const long long q = t * nz + k;
            if (!runs[c].empty() && runs[c].back().second == q && k != 0) ++runs[c].back().second;
            else runs[c].push_back({ q, q + 1 });
            acc += x;
            first = false;
            if (++k == nz) { k = 0; ++p; }
        }
    }
    return runs;
}

Runs make_runs(const std::vector<double> &w, int nz, int n_cta)
{
    static const bool contiguous = getenv("FDTD_PARTITION") && !strcmp(getenv("FDTD_PARTITION"), "contiguous");
    if (contiguous) return contiguous_runs(w, nz, n_cta);
    return (long long)w.size() / nz >= n_cta ? wave_runs(w, nz, n_cta) : lockstep_runs(w, nz, n_cta);
}

// origin (i_org, j_org, k_org) of the tiled box; nz planes per column
void segments_from_runs(int nty, int nz, int TX, int TY, int i_org, int j_org, int k_org, const Runs &runs,
                        std::vector<Segment> &segs, std::vector<int> &seg_begin)
{
    segs.clear();
    seg_begin.assign(runs.size() + 1, 0);
    for (size_t cta = 0; cta < runs.size(); ++cta) {
        seg_begin[cta] = (int)segs.size();
        for (const std::pair<long long, long long> &r : runs[cta]) {
            const long long tile = r.first / nz;
            Segment s{};
            s.i0 = i_org + (int)(tile / nty) * TX; s.j0 = j_org + (int)(tile % nty) * TY;
            s.k0 = k_org + (int)(r.first % nz); s.k1 = s.k0 + (int)(r.second - r.first);
            segs.push_back(s);
        }
    }
    seg_begin[runs.size()] = (int)segs.size();
}

}  // namespace

extern "C" int fdtd_debug_partition(int32_t nx, int32_t ny, int32_t nz, int32_t d, int32_t tile_x, int32_t tile_y,
                                    int32_t n_cta, double wy, double wz, int32_t lockstep, int32_t *segments, int32_t cap)
{
    if (nx < 1 || ny < 1 || nz < 1 || d < 0 || tile_x < 1 || tile_y < 1 || n_cta < 1 || cap < 0 || (cap > 0 && !segments))
        return fdtd_fail(FDTD_EINVAL, "fdtd_debug_partition: bad argument");
    Dims G{};
    G.nx = nx; G.ny = ny; G.nz = nz; G.d = d;
    const int nty = (ny + tile_y - 1) / tile_y, ntx = (nx + tile_x - 1) / tile_x;
    if ((long long)ntx * nty * nz < n_cta) return fdtd_fail(FDTD_EINVAL, "fdtd_debug_partition: more CTAs than (tile, plane) positions");
    const std::vector<double> w = model_cost(G, tile_x, tile_y, wy, wz);
    const Runs runs = !lockstep ? contiguous_runs(w, nz, n_cta)
                      : ((long long)ntx * nty >= n_cta ? wave_runs(w, nz, n_cta) : lockstep_runs(w, nz, n_cta));
    std::vector<Segment> segs;
    std::vector<int> begins;
    segments_from_runs(nty, nz, tile_x, tile_y, 0, 0, 0, runs, segs, begins);
    for (size_t c = 0; c + 1 < begins.size(); ++c)
        for (int q = begins[c]; q < begins[c + 1] && q < cap; ++q) {
            int32_t *o = segments + 5 * (size_t)q;
            o[0] = (int32_t)c; o[1] = segs[q].i0; o[2] = segs[q].j0; o[3] = segs[q].k0; o[4] = segs[q].k1;
        }
    return (int)segs.size();
}

static int calibrate(fdtd_grid *g);

int fused_setup(fdtd_grid *g)
{
    const Dims &G = g->G;
    if (g->desc.path == FDTD_PATH_GENERIC) { g->fused_why_not = "generic path requested"; return FDTD_OK; }
    if (G.periodic) { g->fused_why_not = "periodic grids use the generic kernels"; return FDTD_OK; }
    if (G.nx % 4) { g->fused_why_not = "nx is not a multiple of 4"; return FDTD_OK; }
    if (G.d > 0 && (G.dpx % 4)) { g->fused_why_not = "x-slab psi storage is not float4 aligned (nx < 2*roundup4(d))"; return FDTD_OK; }
    if (G.nc >= (1LL << 31) - 4LL * G.nx * G.ny) { g->fused_why_not = "more than 2^31 cells (32-bit plane offsets)"; return FDTD_OK; }
    if (!get_encode()) { g->fused_why_not = "cuTensorMapEncodeTiled is not available"; return FDTD_OK; }
    int dev = 0, smem_cap = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&smem_cap, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        g->fused_why_not = "cannot query the device";
        return FDTD_OK;
    }

    // ---- tile choice among the compiled shapes: fewest consumer warp-planes per grid plane -------------------------
    int fTX = 0, fTY = 0;
    if (const char *e = getenv("FDTD_TILE")) sscanf(e, "%d,%d", &fTX, &fTY);
    const int tail_bytes = 2 * MAX_ST * 8 + 6 * (2 * G.dpx + 4 * G.d) * 4;     // mbarriers + CPML tables
    const TileImpl *best = nullptr;
    double best_score = -1;
    int best_nst = 0;
    for (int q = 0; q < kNumTiles; ++q) {
        const TileImpl &t = kTiles[q];
        if (!t.launch_fwd) continue;                                 // inverse-only shape
        if (fTX && (t.TX != fTX || t.TY != fTY)) continue;
        const int xs_pitch = G.d > 0 ? (2 * G.dpx * (t.TY + 2) * 4 + 127) / 128 * 128 : 0;
        const int stage = t.stage + 4 * xs_pitch;
        const int nst = std::min(MAX_ST, (smem_cap - t.ring_bytes - tail_bytes - 1024) / stage);
        if (nst < 3) continue;                                   // previous plane held + current + one in flight
        const long long ntx = (G.nx + t.TX - 1) / t.TX, nty = (G.ny + t.TY - 1) / t.TY;
        const double eff = ((double)G.nx / 4 * G.ny) / ((double)ntx * nty * t.ncw * 32);
        const double fill = std::min(1.0, (double)ntx * nty * G.nz / (8.0 * n_sm));   // enough planes per CTA to amortise prologues
        const double warps = std::min(1.0, t.ncw / 10.0);                             // enough warps to hide latency
        const double score = eff * fill * warps;
        if (score > best_score) { best_score = score; best = &t; best_nst = nst; }
    }
    if (!best) { g->fused_why_not = "no compiled tile shape fits"; return FDTD_OK; }

    FusedState *F = new FusedState();
    g->fused = F;
    F->tile = best; F->TX = best->TX; F->TY = best->TY; F->nst = best_nst;
    if (const char *e = getenv("FDTD_NST")) F->nst = std::max(3, std::min(best_nst, atoi(e)));
    const int xs_bytes = G.d > 0 ? 2 * G.dpx * (best->TY + 2) * 4 : 0, xs_pitch = (xs_bytes + 127) / 128 * 128;
    const int stage_bytes = best->stage + 4 * xs_pitch;
    F->smem = (size_t)F->nst * stage_bytes + best->ring_bytes + tail_bytes;
    int rc;
    if ((rc = g->alloc((void **)&F->bufB, (size_t)G.nc * 6 * sizeof(float)))) return rc;
    if ((rc = g->alloc_psi(g->psiE[1])) || (rc = g->alloc_psi(g->psiH[1]))) return rc;
    for (int q = 0; q < 3; ++q) {
        if ((rc = g->alloc((void **)&F->d_maps[q], sizeof(CUtensorMap) * 24))) return rc;
        if (cudaMallocHost((void **)&F->h_maps[q], sizeof(CUtensorMap) * 24) != cudaSuccess) {
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
    // one CTA per SM as soon as each gets two planes: a small grid is bound by the planes a CTA marches one after the other
    // (~2 us each, latency), not by the prologue plane a shorter run adds (64^3, C2 / C5: 6 planes per run 17.5 / 19.1 us per
    // forward / adjoint step, 4.3 planes per run on all 148 SMs 14.3 / 15.6 us; a second wave of CTAs: 18 / 22 us)
    int n_cta = (int)std::min<long long>(n_sm, std::max<long long>(1, total / 2));
    if (const char *e = getenv("FDTD_NCTA")) n_cta = std::max(1, atoi(e));
    double wy = 1.0, wz = 0.8;                   // starting point of the cost model (measured on C3); see calibrate()
    if (const char *e = getenv("FDTD_WY")) wy = atof(e);
    if (const char *e = getenv("FDTD_WZ")) wz = atof(e);
    const int n_rot = 1;
    F->n_cta = n_cta; F->n_rot = n_rot;
    std::vector<Segment> all;
    std::vector<int> begins;
    segments_from_runs(nty, G.nz, F->TX, F->TY, 0, 0, 0, make_runs(model_cost(G, F->TX, F->TY, wy, wz), G.nz, n_cta), all, begins);
    g->partition = t_partition_kind;
    F->seg_cap = (size_t)n_cta + (size_t)ntx * nty + 8;        // a run adds at most one segment per column boundary
    const size_t stride = F->seg_cap;
    for (int q = 0; q < 2; ++q) {
        if ((rc = g->alloc((void **)&F->d_segs[q], F->seg_cap * sizeof(Segment)))) return rc;
        if ((rc = g->alloc((void **)&F->d_seg_begin[q], begins.size() * sizeof(int)))) return rc;
        if (cudaMemcpy(F->d_segs[q], all.data(), all.size() * sizeof(Segment), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(F->d_seg_begin[q], begins.data(), begins.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
            (void)cudaGetLastError();
            return fdtd_fail(FDTD_ECUDA, "upload of the segment table failed");
        }
    }
    if ((rc = g->alloc((void **)&F->d_cta_t, 2 * (size_t)n_cta * sizeof(unsigned long long)))) return rc;

    // ---- inverse step kernel: tile shape (10 boxes per stage), segments over the interior box ----------------------
    {
        const TileImpl *ib = nullptr;
        double ib_score = -1;
        int ib_nst = 0;
        int iTX = 0, iTY = 0;
        if (const char *e = getenv("FDTD_ITILE")) sscanf(e, "%d,%d", &iTX, &iTY);
        const int x0 = G.lo[0] / 4 * 4;                       // first tile column (float4 aligned)
        const int nx_i = G.hi[0] - x0, ny_i = G.hi[1] - G.lo[1], nz_i = G.hi[2] - G.lo[2];
        for (int q = 0; q < kNumTiles; ++q) {
            const TileImpl &t = kTiles[q];
            if (iTX && (t.TX != iTX || t.TY != iTY)) continue;
            int nst = std::min(MAX_ST, (smem_cap - t.iring_bytes - tail_bytes - 1024) / t.istage);
            if (const char *e = getenv("FDTD_INST")) nst = std::min(nst, atoi(e));
            // every stage is self-contained: one in use, the others in flight; two are enough (measured on C3: 100 x 11
            // with 2 or 3 stages 92 us; 176 x 7, 192 x 7, 200 x 7 with 2 stages 84-86 us: one tile column over the box wins)
            if (nst < 2) continue;
            const long long ntx = (nx_i + t.TX - 1) / t.TX, nty = (ny_i + t.TY - 1) / t.TY;
            const double eff = ((double)(G.hi[0] - G.lo[0]) / 4 * ny_i) / ((double)ntx * nty * t.ncw * 32);
            const double fill = std::min(1.0, (double)ntx * nty * nz_i / (8.0 * n_sm));
            const double warps = std::min(1.0, t.ncw / 10.0);
            const double score = eff * fill * warps;
            if (score > ib_score) { ib_score = score; ib = &t; ib_nst = nst; }
        }
        if (ib && nx_i > 0 && ny_i > 0 && nz_i > 0) {
            // tiles start at row lo_y (their first halo row is lo_y - 1) and at column x0
            const int ntx = (nx_i + ib->TX - 1) / ib->TX, nty = (ny_i + ib->TY - 1) / ib->TY;
            const long long itotal = (long long)ntx * nty * nz_i;
            int in_cta = (int)std::min<long long>(n_sm, std::max<long long>(1, itotal / 2));      // (64^3: 19.6 -> 14.8 us)
            if (const char *e = getenv("FDTD_INV_NCTA")) in_cta = std::max(1, atoi(e));
            std::vector<Segment> isegs;
            std::vector<int> ibeg;
            segments_from_runs(nty, nz_i, ib->TX, ib->TY, x0, G.lo[1], G.lo[2],
                               make_runs(std::vector<double>((size_t)itotal, 1.0), nz_i, in_cta), isegs, ibeg);
            if ((rc = g->alloc((void **)&F->d_isegs, isegs.size() * sizeof(Segment)))) return rc;
            if ((rc = g->alloc((void **)&F->d_iseg_begin, ibeg.size() * sizeof(int)))) return rc;
            if (cudaMemcpy(F->d_isegs, isegs.data(), isegs.size() * sizeof(Segment), cudaMemcpyHostToDevice) != cudaSuccess ||
                cudaMemcpy(F->d_iseg_begin, ibeg.data(), ibeg.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
                (void)cudaGetLastError();
                return fdtd_fail(FDTD_ECUDA, "upload of the inverse segment table failed");
            }
            F->itile = ib; F->inst = ib_nst; F->in_cta = in_cta;
            const int istage = ib->istage;
            F->ismem = (size_t)ib_nst * istage + ib->iring_bytes + tail_bytes;
            InvParams &I = F->ip;
            I.G = G; I.segs = F->d_isegs; I.seg_begin = F->d_iseg_begin; I.step = g->d_step;
            I.nst = ib_nst; I.stage = istage;
            I.bias = 0; I.n_steps = 1 << 30;
            if (ib->set_smem_inv(F->ismem) != cudaSuccess) { (void)cudaGetLastError(); F->itile = nullptr; }

            // ---- pipelined reverse sweep (enqueue_bwd): launch n = {adjoint step n, inverse step n+1, injection n} ------
            // FDTD_REVERSE_SWEEP = grouped (default): both kernels keep their full grids; they cannot share an SM (shared
            //   memory), so the CTAs of one follow the CTAs of the other SM by SM without a kernel boundary in between
            //   (C3: 125.1 vs 134.1 us per reverse step);
            // = split: disjoint SMs, divided by the kernels' bytes (the inverse step's weighted 1.3; C3: 129.1 us: each
            //   CTA keeps one ~50 KB stage in flight per plane, so neither kernel gets faster per SM when it owns fewer);
            // = sequential: one kernel after the other (round-1 checkpoints A-D).
            F->n_adj = n_cta;
            const char *sweep = getenv("FDTD_REVERSE_SWEEP");
            const bool full = !sweep || !strcmp(sweep, "grouped");
            if (F->itile && full) {
                F->n_inv_p = in_cta; F->d_isegs_p = F->d_isegs; F->d_iseg_begin_p = F->d_iseg_begin;
                g->pipelined_inverse_ctas = in_cta;
            } else if (F->itile && n_cta == n_sm && !strcmp(sweep, "split")) {
                const double slab = 2.0 * G.d * ((double)G.ny * G.nz + (double)G.nx * G.nz + (double)G.nx * G.ny);
                const double b_adj = 52.0 * G.nc + 32.0 * slab;
                const double gcells = (double)(G.ghi[0] - G.glo[0]) * (G.ghi[1] - G.glo[1]) * (G.ghi[2] - G.glo[2]);
                const double b_inv = 1.3 * (64.0 * (double)(G.hi[0] - G.lo[0]) * ny_i * nz_i + 8.0 * gcells);
                int k = (int)std::lround(n_sm * b_inv / (b_adj + b_inv));
                if (const char *e = getenv("FDTD_INV_CTAS")) k = atoi(e);
                k = std::max(1, std::min(k, n_sm / 2));
                const int n_adj_p = n_sm - k;
                if (itotal >= 4LL * k && total >= 8LL * n_adj_p) {
                    std::vector<Segment> psegs;
                    std::vector<int> pbeg;
                    segments_from_runs(nty, nz_i, ib->TX, ib->TY, x0, G.lo[1], G.lo[2],
                                       make_runs(std::vector<double>((size_t)itotal, 1.0), nz_i, k), psegs, pbeg);
                    if ((rc = g->alloc((void **)&F->d_isegs_p, psegs.size() * sizeof(Segment)))) return rc;
                    if ((rc = g->alloc((void **)&F->d_iseg_begin_p, pbeg.size() * sizeof(int)))) return rc;
                    if (cudaMemcpy(F->d_isegs_p, psegs.data(), psegs.size() * sizeof(Segment), cudaMemcpyHostToDevice) != cudaSuccess ||
                        cudaMemcpy(F->d_iseg_begin_p, pbeg.data(), pbeg.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
                        (void)cudaGetLastError();
                        return fdtd_fail(FDTD_ECUDA, "upload of the inverse segment table failed");
                    }
                    F->n_inv_p = k; F->n_adj = n_adj_p;
                    g->pipelined_inverse_ctas = k;
                    const int nty_s = (G.ny + F->TY - 1) / F->TY;
                    segments_from_runs(nty_s, G.nz, F->TX, F->TY, 0, 0, 0, make_runs(model_cost(G, F->TX, F->TY, wy, wz), G.nz, F->n_adj), all, begins);
                    if (cudaMemcpy(F->d_segs[1], all.data(), all.size() * sizeof(Segment), cudaMemcpyHostToDevice) != cudaSuccess ||
                        cudaMemcpy(F->d_seg_begin[1], begins.data(), begins.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
                        (void)cudaGetLastError();
                        return fdtd_fail(FDTD_ECUDA, "upload of the segment table failed");
                    }
                }
            }
        }
    }
    if (F->n_adj == 0) F->n_adj = n_cta;

    // ---- kernel parameters that do not depend on the call -----------------------------------------------------------
    StepParams &P = F->sp;
    P.G = G; P.T = g->T; P.segs = F->d_segs[0]; P.seg_begin = F->d_seg_begin[0];
    P.n_rot = n_rot; P.seg_stride = (int)stride; P.n_cta = n_cta;
    P.step = g->d_step; P.step_next = nullptr; P.step_delta = 0;
    P.nst = F->nst;
    // whole columns dealt out in waves (more tile columns than CTAs): the CTAs of a wave must stay on the same plane for the
    // halo rows to be L2 hits, and a producer that runs a second plane ahead lets them drift: measured at 512^3, forward /
    // adjoint 1494 / 1527 us held against 1700 / 1826 us released early; with lock-step runs (C3) early release wins, 97.8 /
    // 103.8 against 98.6 / 106.4 us
    P.hold = getenv("FDTD_HOLD") ? atoi(getenv("FDTD_HOLD")) : (g->partition == FDTD_PARTITION_WAVES ? 1 : 0);
    P.stage = stage_bytes; P.xs_bytes = xs_bytes; P.xs_pitch = xs_pitch;
    P.dbg = getenv("FDTD_DBG") ? atoi(getenv("FDTD_DBG")) : 0;
    P.dbg_t = nullptr;
    if (best->set_smem(F->smem) != cudaSuccess) {
        (void)cudaGetLastError();
        g->fused_why_not = "cannot reserve shared memory";
        return FDTD_OK;
    }
    g->path = FDTD_PATH_FUSED;
    g->fused_backward_ready = true;
    g->tile_x = F->TX; g->tile_y = F->TY;
    g->tile_z = (int)std::min<long long>(G.nz, total / n_cta);
    if (!getenv("FDTD_NO_CALIBRATE") && total >= 8LL * n_cta) return calibrate(g);
    return FDTD_OK;
}

int fused_alloc_backward(fdtd_grid *g)
{
    FusedState *F = g->fused;
    if (!F || F->lamB) return FDTD_OK;
    return g->alloc((void **)&F->lamB, (size_t)g->G.nc * 6 * sizeof(float));
}

void fused_teardown(fdtd_grid *g)
{
    if (g->fused) {
        for (int q = 0; q < 3; ++q) if (g->fused->h_maps[q]) cudaFreeHost(g->fused->h_maps[q]);
        if (g->fused->maps_done) cudaEventDestroy(g->fused->maps_done);
    }
    delete g->fused;
    g->fused = nullptr;
}

namespace {

// (re)builds one tensor-map table when the volume it was built for changed.
//   which = 0: volumes A/B = fields / bufB;  which = 1: lam / lamB
int build_maps(fdtd_grid *g, int which, float *volA, float *volB, const float *ie, cudaStream_t st)
{
    FusedState *F = g->fused;
    const Dims &G = g->G;
    if (F->maps_key[which][0] == volA && F->maps_key[which][1] == ie) return FDTD_OK;
    const int PW = F->TX + 8, ROWS = F->TY + 2;
    if (cudaEventSynchronize(F->maps_done) != cudaSuccess) { (void)cudaGetLastError(); }   // earlier upload finished
    CUtensorMap *H = F->h_maps[which];
    bool ok = true;
    float *bufs[2] = { volA, volB };
    // components 3-5 (the H-type operand F of phase A) are differenced: boxes with the row below the tile; components 0-2 and
    // inv_eps are read at a thread's own cells only: one row less
    for (int set = 0; set < 2; ++set)
        for (int c = 0; c < 6; ++c)
            ok &= encode3d(&H[set * 6 + c], bufs[set] + (long long)c * G.nc, G.nx, G.ny, G.nz, G.nx,
                           (long long)G.nx * G.ny, PW, c < 3 ? ROWS - 1 : ROWS);
    ok &= encode3d(&H[12], ie, G.nx, G.ny, G.nz, G.nx, (long long)G.nx * G.ny, PW, ROWS - 1);
    if (G.d > 0) {
        // x-slab states (c=z,s=0) and (c=y,s=1): layout [nz][ny][2*dpx], box = whole storage rows of the tile's rows
        for (int set = 0; set < 2; ++set)
            for (int fam = 0; fam < 2; ++fam) {
                const PsiSet &ps = which ? (fam ? g->lpsiH[set] : g->lpsiE[set]) : (fam ? g->psiH[set] : g->psiE[set]);
                const float *xa[2] = { ps.p[2][0], ps.p[1][1] };
                for (int a = 0; a < 2; ++a)
                    ok &= encode3d(&H[13 + set * 4 + fam * 2 + a], xa[a], 2 * G.dpx, G.ny, G.nz, 2 * G.dpx,
                                   (long long)2 * G.dpx * G.ny, 2 * G.dpx, ROWS);
            }
    }
    if (!ok) return fdtd_fail(FDTD_ECUDA, "cuTensorMapEncodeTiled failed");
    cudaError_t e = cudaMemcpyAsync(F->d_maps[which], H, sizeof(CUtensorMap) * 21, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaEventRecord(F->maps_done, st);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, std::string("tensor map upload: ") + cudaGetErrorString(e)); }
    F->maps_key[which][0] = volA; F->maps_key[which][1] = ie;
    return FDTD_OK;
}

// the inverse kernel's table: primal volumes, inv_eps and the lamE' components of both cotangent volumes
int build_inv_maps(fdtd_grid *g, float *volA, float *volB, const float *ie, float *lamA, float *lamB, cudaStream_t st)
{
    FusedState *F = g->fused;
    const Dims &G = g->G;
    if (F->maps_key[2][0] == volA && F->maps_key[2][1] == ie) return FDTD_OK;
    const int TXi = F->itile->TX, TYi = F->itile->TY;
    if (cudaEventSynchronize(F->maps_done) != cudaSuccess) { (void)cudaGetLastError(); }
    CUtensorMap *H = F->h_maps[2];
    bool ok = true;
    float *bufs[2] = { volA, volB }, *lams[2] = { lamA, lamB };
    const long long pl = (long long)G.nx * G.ny;
    // three box shapes (see k_inverse): A [TY+2][TX+8], B [TY+1][TX+4], C [TY][TX]
    for (int set = 0; set < 2; ++set) {
        for (int c = 0; c < 3; ++c)
            ok &= encode3d(&H[set * 3 + c], bufs[set] + (long long)c * G.nc, G.nx, G.ny, G.nz, G.nx, pl, TXi + 8, TYi + 2);
        for (int q = 0; q < 5; ++q) {
            const int comp = q < 3 ? 3 + q : q - 3;                  // H'_x, H'_y, H'_z, E'_x, E'_y
            ok &= encode3d(&H[6 + set * 5 + q], bufs[set] + (long long)comp * G.nc, G.nx, G.ny, G.nz, G.nx, pl, TXi + 4, TYi + 1);
        }
        for (int c = 0; c < 3; ++c)
            ok &= encode3d(&H[17 + set * 3 + c], lams[set] + (long long)c * G.nc, G.nx, G.ny, G.nz, G.nx, pl, TXi, TYi);
    }
    ok &= encode3d(&H[16], ie, G.nx, G.ny, G.nz, G.nx, pl, TXi, TYi);
    if (!ok) return fdtd_fail(FDTD_ECUDA, "cuTensorMapEncodeTiled failed");
    cudaError_t e = cudaMemcpyAsync(F->d_maps[2], H, sizeof(CUtensorMap) * 23, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaEventRecord(F->maps_done, st);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, std::string("tensor map upload: ") + cudaGetErrorString(e)); }
    F->maps_key[2][0] = volA; F->maps_key[2][1] = ie;
    return FDTD_OK;
}

}  // namespace

// Measures the CTAs of both step kernels on scratch volumes and moves the cuts of the work sequence until the
// CTAs finish together: a CTA's measured time is spread over its positions in proportion to the current cost
// estimate, the new cuts equalise that.  Static cost weights cannot capture how the per-plane cost of a slab
// tile depends on what the neighbouring SMs are doing; five rounds of two launches per kernel do (~3 ms at C3).
static int calibrate(fdtd_grid *g)
{
    FusedState *F = g->fused;
    const Dims &G = g->G;
    const size_t vol = (size_t)G.nc * sizeof(float);
    float *T = nullptr, *tie = nullptr;
    if (cudaMalloc((void **)&T, 6 * vol) != cudaSuccess || cudaMalloc((void **)&tie, (G.aniso ? 3 : 1) * vol) != cudaSuccess) {
        (void)cudaGetLastError();
        if (T) cudaFree(T);
        return FDTD_OK;                                   // no room for the scratch volumes: keep the model's cuts
    }
    auto done = [&](int rc) { cudaFree(T); cudaFree(tie); F->maps_key[0][0] = nullptr; return rc; };
    cudaMemset(T, 0, 6 * vol); cudaMemset(F->bufB, 0, 6 * vol); cudaMemset(tie, 0, (G.aniso ? 3 : 1) * vol);
    cudaMemset(g->d_step, 0, sizeof(int));
    int rc;
    for (int q = 0; q < 2; ++q)
        if ((rc = g->zero_psi(g->psiE[q], 0)) || (rc = g->zero_psi(g->psiH[q], 0))) return done(rc);
    if ((rc = build_maps(g, 0, T, F->bufB, tie, 0))) return done(rc);
    StepParams P = F->sp;
    P.maps = F->d_maps[0];
    P.buf[0] = T; P.buf[1] = F->bufB;
    P.ie = tie; P.im = nullptr;
    for (int q = 0; q < 2; ++q) { P.psiE[q] = g->psiE[q]; P.psiH[q] = g->psiH[q]; }
    P.n_src = P.n_det = P.total_freq = 0;
    P.sEl = P.sHl = P.dEl = P.dHl = 1 << 30; P.sEh = P.sHh = P.dEh = P.dHh = -1;
    P.cs = nullptr;
    P.dbg_t = F->d_cta_t;
    std::vector<unsigned long long> t(2 * (size_t)F->n_cta);
    std::vector<Segment> segs;
    std::vector<int> begins;
    const int nty = (G.ny + F->TY - 1) / F->TY;
    const std::vector<int> cls = column_classes(G, F->TX, F->TY);
    // Rounds: first the cost model on a grid of (wy, wz) -- with the lock-step split the cuts move in whole planes
    // for all columns of a class at once, so the span is a rugged function of the weights and the best of a few
    // candidates beats gradient-like feedback (measured on C3: the feedback rounds alone never got below the
    // model's 94.8 us) -- then two feedback rounds from the best candidate.
    static const double cand[][2] = { { 1.0, 0.8 }, { 0.75, 0.55 }, { 0.75, 0.8 }, { 0.75, 1.05 }, { 1.0, 0.55 }, { 1.0, 1.05 },
                                      { 0.5, 0.8 }, { 0.5, 1.05 }, { 1.25, 0.8 }, { 1.25, 1.05 }, { 1.0, 0.3 }, { 0.75, 0.3 } };
    const int n_grid = G.d > 0 ? (int)(sizeof(cand) / sizeof(cand[0])) : 1;
    // (round 2: chaining up to ten damped feedback rounds after the candidates was measured and dropped -- the spans stay
    // at 94-100 us forward and get worse, 104-106 us, for the adjoint kernel: profiles/r2_bound_experiments.md)
    const int cal_iters = getenv("FDTD_CAL_ITERS") ? std::max(1, atoi(getenv("FDTD_CAL_ITERS"))) : n_grid + 2;
    for (int mode = 0; mode < 2; ++mode) {
        const int n_cta = mode ? F->n_adj : F->n_cta;
        P.n_cta = n_cta;
        std::vector<double> w, best_fb;
        Runs runs, best_runs;
        double best = 1e30;
        P.segs = F->d_segs[mode]; P.seg_begin = F->d_seg_begin[mode];
        for (int it = 0; it < cal_iters; ++it) {
            if (it < n_grid) w = model_cost(G, F->TX, F->TY, cand[it][0], cand[it][1]); else w = best_fb;
            runs = make_runs(w, G.nz, n_cta);
            segments_from_runs(nty, G.nz, F->TX, F->TY, 0, 0, 0, runs, segs, begins);
            if (segs.size() > F->seg_cap) continue;
            if (cudaMemcpy(F->d_segs[mode], segs.data(), segs.size() * sizeof(Segment), cudaMemcpyHostToDevice) != cudaSuccess ||
                cudaMemcpy(F->d_seg_begin[mode], begins.data(), begins.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess)
                return done(fdtd_fail(FDTD_ECUDA, "calibration: upload of the segment table failed"));
            for (int rep = 0; rep < 3; ++rep) {           // the timestamps of the last launch stay
                if (mode) F->tile->launch_adj(P, n_cta, F->smem, 0); else F->tile->launch_fwd(P, n_cta, F->smem, 0);
            }
            if (cudaDeviceSynchronize() != cudaSuccess ||
                cudaMemcpy(t.data(), F->d_cta_t, 2 * (size_t)n_cta * sizeof(unsigned long long), cudaMemcpyDeviceToHost) != cudaSuccess) {
                cudaError_t e = cudaGetLastError();
                return done(fdtd_fail(FDTD_ECUDA, std::string("calibration launch: ") + cudaGetErrorString(e)));
            }
            unsigned long long t0 = ~0ull, t1 = 0;
            for (int c = 0; c < n_cta; ++c) { t0 = std::min(t0, t[2 * c]); t1 = std::max(t1, t[2 * c + 1]); }
            const double span = (double)(t1 - t0) * 1e-3;
            if (getenv("FDTD_VERBOSE") && atoi(getenv("FDTD_VERBOSE")) > 1) fprintf(stderr, "fdtd:   calibration round %d: %.1f us\n", it, span);
            // spread each CTA's time over its positions in proportion to the current estimate; columns of a class
            // then share the mean profile (identical cuts keep them in lock step)
            for (int c = 0; c < n_cta; ++c) {
                double sum = 0.0;
                for (const std::pair<long long, long long> &r : runs[c]) for (long long q = r.first; q < r.second; ++q) sum += w[q];
                const double scale = (double)(t[2 * c + 1] - t0) / sum;
                for (const std::pair<long long, long long> &r : runs[c]) for (long long q = r.first; q < r.second; ++q) w[q] *= scale;
            }
            average_classes(w, cls, G.nz);
            if (span < best) { best = span; best_runs = runs; best_fb = w; if (mode == 0) g->partition = t_partition_kind; }
        }
        if (best_runs.empty()) return done(fdtd_fail(FDTD_ECUDA, "calibration: no partition fits the segment table"));
        segments_from_runs(nty, G.nz, F->TX, F->TY, 0, 0, 0, best_runs, segs, begins);
        if (cudaMemcpy(F->d_segs[mode], segs.data(), segs.size() * sizeof(Segment), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(F->d_seg_begin[mode], begins.data(), begins.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess)
            return done(fdtd_fail(FDTD_ECUDA, "calibration: upload of the segment table failed"));
        F->calibrated_us[mode] = best;
        if (getenv("FDTD_VERBOSE")) fprintf(stderr, "fdtd: calibrated %s step kernel: %.1f us per launch\n", mode ? "adjoint" : "forward", best);
        if (getenv("FDTD_VERBOSE") && atoi(getenv("FDTD_VERBOSE")) > 2) {
            // per-CTA durations of four successive launches of the final partition: is a slow CTA slow every time?
            std::vector<std::vector<double>> dur(4, std::vector<double>(n_cta));
            for (int rep = 0; rep < 4; ++rep) {
                if (mode) F->tile->launch_adj(P, n_cta, F->smem, 0); else F->tile->launch_fwd(P, n_cta, F->smem, 0);
                cudaDeviceSynchronize();
                cudaMemcpy(t.data(), F->d_cta_t, 2 * (size_t)n_cta * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
                for (int c = 0; c < n_cta; ++c) dur[rep][c] = (double)(t[2 * c + 1] - t[2 * c]) * 1e-3;
            }
            for (int c = 0; c < n_cta; ++c) {
                double cost = 0.0;
                for (const std::pair<long long, long long> &r : best_runs[c]) cost += (double)(r.second - r.first);
                fprintf(stderr, "fdtd:   cta %3d planes %5.0f segs %zu durations %.1f %.1f %.1f %.1f\n", c, cost, best_runs[c].size(),
                        dur[0][c], dur[1][c], dur[2][c], dur[3][c]);
            }
        }
    }
    cudaMemset(F->bufB, 0, 6 * vol);
    return done(FDTD_OK);
}

// run_steps lives in fdtd_api.cu; reached through small trampolines
int fdtd_run_steps_fwd(fdtd_grid *g, const std::string &key, int n_steps, int launches_per_step, cudaStream_t st,
                       void (*enqueue)(void *, cudaStream_t), void *ctx);
int fdtd_run_steps_bwd(fdtd_grid *g, const std::string &key, int n_steps, int launches_per_step, cudaStream_t st,
                       void (*enqueue)(void *, cudaStream_t), void *ctx);

namespace {
// fork: the side streams wait for what the main stream has enqueued so far; join: the main stream waits for them.
// While profiling everything stays on the main stream's timeline between the two events of the caller's ProfScope
// (the side streams still run concurrently: the span measures the group).
void fork_side(fdtd_grid *g, cudaStream_t cs, int n_side)
{
    cudaEventRecord(g->fork_ev, cs);
    for (int q = 0; q < n_side; ++q) cudaStreamWaitEvent(g->side_stream[q], g->fork_ev, 0);
}
void join_side(fdtd_grid *g, cudaStream_t cs, int n_side)
{
    for (int q = 0; q < n_side; ++q) {
        cudaEventRecord(g->join_ev[q], g->side_stream[q]);
        cudaStreamWaitEvent(cs, g->join_ev[q], 0);
    }
}

// N3: the attached neighbours of the volumes this sweep writes (which = 0 primal, 1 cotangents)
void set_peers(const fdtd_grid *g, int which, StepParams &P)
{
    P.peer_on = 0;
    P.own_lo = g->desc.z_ghost_lo; P.own_hi = g->G.nz - 1 - g->desc.z_ghost_hi;
    for (int sd = 0; sd < 2; ++sd) {
        const fdtd_grid::PeerLink &L = g->peer[which][sd];
        P.peer[sd][0] = L.vol[0]; P.peer[sd][1] = L.vol[1]; P.peer_nc[sd] = L.nc;
        if (L.vol[0]) P.peer_on |= 1 << sd;
    }
}

// N3, device-side ordering of the slabs (halo_sync.cu): active when every attached side has a flag
struct HaloSync {                                   // (no padding: it is part of the graph key)
    const int *mine[2] = { nullptr, nullptr };      // my flags, written by the neighbour below / above
    int *theirs[2] = { nullptr, nullptr };          // my flag in the set of the neighbour below / above
    int *err = nullptr;
    long long active = 0;
};
HaloSync halo_sync_of(const fdtd_grid *g, int which, int peer_on)
{
    HaloSync H;
    if (!peer_on || !g->d_hflags) return H;
    for (int sd = 0; sd < 2; ++sd) {
        if (!((peer_on >> sd) & 1)) continue;
        if (!g->peer[which][sd].flag) return HaloSync{};      // a side without a flag: the host orders the steps
        H.mine[sd] = g->d_hflags + which * 2 + sd;
        H.theirs[sd] = g->peer[which][sd].flag;
    }
    H.active = 1; H.err = g->d_herr;
    return H;
}

struct FwdCtx {
    fdtd_grid *g; StepParams P; bool recording; float *A; float *B; int n_steps;
    const std::vector<TimeDetDev> *TD; const float *ie; const float *im;
    HaloSync hs;
};
// forward step n; with the recorder on, k_record_pipe runs beside it on a side stream: both only read buffer n&1
// (pre-step H of step n -> rec[n], E' of step n-1 -> rec[n-1]); the step after next overwrites that buffer, so the
// join comes before the next step.  fused_forward() adds the last E' record after the loop.
void enqueue_fwd(void *vctx, cudaStream_t cs)
{
    FwdCtx *c = (FwdCtx *)vctx;
    fdtd_grid *g = c->g;
    FusedState *F = g->fused;
    StepParams Q = c->P;
    Q.step = g->step_in(); Q.step_next = g->step_out(); Q.step_delta = 1;
    // N3: the neighbours must have reached state n (their step n-1 stored my ghost planes) before anything reads buffer n&1
    if (c->hs.active) launch_halo_wait(c->hs.mine[0], c->hs.mine[1], g->step_in(), 0, 0, 1, c->hs.err, cs);
    ProfScope p(g, fdtd_grid::PC_FUSED_FWD, cs);
    if (c->recording) {
        fork_side(g, cs, 1);
        launch_record_pipe(g->G, g->R, c->A, c->B, g->rec, g->step_in(), c->n_steps, g->side_stream[0]);
    }
    F->tile->launch_fwd(Q, F->n_cta, F->smem, cs);
    if (c->recording) join_side(g, cs, 1);
    if (c->hs.active) launch_halo_signal(c->hs.theirs[0], c->hs.theirs[1], g->step_in(), 1, cs);      // state n+1 reached
    // N2: time-domain detectors on the state step n just wrote (volume (n+1)&1)
    for (const TimeDetDev &q : *c->TD) launch_time_detect(g->G, c->A, c->B, 1, c->ie, c->im, q, g->red, g->step_in(), cs);
    // N4, replay of a segment in the checkpointed reverse sweep: D = dE'/d inv_eps of step n from the two volumes
    if (g->ck_store) {
        launch_dE_store(g->G, c->A, c->B, g->dE, g->ck_every, 0, c->ie, g->sigma, g->step_in(), cs);
        for (int q = 0; q < c->P.n_src; ++q)
            if (c->P.src[q].comp < 3) launch_dE_source(g->G, g->dE, g->ck_every, c->P.src[q], c->ie, g->sigma, g->step_in(), cs);
    }
    ++g->enq_step;
}

struct BwdCtx {
    fdtd_grid *g; StepParams P; InvParams I; bool fused_inv; bool fused_det; bool pipelined; bool want_grad; float *bufB; float *fields; const float *ie; const float *im; float *grad; float *lamA; float *lamB;
    const std::vector<SourceDev> *S; const std::vector<DetectorDev> *D; int total_freq;
    const std::vector<TimeDetDev> *TD; float *grad_mu;
    HaloSync hs; int n_total;
};
// Reverse step n.  One kernel after the other: B1 (detector cotangents into the volume about to be read), B2+B5
// (fused adjoint step), face injection, then the primal inverse step B3+B4 with lamE' taken from the volume the
// adjoint step just wrote.
// Pipelined (c->pipelined; see fused_setup for the variants): launch n is a group of three kernels without an
// order among them, the adjoint step n (n_adj CTAs), the inverse step n+1 (n_inv_p CTAs; nothing at the first
// launch) and the face injection for step n.  All three
// depend only on launch n+1: inverse step n+1 reads primal volume n&1 and the lamE' that adjoint step n+1 wrote
// into cotangent volume (n+1)&1 (adjoint step n only reads it) and writes the box of primal volume (n+1)&1; the
// injection for step n writes cells outside the box of that same volume.  fused_backward() adds inverse step 0.
void enqueue_bwd(void *vctx, cudaStream_t cs)
{
    BwdCtx *c = (BwdCtx *)vctx;
    fdtd_grid *g = c->g;
    FusedState *F = g->fused;
    const Dims &G = g->G;
    StepParams Q = c->P;
    Q.step = g->step_in(); Q.step_next = g->step_out(); Q.step_delta = -1;
    // N3: reverse step n reads the cotangents of state n+1; the seed (state n_total) is the caller's
    if (c->hs.active) launch_halo_wait(c->hs.mine[0], c->hs.mine[1], g->step_in(), 1, c->n_total, -1, c->hs.err, cs);
    if (c->pipelined) {
        ProfScope p(g, fdtd_grid::PC_FUSED_BWD, cs);
        const int n_side = G.d > 0 ? 2 : 1;
        fork_side(g, cs, n_side);
        InvParams J = c->I;
        J.step = g->step_in();
        F->itile->launch_inv(J, F->n_inv_p, F->ismem, g->side_stream[0]);
        if (G.d > 0) launch_inject_pipe(G, g->R, c->fields, c->bufB, g->rec, g->step_in(), g->side_stream[1]);
        F->tile->launch_adj(Q, F->n_adj, F->smem, cs);
        join_side(g, cs, n_side);
        if (c->hs.active) launch_halo_signal(c->hs.theirs[0], c->hs.theirs[1], g->step_in(), 0, cs);      // state n reached
        ++g->enq_step; ++g->enq_inv;
        return;
    }
    // N2 transposes first: they act on the state after step n (primal volume (n+1)&1 when the fused inverse step
    // ping-pongs, else `fields`), into the cotangent volume the adjoint step is about to read ((n+1)&1)
    if (!c->TD->empty()) { ProfScope p(g, fdtd_grid::PC_SRC_DET, cs);
      for (const TimeDetDev &q : *c->TD)
          launch_time_detect_adjoint(G, c->lamA, c->lamB, c->fields, c->fused_inv ? c->bufB : nullptr, 1, c->ie, c->im,
                                     c->im != nullptr, q, c->grad, g->step_in(), cs); }
    if (!c->fused_det) { ProfScope p(g, fdtd_grid::PC_SRC_DET, cs);
      for (const DetectorDev &dt : *c->D)
          if (dt.phasor) launch_detector_adjoint_pp(G, c->lamA, c->lamB, dt, g->d_cs, c->total_freq, g->step_in(), c->im, cs); }
    // the face injection (it writes cells of the primal volume, which the adjoint step never touches) runs beside it
    const bool side_inject = c->fused_inv && G.d > 0;       // fused_inv implies want_grad
    { ProfScope p(g, fdtd_grid::PC_FUSED_BWD, cs);
      if (side_inject) {
          fork_side(g, cs, 1);
          launch_inject_pipe(G, g->R, c->fields, c->bufB, g->rec, g->step_in(), g->side_stream[0]);
      }
      F->tile->launch_adj(Q, F->n_adj, F->smem, cs);
      ++g->enq_step;
      if (side_inject) join_side(g, cs, 1); }
    if (c->hs.active) launch_halo_signal(c->hs.theirs[0], c->hs.theirs[1], g->step_in(), 0, cs);          // state n reached
    // N4, checkpointed reverse sweep: g += lamE' . D with lamE' in the volume the adjoint step just wrote (n&1), or, for a
    // lossy medium (the volume holds Ca lamE'), in the scratch volumes
    if (g->ck_gradhook) { ProfScope p(g, fdtd_grid::PC_INV_E_GRAD, cs);
      launch_grad_from_dE(G, Q.e2_out ? Q.e2_out : c->lamA, Q.e2_out ? Q.e2_out : c->lamB, g->dE, g->ck_every, g->ck_gradhook, g->step_in(), cs); }
    if (c->fused_inv) {
        InvParams J = c->I;
        J.step = g->step_in();
        { ProfScope p(g, fdtd_grid::PC_FUSED_INV, cs); F->itile->launch_inv(J, F->in_cta, F->ismem, cs); }
        ++g->enq_inv;
        return;
    }
    if (!c->want_grad) return;
    { ProfScope p(g, fdtd_grid::PC_SRC_DET, cs);
      for (const SourceDev &s : *c->S) if (s.comp >= 3) launch_add_source(G, c->fields, s, g->step_in(), -1.f, cs); }
    if (G.d > 0) { ProfScope p(g, fdtd_grid::PC_INJECT, cs); launch_inject(G, g->R, c->fields, g->rec, g->step_in(), cs); }
    // N4: the cotangent of the post-step H is still in the volume adjoint step n read, (n+1)&1 (scaled by im with inv_mu)
    { ProfScope p(g, fdtd_grid::PC_INV_H, cs);
      launch_inv_H(G, c->fields, c->im, cs, c->lamA, c->lamB, g->step_in(), c->im != nullptr, c->grad_mu); }
    { ProfScope p(g, fdtd_grid::PC_SRC_DET, cs);
      for (const SourceDev &s : *c->S) if (s.comp < 3) launch_add_source(G, c->fields, s, g->step_in(), -1.f, cs); }
    { ProfScope p(g, fdtd_grid::PC_INV_E_GRAD, cs);
      launch_inv_E_grad_pp(G, c->fields, c->ie, c->lamA, c->lamB, g->step_in(), c->grad, cs); }
}
}  // namespace

int fused_forward(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                  const std::vector<SourceDev> &S, const std::vector<DetectorDev> &D, const std::vector<TimeDetDev> &TD,
                  int total_freq, int n_begin, int n_end, int n_total, bool recording, cudaStream_t st)
{
    // steps n_begin .. n_end-1 of a run of n_total; state n lives in volume n&1 (0: fields, 1: the grid's copy) between
    // the calls of a range sequence and is brought back to `fields` by the call that ends the run
    const int n_steps = n_total, n_count = n_end - n_begin;
    FusedState *F = g->fused;
    if ((int)S.size() > MAX_SRC || (int)D.size() > MAX_DET)
        return fdtd_fail(FDTD_EINVAL, "the fused path takes at most 4 sources and 4 detectors (use FDTD_PATH_GENERIC)");
    int rc = build_maps(g, 0, fields, F->bufB, inv_eps, st);
    if (rc) return rc;
    for (int q = 0; q < 2 && n_begin == 0; ++q)
        if ((rc = g->zero_psi(g->psiE[q], st)) || (rc = g->zero_psi(g->psiH[q], st))) return rc;
    FwdCtx ctx{ g, F->sp, recording, fields, F->bufB, n_steps, &TD, inv_eps, inv_mu };
    StepParams &P = ctx.P;
    P.maps = F->d_maps[0];
    P.buf[0] = fields; P.buf[1] = F->bufB;
    P.ie = inv_eps; P.im = inv_mu; P.sigma = g->sigma; P.e2_out = nullptr;
    for (int q = 0; q < 2; ++q) { P.psiE[q] = g->psiE[q]; P.psiH[q] = g->psiH[q]; }
    P.n_src = (int)S.size(); P.n_det = (int)D.size(); P.total_freq = total_freq;
    for (size_t q = 0; q < S.size(); ++q) P.src[q] = S[q];
    for (size_t q = 0; q < D.size(); ++q) P.det[q] = D[q];
    P.cs = g->d_cs;
    set_peers(g, 0, P);
    ctx.hs = halo_sync_of(g, 0, P.peer_on);
    if (ctx.hs.active && n_total < 3) return fdtd_fail(FDTD_EINVAL, "device-side ordering of the slabs (fdtd_halo_attach_flags) needs runs of at least 3 steps");
    if (P.peer_on && n_count > 1 && !ctx.hs.active)
        return fdtd_fail(FDTD_EINVAL, "with attached neighbours (fdtd_halo_attach) and no flags (fdtd_halo_attach_flags) a range call advances one step: the caller orders the slabs after every step");
    P.sEl = P.sHl = P.dEl = P.dHl = 1 << 30; P.sEh = P.sHh = P.dEh = P.dHh = -1;
    for (const SourceDev &q : S) {
        if (q.comp < 3) { P.sEl = std::min(P.sEl, q.lo[2]); P.sEh = std::max(P.sEh, q.hi[2]); }
        else { P.sHl = std::min(P.sHl, q.lo[2]); P.sHh = std::max(P.sHh, q.hi[2]); }
    }
    for (const DetectorDev &q : D) {
        if (q.mask & 7) { P.dEl = std::min(P.dEl, q.lo[2]); P.dEh = std::max(P.dEh, q.hi[2]); }
        if (q.mask >> 3) { P.dHl = std::min(P.dHl, q.lo[2]); P.dHh = std::max(P.dHh, q.hi[2]); }
    }
    std::string key("ff");
    key.append((const char *)&P, sizeof(P));
    key.push_back(recording ? 1 : 0);
    key.append((const char *)&n_steps, recording ? sizeof(n_steps) : 0);
    if (!TD.empty()) key.append((const char *)TD.data(), TD.size() * sizeof(TimeDetDev));
    int n_store = 0;
    if (g->ck_store) { n_store = 1; for (const SourceDev &q : S) if (q.comp < 3) ++n_store; }
    key.push_back((char)n_store);
    key.append((const char *)&ctx.hs, sizeof(ctx.hs));
    rc = fdtd_run_steps_fwd(g, key, n_count, 1 + (recording ? 1 : 0) + (int)TD.size() + n_store + (ctx.hs.active ? 2 : 0), st, enqueue_fwd, &ctx);
    if (rc) return rc;
    if (n_end != n_total || g->replaying) return FDTD_OK;      // (replaying: the checkpointed reverse sweep leaves the state in its volume)
    if (recording) {      // E' of the last step; the p-th step of the call read counter slot p&1, so the count sits in slot n_count&1
        ProfScope p(g, fdtd_grid::PC_RECORD, st);
        launch_record_pipe(g->G, g->R, fields, F->bufB, g->rec, g->d_step + (n_count & 1), n_steps, st);
        g->kernel_launches += 1;
    }
    if (n_steps & 1) {
        cudaError_t e = cudaMemcpyAsync(fields, F->bufB, (size_t)g->G.nc * 6 * sizeof(float), cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, cudaGetErrorString(e)); }
    }
    return FDTD_OK;
}

// The cotangent seed is in g->lam; reverse step n reads volume (n+1)&1 and writes n&1, so after step 0 the
// result is back in volume 0 = g->lam.
int fused_backward(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                   const std::vector<SourceDev> &S, const std::vector<DetectorDev> &D, const std::vector<TimeDetDev> &TD,
                   int total_freq, int n_hi, int n_lo, int n_total, float *dL_dinv_eps, bool seeded_H, cudaStream_t st,
                   float *dL_dinv_mu)
{
    // reverse steps n_hi-1 .. n_lo of a run of n_total (fdtd_backward: n_steps-1 .. 0).  Between the calls of a range
    // sequence the cotangents after reverse step n live in volume n&1 (0: g->lam) and the reconstructed state n in
    // primal volume n&1 (0: fields); the seed and state n_total are placed by the call that starts at n_total.
    const int n_steps = n_total, n_count = n_hi - n_lo;
    const bool first = n_hi == n_total, whole = first && n_lo == 0;
    FusedState *F = g->fused;
    const size_t vol6 = (size_t)g->G.nc * 6 * sizeof(float);
    int rc;
    if ((rc = fused_alloc_backward(g))) return rc;
    if ((rc = build_maps(g, 1, g->lam, F->lamB, inv_eps, st))) return rc;
    // with inv_mu the sweep runs on Lambda_H = im lamH (see k_step); fdtd_backward scales the result back
    // (the seed sits in the volume of state n_steps already -- fdtd_api.cu seeds fused_volume(.., 1, n_steps) -- so that nothing
    // is written to the other volume before the first step: with N3 peer stores a neighbour's first step may already have
    // stored its boundary plane there)
    if (first && inv_mu && seeded_H) launch_scale_H(g->G, (n_steps & 1) ? F->lamB : g->lam, inv_mu, false, st);
    const bool want_grad = dL_dinv_eps != nullptr;      // false: adjoint sweep only, the primal volumes are not touched
    // N4: dL/d inv_mu is formed in the inverse step from lamH' of volume (n+1)&1, which adjoint step n-1 overwrites: the
    // inverse step of step n must then run before adjoint step n-1 (no pipelined sweep)
    const bool fused_inv = want_grad && F->itile != nullptr && (int)S.size() <= MAX_SRC && !getenv("FDTD_GENERIC_INVERSE");
    // B1 inside the adjoint kernel when every detector with a cotangent is on E components (else a kernel per detector)
    bool fused_det = (int)D.size() <= MAX_DET;
    for (const DetectorDev &dt : D) if (dt.phasor && (dt.mask >> 3)) fused_det = false;
    // while profiling (events around every launch) the kernels run one after the other, so each is timed alone
    // (time-domain detector transposes read the primal state after step n, which the pipelined sweep is still writing)
    const bool pipelined = fused_inv && fused_det && F->n_inv_p > 0 && !g->profiling && TD.empty() && whole && !dL_dinv_mu;
    BwdCtx ctx{ g, F->sp, F->ip, fused_inv, fused_det, pipelined, want_grad, F->bufB, fields, inv_eps, inv_mu, dL_dinv_eps, g->lam, F->lamB, &S, &D, total_freq, &TD, dL_dinv_mu };
    if (fused_inv) {
        // reverse step n reads primal volume (n+1)&1 and writes n&1: state n_steps must sit in volume n_steps&1
        if ((rc = build_inv_maps(g, fields, F->bufB, inv_eps, g->lam, F->lamB, st))) return rc;
        if (first && (n_steps & 1)) {
            cudaError_t e = cudaMemcpyAsync(F->bufB, fields, vol6, cudaMemcpyDeviceToDevice, st);
            if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, cudaGetErrorString(e)); }
        }
        InvParams &I = ctx.I;
        I.maps = F->d_maps[2];
        I.buf[0] = fields; I.buf[1] = F->bufB; I.grad = dL_dinv_eps; I.im = inv_mu; I.ie = inv_eps;
        I.gmu = dL_dinv_mu; I.lamH[0] = g->lam + 3 * (size_t)g->G.nc; I.lamH[1] = F->lamB + 3 * (size_t)g->G.nc;
        I.n_src = (int)S.size();
        I.sEl = I.sHl = 1 << 30; I.sEh = I.sHh = -1;
        for (size_t q = 0; q < S.size(); ++q) {
            I.src[q] = S[q];
            if (S[q].comp < 3) { I.sEl = std::min(I.sEl, S[q].lo[2]); I.sEh = std::max(I.sEh, S[q].hi[2]); }
            else { I.sHl = std::min(I.sHl, S[q].lo[2]); I.sHh = std::max(I.sHh, S[q].hi[2]); }
        }
        if (pipelined) { I.segs = F->d_isegs_p; I.seg_begin = F->d_iseg_begin_p; I.bias = 1; I.n_steps = n_steps; }
    }
    StepParams &P = ctx.P;
    P.maps = F->d_maps[1];
    P.segs = F->d_segs[1]; P.seg_begin = F->d_seg_begin[1];
    P.buf[0] = g->lam; P.buf[1] = F->lamB;
    P.ie = inv_eps; P.im = inv_mu; P.sigma = g->sigma; P.e2_out = g->sigma ? g->ck_e2 : nullptr;
    for (int q = 0; q < 2; ++q) { P.psiE[q] = g->lpsiE[q]; P.psiH[q] = g->lpsiH[q]; }
    P.n_src = 0; P.n_det = 0; P.total_freq = total_freq;
    P.sEl = P.sHl = P.dEl = P.dHl = 1 << 30; P.sEh = P.sHh = P.dEh = P.dHh = -1;
    if (fused_det) {
        P.n_det = (int)D.size();
        for (size_t q = 0; q < D.size(); ++q) {
            P.det[q] = D[q];
            if (D[q].phasor) { P.dEl = std::min(P.dEl, D[q].lo[2]); P.dEh = std::max(P.dEh, D[q].hi[2]); }
        }
    }
    P.cs = g->d_cs;
    set_peers(g, 1, P);
    ctx.hs = halo_sync_of(g, 1, P.peer_on);
    if (ctx.hs.active && n_total < 3) return fdtd_fail(FDTD_EINVAL, "device-side ordering of the slabs (fdtd_halo_attach_flags) needs runs of at least 3 steps");
    ctx.n_total = n_total;
    if (P.peer_on && n_count > 1 && !ctx.hs.active)
        return fdtd_fail(FDTD_EINVAL, "with attached neighbours (fdtd_halo_attach) and no flags (fdtd_halo_attach_flags) a range call advances one step: the caller orders the slabs after every step");
    int n_adj = 0;
    for (const DetectorDev &dt : D) if (dt.phasor) ++n_adj;
    std::string key(fused_inv ? "fB" : "fb");
    key.append((const char *)&P, sizeof(P));
    if (fused_inv) key.append((const char *)&ctx.I, sizeof(ctx.I));
    key.append((const char *)&fields, sizeof(fields));
    key.append((const char *)&dL_dinv_eps, sizeof(dL_dinv_eps));
    key.append((const char *)&dL_dinv_mu, sizeof(dL_dinv_mu));
    key.append((const char *)&g->ck_gradhook, sizeof(g->ck_gradhook));
    if (!S.empty()) key.append((const char *)S.data(), S.size() * sizeof(SourceDev));
    if (!D.empty()) key.append((const char *)D.data(), D.size() * sizeof(DetectorDev));
    if (!TD.empty()) key.append((const char *)TD.data(), TD.size() * sizeof(TimeDetDev));
    const int n_inj = g->G.d > 0 ? 1 : 0;
    key.append((const char *)&ctx.hs, sizeof(ctx.hs));
    key.append((const char *)&ctx.n_total, sizeof(ctx.n_total));
    const int launches = (ctx.hs.active ? 2 : 0) + (int)TD.size() + (g->ck_gradhook ? 1 : 0) + (!want_grad ? 1 + (fused_det ? 0 : n_adj)
                         : (fused_inv ? 2 + (fused_det ? 0 : n_adj) + n_inj : 3 + (fused_det ? 0 : n_adj) + (int)S.size() + n_inj));
    rc = fdtd_run_steps_bwd(g, key, n_count, launches, st, enqueue_bwd, &ctx);
    if (rc || !pipelined) return rc;
    // inverse step 0 on every SM; reverse step p read counter slot p&1 (p counted from the end), so -1 sits in slot n_steps&1
    InvParams J = ctx.I;
    J.segs = F->d_isegs; J.seg_begin = F->d_iseg_begin;
    J.step = g->d_step + (n_steps & 1);
    { ProfScope p(g, fdtd_grid::PC_FUSED_INV, st); F->itile->launch_inv(J, F->in_cta, F->ismem, st); }
    g->kernel_launches += 1;
    g->fused_inverse_launches += 1;
    return FDTD_OK;
}

float *fused_volume(fdtd_grid *g, float *fields, int which, int n)
{
    FusedState *F = g->fused;
    if (which == 0) return (n & 1) ? F->bufB : fields;
    return (n & 1) ? F->lamB : g->lam;
}
