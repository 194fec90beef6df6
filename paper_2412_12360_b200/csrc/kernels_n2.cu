// kernels_n2.cu -- the paper's source / detector set beyond the running DFT:
//   time-domain snapshot and energy detectors with their transposes ("access to intermediate fields,
//   energy, Poynting flux"; reading R23), Poynting flux through a plane from the DFT phasors with and without
//   Yee co-location (L70, L148; reading R24) and its VJP, and the auxiliary 1-D leapfrog that generates the two
//   waveforms of a one-directional TFSF plane source (L72, L130; reading R25).
// Product code: shares nothing with oracle/.
#include <algorithm>
#include "fdtd_internal.h"

namespace fdtd {

namespace {

__device__ __forceinline__ long long lin(const Dims &G, int i, int j, int k)
{
    return ((long long)k * G.ny + j) * G.nx + i;
}

// Sum of the per-thread values `v` over the whole launch, written to *out by the block that finishes last:
// block partials in fixed slots, summed in slot order, so the result does not depend on the block schedule.
__device__ void block_sum_to(double v, const ReduceScratch &rs, float *out)
{
    __shared__ double sh[32];
    __shared__ bool last;
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = lane < (int)(blockDim.x >> 5) ? sh[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) {
            rs.partial[blockIdx.x] = v;
            __threadfence();
            last = atomicAdd(rs.ticket, 1u) == gridDim.x - 1;
        }
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double s = 0.0;
    for (unsigned b = threadIdx.x; b < gridDim.x; b += blockDim.x) s += *((volatile double *)rs.partial + b);
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    __syncthreads();
    if (lane == 0) sh[warp] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
        *out = (float)t;
        *rs.ticket = 0u;
    }
}

// ------------------------------------------------------------------------------------------ snapshot
template <bool ADJ>
__global__ void k_snapshot(Dims G, float *__restrict__ vA, float *__restrict__ vB, int par_off, TimeDetDev td,
                           const int *__restrict__ step, const float *__restrict__ scale_H)
{
    const int n = *step;
    if ((n + 1) % td.stride) return;
    float *v = (vB && ((n + par_off) & 1)) ? vB : vA;
    const long long rec = (n + 1) / td.stride - 1;
    const int bx = td.hi[0] - td.lo[0], by = td.hi[1] - td.lo[1], bz = td.hi[2] - td.lo[2];
    const long long bc = (long long)bx * by * bz;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < bc; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % bx), j = (int)((t / bx) % by), k = (int)(t / ((long long)bx * by));
        const long long p = lin(G, td.lo[0] + i, td.lo[1] + j, td.lo[2] + k);
        int ci = 0;
        for (int c = 0; c < 6; ++c) {
            if (!((td.mask >> c) & 1)) continue;
            float *o = td.out + (rec * td.ncomp + ci) * bc + t;
            if (!ADJ) *o = v[c * G.nc + p];
            else v[c * G.nc + p] += (scale_H && c >= 3) ? *o * __ldg(scale_H + p) : *o;
            ++ci;
        }
    }
}

// ------------------------------------------------------------------------------------------ energy
// W = sum_cells 1/2 (sum_c E_c^2 / ie + H_c^2 / im), six components at the same index (L70: no co-location)
__global__ void __launch_bounds__(256) k_energy(Dims G, const float *__restrict__ vA, const float *__restrict__ vB, int par_off,
                                                const float *__restrict__ ie, const float *__restrict__ im, TimeDetDev td,
                                                ReduceScratch rs, const int *__restrict__ step)
{
    const int n = *step;
    if ((n + 1) % td.stride) return;
    const float *v = (vB && ((n + par_off) & 1)) ? vB : vA;
    const int bx = td.hi[0] - td.lo[0], by = td.hi[1] - td.lo[1], bz = td.hi[2] - td.lo[2];
    const long long bc = (long long)bx * by * bz;
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < bc; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % bx), j = (int)((t / bx) % by), k = (int)(t / ((long long)bx * by));
        const long long p = lin(G, td.lo[0] + i, td.lo[1] + j, td.lo[2] + k);
        float e2 = 0.f, h2 = 0.f;
        for (int c = 0; c < 3; ++c) {
            const float E = v[c * G.nc + p], H = v[(3 + c) * G.nc + p];
            e2 = fmaf(E, E, e2); h2 = fmaf(H, H, h2);
        }
        acc += 0.5 * ((double)e2 / (double)__ldg(ie + p) + (double)h2 / (im ? (double)__ldg(im + p) : 1.0));
    }
    block_sum_to(acc, rs, td.out + ((n + 1) / td.stride - 1));
}

// transpose: lamE_c += G E_c / ie, lamH_c += G H_c / im (im lamH_c += G H_c when the sweep carries im lamH), and
// the explicit dependence on ie: g += G (-1/2) sum_c E_c^2 / ie^2 on the gradient box
__global__ void k_energy_adjoint(Dims G, float *__restrict__ lA, float *__restrict__ lB, const float *__restrict__ fA,
                                 const float *__restrict__ fB, int par_off, const float *__restrict__ ie,
                                 const float *__restrict__ im, int scaled_H, TimeDetDev td, float *__restrict__ g,
                                 const int *__restrict__ step)
{
    const int n = *step;
    if ((n + 1) % td.stride) return;
    const bool odd = (n + par_off) & 1;
    float *lam = (lB && odd) ? lB : lA;
    const float *f = (fB && odd) ? fB : fA;
    const float Gq = __ldg(td.out + ((n + 1) / td.stride - 1));
    const int bx = td.hi[0] - td.lo[0], by = td.hi[1] - td.lo[1], bz = td.hi[2] - td.lo[2];
    const long long bc = (long long)bx * by * bz;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < bc; t += (long long)gridDim.x * blockDim.x) {
        const int i = td.lo[0] + (int)(t % bx), j = td.lo[1] + (int)((t / bx) % by), k = td.lo[2] + (int)(t / ((long long)bx * by));
        const long long p = lin(G, i, j, k);
        const float e = __ldg(ie + p), re = 1.f / e;
        const float rm = (im && !scaled_H) ? 1.f / __ldg(im + p) : 1.f;
        float e2 = 0.f;
        for (int c = 0; c < 3; ++c) {
            const float E = f[c * G.nc + p], H = f[(3 + c) * G.nc + p];
            lam[c * G.nc + p] += Gq * E * re;
            lam[(3 + c) * G.nc + p] += Gq * H * rm;
            e2 = fmaf(E, E, e2);
        }
        const bool ing = i >= G.glo[0] && i < G.ghi[0] && j >= G.glo[1] && j < G.ghi[1] && k >= G.glo[2] && k < G.ghi[2];
        if (g && ing) g[p] += Gq * -0.5f * e2 * re * re;
    }
}

// ------------------------------------------------------------------------------------------ Poynting flux (R24)
// The detector box is a slab normal to `axis` a (one plane thick, or two with co-location) whose mask holds the
// tangential components E_b, E_c, H_b, H_c; slots = index of each among the detector's components.
struct FluxGeom {
    int ext[3];
    int a, t1;                 // normal axis, plane of E (and of the upper H) inside the box
    int sEb, sEc, sHb, sHc, ncomp;
    long long bc;
    int interpolate;
    float cw, sw;              // cos, sin(omega_f / 2): H is stamped half a step late
};

__device__ __forceinline__ bool flux_cell(const FluxGeom &q, long long t, long long &cell, long long &cellm)
{
    const long long plane_cells = q.bc / q.ext[q.a];
    if (t >= plane_cells) return false;
    int u = (q.a + 1) % 3, v = (q.a + 2) % 3;
    if (u > v) { const int w = u; u = v; v = w; }
    int pos[3];
    pos[u] = (int)(t % q.ext[u]); pos[v] = (int)(t / q.ext[u]); pos[q.a] = q.t1;
    cell = ((long long)pos[2] * q.ext[1] + pos[1]) * q.ext[0] + pos[0];
    pos[q.a] -= 1;
    cellm = q.interpolate ? ((long long)pos[2] * q.ext[1] + pos[1]) * q.ext[0] + pos[0] : cell;
    return true;
}

__global__ void __launch_bounds__(256) k_flux(FluxGeom q, const float2 *__restrict__ P, float *__restrict__ out, ReduceScratch rs)
{
    double acc = 0.0;
    const long long plane_cells = q.bc / q.ext[q.a];
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < plane_cells; t += (long long)gridDim.x * blockDim.x) {
        long long cell, cellm;
        flux_cell(q, t, cell, cellm);
#pragma unroll
        for (int pr = 0; pr < 2; ++pr) {          // pair 0: E_b with H_c (+), pair 1: E_c with H_b (-)
            const int sE = pr ? q.sEc : q.sEb, sH = pr ? q.sHb : q.sHc;
            const float2 E = __ldg(P + (long long)sE * q.bc + cell);
            const float2 H1 = __ldg(P + (long long)sH * q.bc + cell), H0 = __ldg(P + (long long)sH * q.bc + cellm);
            const float hr = q.interpolate ? 0.5f * (H0.x + H1.x) : H1.x, hi = q.interpolate ? 0.5f * (H0.y + H1.y) : H1.y;
            const float tr = hr * q.cw + hi * q.sw, ti = hi * q.cw - hr * q.sw;       // H~ = exp(-i w/2) Hbar
            const float s = 0.5f * (E.x * tr + E.y * ti);
            acc += pr ? -(double)s : (double)s;
        }
    }
    block_sum_to(acc, rs, out);
}

// dL_dphasor of frequency f (zero-filled by the caller): every entry is written by exactly one thread
__global__ void k_flux_vjp(FluxGeom q, const float2 *__restrict__ P, const float *__restrict__ dL_dflux, float2 *__restrict__ dP)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long cell, cellm;
    if (!flux_cell(q, t, cell, cellm)) return;
    const float Gf = __ldg(dL_dflux);
#pragma unroll
    for (int pr = 0; pr < 2; ++pr) {
        const int sE = pr ? q.sEc : q.sEb, sH = pr ? q.sHb : q.sHc;
        const float G = (pr ? -0.5f : 0.5f) * Gf;
        const float2 E = __ldg(P + (long long)sE * q.bc + cell);
        const float2 H1 = __ldg(P + (long long)sH * q.bc + cell), H0 = __ldg(P + (long long)sH * q.bc + cellm);
        const float hr = q.interpolate ? 0.5f * (H0.x + H1.x) : H1.x, hi = q.interpolate ? 0.5f * (H0.y + H1.y) : H1.y;
        const float tr = hr * q.cw + hi * q.sw, ti = hi * q.cw - hr * q.sw;
        dP[(long long)sE * q.bc + cell] = make_float2(G * tr, G * ti);
        const float dtr = G * E.x, dti = G * E.y;
        const float dhr = dtr * q.cw - dti * q.sw, dhi = dtr * q.sw + dti * q.cw;
        if (q.interpolate) {
            dP[(long long)sH * q.bc + cell] = make_float2(0.5f * dhr, 0.5f * dhi);
            dP[(long long)sH * q.bc + cellm] = make_float2(0.5f * dhr, 0.5f * dhi);
        } else {
            dP[(long long)sH * q.bc + cell] = make_float2(dhr, dhi);
        }
    }
}

bool flux_geom(const DetectorDev &dt, int axis, int interpolate, float cw, float sw, FluxGeom &q)
{
    const int a = axis, b = (a + 1) % 3, c = (a + 2) % 3;
    const int need = (1 << b) | (1 << c) | (1 << (3 + b)) | (1 << (3 + c));
    if ((dt.mask & need) != need) return false;
    for (int x = 0; x < 3; ++x) q.ext[x] = dt.hi[x] - dt.lo[x];
    if (q.ext[a] != (interpolate ? 2 : 1)) return false;
    auto slot = [&](int comp) { int ci = 0; for (int x = 0; x < comp; ++x) ci += (dt.mask >> x) & 1; return ci; };
    q.a = a; q.t1 = q.ext[a] - 1;
    q.sEb = slot(b); q.sEc = slot(c); q.sHb = slot(3 + b); q.sHc = slot(3 + c);
    q.ncomp = dt.ncomp;
    q.bc = (long long)q.ext[0] * q.ext[1] * q.ext[2];
    q.interpolate = interpolate; q.cw = interpolate ? cw : 1.f; q.sw = interpolate ? sw : 0.f;
    return true;
}

// ------------------------------------------------------------------------------------------ TFSF auxiliary grid (R25)
// 1-D leapfrog of the plane wave restricted to its axis, one CTA, both arrays in shared memory:
//   e[m] += sgn S ie (h[m] - h[m-1]);  h[m] += sgn S im (e[m+1] - e[m]);  hard source e[0] = base[n]
//   wE[n] = -sgn S ie h[m0-1] (before the e update),  wH[n] = -dir sgn S im e[m0] (after it),  m0 = 2.
// Only nodes the pulse can have reached (m <= n + 2) are touched.
__global__ void __launch_bounds__(1024) k_tfsf_aux(float S, float ie, float im, float sgn, float dir_sign, int n_steps, int L,
                                                   const float *__restrict__ base, float *__restrict__ wE, float *__restrict__ wH)
{
    extern __shared__ float sm[];
    float *e = sm, *h = sm + (L + 1);
    for (int m = threadIdx.x; m <= L; m += blockDim.x) { e[m] = 0.f; h[m] = 0.f; }
    __syncthreads();
    const int m0 = 2;
    const float ce = sgn * S * ie, ch = sgn * S * im;
    for (int n = 0; n < n_steps; ++n) {
        const int reach = min(L - 1, n + 3);
        if (threadIdx.x == 0) wE[n] = -ce * h[m0 - 1];
        for (int m = 1 + threadIdx.x; m <= reach; m += blockDim.x) e[m] += ce * (h[m] - h[m - 1]);
        if (threadIdx.x == 0) e[0] = __ldg(base + n);
        __syncthreads();
        if (threadIdx.x == 0) wH[n] = -dir_sign * ch * e[m0];
        for (int m = threadIdx.x; m <= min(L - 2, reach); m += blockDim.x) h[m] += ch * (e[m + 1] - e[m]);
        __syncthreads();
    }
}

unsigned blocks_for(long long n) { return (unsigned)std::max<long long>(1, std::min<long long>((n + 255) / 256, RED_BLOCKS)); }

}  // namespace

void launch_time_detect(const Dims &G, const float *volA, const float *volB, int par_off, const float *ie, const float *im,
                        const TimeDetDev &td, const ReduceScratch &rs, const int *step, cudaStream_t st)
{
    const long long n = (long long)(td.hi[0] - td.lo[0]) * (td.hi[1] - td.lo[1]) * (td.hi[2] - td.lo[2]);
    if (td.kind == 0)
        k_snapshot<false><<<blocks_for(n), 256, 0, st>>>(G, const_cast<float *>(volA), const_cast<float *>(volB), par_off, td, step, nullptr);
    else
        k_energy<<<blocks_for(n), 256, 0, st>>>(G, volA, volB, par_off, ie, im, td, rs, step);
}

void launch_time_detect_adjoint(const Dims &G, float *lamA, float *lamB, const float *fA, const float *fB, int par_off,
                                const float *ie, const float *im, bool scaled_H, const TimeDetDev &td, float *g,
                                const int *step, cudaStream_t st)
{
    const long long n = (long long)(td.hi[0] - td.lo[0]) * (td.hi[1] - td.lo[1]) * (td.hi[2] - td.lo[2]);
    if (td.kind == 0)
        k_snapshot<true><<<blocks_for(n), 256, 0, st>>>(G, lamA, lamB, par_off, td, step, scaled_H ? im : nullptr);
    else
        k_energy_adjoint<<<blocks_for(n), 256, 0, st>>>(G, lamA, lamB, fA, fB, par_off, ie, im, scaled_H ? 1 : 0, td, g, step);
}

void launch_flux(const DetectorDev &dt, const float *phasor, int axis, int interpolate, int f, float cw, float sw,
                 float *flux, const ReduceScratch &rs, cudaStream_t st)
{
    FluxGeom q;
    if (!flux_geom(dt, axis, interpolate, cw, sw, q)) return;
    const float2 *P = reinterpret_cast<const float2 *>(phasor) + (long long)f * q.ncomp * q.bc;
    k_flux<<<blocks_for(q.bc / q.ext[q.a]), 256, 0, st>>>(q, P, flux + f, rs);
}

void launch_flux_vjp(const DetectorDev &dt, const float *phasor, int axis, int interpolate, int f, float cw, float sw,
                     const float *dL_dflux, float *dL_dphasor, cudaStream_t st)
{
    FluxGeom q;
    if (!flux_geom(dt, axis, interpolate, cw, sw, q)) return;
    const long long off = (long long)f * q.ncomp * q.bc;
    const long long cells = q.bc / q.ext[q.a];
    k_flux_vjp<<<(unsigned)((cells + 255) / 256), 256, 0, st>>>(q, reinterpret_cast<const float2 *>(phasor) + off, dL_dflux + f,
                                                                 reinterpret_cast<float2 *>(dL_dphasor) + off);
}

cudaError_t launch_tfsf_aux(float S, float ie, float im, float sgn, float dir_sign, int n_steps, const float *base,
                            float *wE, float *wH, cudaStream_t st)
{
    const int L = 2 + n_steps / 2 + 16;          // the far wall is out of causal reach of the interface node
    const size_t smem = 2 * (size_t)(L + 1) * sizeof(float);
    if (smem > 200 * 1024) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(k_tfsf_aux, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_tfsf_aux<<<1, 1024, smem, st>>>(S, ie, im, sgn, dir_sign, n_steps, L, base, wE, wH);
    return cudaGetLastError();
}

}  // namespace fdtd
