// kernels_generic.cu -- one-thread-per-cell kernels for every row of the hot path.
//
// These are the general path: any grid size, periodic or zero-padded walls, in-place updates.
// They serve periodic grids and sizes the fused TMA kernels do not take, and they are the
// simple statement the fused kernels are cross-checked against on the GPU.
// Formulas: include/fdtd.h (conventions) and DESIGN.md section 2; Eq. 1-2, L72, L84.
#include <algorithm>
#include <cuda_fp16.h>
#include "fdtd_internal.h"

namespace fdtd {

namespace {

constexpr int BX = 64, BY = 4;

__device__ __forceinline__ long long lin(const Dims &G, int i, int j, int k)
{
    return ((long long)k * G.ny + j) * G.nx + i;
}

// neighbour fetch with wrap (periodic) or zero (walls); offsets are at most +-1
template <bool PER>
__device__ __forceinline__ float fetch(const Dims &G, const float *__restrict__ F, int i, int j, int k)
{
    if (PER) {
        i = i < 0 ? i + G.nx : (i >= G.nx ? i - G.nx : i);
        j = j < 0 ? j + G.ny : (j >= G.ny ? j - G.ny : j);
        k = k < 0 ? k + G.nz : (k >= G.nz ? k - G.nz : k);
    } else if (i < 0 || i >= G.nx || j < 0 || j >= G.ny || k < 0 || k >= G.nz) {
        return 0.f;
    }
    return __ldg(F + lin(G, i, j, k));
}

#define CELL_IJK()                                                   \
    const int i = blockIdx.x * BX + threadIdx.x;                     \
    const int j = blockIdx.y * BY + threadIdx.y;                     \
    const int k = blockIdx.z;                                        \
    if (i >= G.nx || j >= G.ny) return;                              \
    const long long p = lin(G, i, j, k);                             \
    const int pos[3] = { i, j, k };                                  \
    (void)pos;

// ------------------------------------------------------------------------------------------ F1+F2
// N4 (reading R29): with a conductivity volume the update is E' = Ca E + Cb S ie bracket, beta = sigma S ie / 2,
// Ca = (1 - beta)/(1 + beta), Cb = 1/(1 + beta)
template <bool PER>
__global__ void __launch_bounds__(BX *BY) k_update_E(Dims G, Tables T, float *__restrict__ f,
                                                     const float *__restrict__ ie, PsiSet psi, const float *__restrict__ sigma)
{
    CELL_IJK();
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        const float e = __ldg(ie + (G.aniso ? c * G.nc : 0) + p);            // reading R30: one volume per component when aniso
        const float beta = sigma ? 0.5f * __ldg(sigma + p) * G.S * e : 0.f;
        const float Ca = (1.f - beta) / (1.f + beta), Cb = 1.f / (1.f + beta);
        const float sie = (sigma ? Cb : 1.f) * G.S * e;
        const float *Hb = f + (3 + b) * G.nc, *Ha = f + (3 + a) * G.nc;
        const float d1 = Hb[p] - fetch<PER>(G, Hb, i - (a == 0), j - (a == 1), k - (a == 2));
        const float d2 = Ha[p] - fetch<PER>(G, Ha, i - (b == 0), j - (b == 1), k - (b == 2));
        float t = __ldg(T.ik[0][a] + pos[a]) * d1 - __ldg(T.ik[0][b] + pos[b]) * d2;
        if (G.d > 0) {
            const long long s0 = psi_index(G, a, i, j, k);
            if (s0 >= 0) {
                const float ps = __ldg(T.b[0][a] + pos[a]) * psi.p[c][0][s0] + __ldg(T.a[0][a] + pos[a]) * d1;
                psi.p[c][0][s0] = ps;
                t += ps;
            }
            const long long s1 = psi_index(G, b, i, j, k);
            if (s1 >= 0) {
                const float ps = __ldg(T.b[0][b] + pos[b]) * psi.p[c][1][s1] + __ldg(T.a[0][b] + pos[b]) * d2;
                psi.p[c][1][s1] = ps;
                t -= ps;
            }
        }
        if (sigma) f[c * G.nc + p] = fmaf(Ca, f[c * G.nc + p], sie * t);
        else f[c * G.nc + p] += sie * t;
    }
}

// ------------------------------------------------------------------------------------------ F4+F5
template <bool PER>
__global__ void __launch_bounds__(BX *BY) k_update_H(Dims G, Tables T, float *__restrict__ f,
                                                     const float *__restrict__ im, PsiSet psi)
{
    CELL_IJK();
    const float sim = G.S * (im ? __ldg(im + p) : 1.f);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        const float *Eb = f + b * G.nc, *Ea = f + a * G.nc;
        const float d1 = fetch<PER>(G, Eb, i + (a == 0), j + (a == 1), k + (a == 2)) - Eb[p];
        const float d2 = fetch<PER>(G, Ea, i + (b == 0), j + (b == 1), k + (b == 2)) - Ea[p];
        float t = __ldg(T.ik[1][a] + pos[a]) * d1 - __ldg(T.ik[1][b] + pos[b]) * d2;
        if (G.d > 0) {
            const long long s0 = psi_index(G, a, i, j, k);
            if (s0 >= 0) {
                const float ps = __ldg(T.b[1][a] + pos[a]) * psi.p[c][0][s0] + __ldg(T.a[1][a] + pos[a]) * d1;
                psi.p[c][0][s0] = ps;
                t += ps;
            }
            const long long s1 = psi_index(G, b, i, j, k);
            if (s1 >= 0) {
                const float ps = __ldg(T.b[1][b] + pos[b]) * psi.p[c][1][s1] + __ldg(T.a[1][b] + pos[b]) * d2;
                psi.p[c][1][s1] = ps;
                t -= ps;
            }
        }
        f[(3 + c) * G.nc + p] -= sim * t;
    }
}

// ------------------------------------------------------------------------------------------ F3/F6
__global__ void k_add_source(Dims G, float *__restrict__ f, SourceDev s, const int *__restrict__ step, float sign)
{
    const int bx = s.hi[0] - s.lo[0], by = s.hi[1] - s.lo[1], bz = s.hi[2] - s.lo[2];
    const long long n_cells = (long long)bx * by * bz;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_cells) return;
    const int i = (int)(t % bx), j = (int)((t / bx) % by), k = (int)(t / ((long long)bx * by));
    const float w = sign * __ldg(s.waveform + *step);
    const float pr = s.profile ? __ldg(s.profile + t) : 1.f;
    f[s.comp * G.nc + lin(G, s.lo[0] + i, s.lo[1] + j, s.lo[2] + k)] += pr * w;
}

// ------------------------------------------------------------------------------------------ F7 / B1
// cs_table: [max_steps][total_freq][2] = (cos, sin) of omega_f*(n+1), built on the host in fp64 (R13)
template <bool ADJ>
__global__ void k_detector(Dims G, float *__restrict__ f, DetectorDev dt, const float *__restrict__ cs,
                           int total_freq, const int *__restrict__ step, float *__restrict__ f2, int par_off,
                           const float *__restrict__ med_H)
{
    if (f2 && ((*step + par_off) & 1)) f = f2;       // ping-pong volumes of the fused path
    const int bx = dt.hi[0] - dt.lo[0], by = dt.hi[1] - dt.lo[1], bz = dt.hi[2] - dt.lo[2];
    const long long bc = (long long)bx * by * bz;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= bc) return;
    const int i = (int)(t % bx), j = (int)((t / bx) % by), k = (int)(t / ((long long)bx * by));
    const long long p = lin(G, dt.lo[0] + i, dt.lo[1] + j, dt.lo[2] + k);
    const float *csn = cs + ((long long)(*step) * total_freq + dt.cs_off) * 2;
    int ci = 0;
    for (int c = 0; c < 6; ++c) {
        if (!((dt.mask >> c) & 1)) continue;
        if (!ADJ) {
            const float v = f[c * G.nc + p];
            for (int q = 0; q < dt.n_freq; ++q) {
                float2 *P = reinterpret_cast<float2 *>(dt.phasor) + ((long long)q * dt.ncomp + ci) * bc + t;
                float2 acc = *P;
                acc.x += v * __ldg(csn + 2 * q);
                acc.y -= v * __ldg(csn + 2 * q + 1);
                *P = acc;
            }
        } else {
            float acc = 0.f;
            for (int q = 0; q < dt.n_freq; ++q) {
                const float2 Gq = __ldg(reinterpret_cast<const float2 *>(dt.phasor) + ((long long)q * dt.ncomp + ci) * bc + t);
                acc += Gq.x * __ldg(csn + 2 * q) - Gq.y * __ldg(csn + 2 * q + 1);
            }
            if (med_H && c >= 3) acc *= __ldg(med_H + p);
            f[c * G.nc + p] += acc;
        }
        ++ci;
    }
}

// N4, lossy E update: lamE_c *= Ca after the adjoint of the E update
__global__ void k_lossy_scale_E(Dims G, float *__restrict__ lam, const float *__restrict__ ie, const float *__restrict__ sigma)
{
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < G.nc; p += (long long)gridDim.x * blockDim.x) {
        for (int c = 0; c < 3; ++c) {
            const float beta = 0.5f * __ldg(sigma + p) * G.S * __ldg(ie + (G.aniso ? c * G.nc : 0) + p);
            lam[c * G.nc + p] *= (1.f - beta) / (1.f + beta);
        }
    }
}

// lamH <-> im lamH on the three H volumes (fused reverse sweep with inv_mu)
__global__ void k_scale_H(float *__restrict__ lamH, const float *__restrict__ im, long long nc, bool inverse)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < 3 * nc; t += (long long)gridDim.x * blockDim.x) {
        const float m = __ldg(im + t % nc);
        lamH[t] = inverse ? lamH[t] / m : lamH[t] * m;
    }
}

// ------------------------------------------------------------------------------------------ F8
// One thread per float of a step's record.  INJECT=false: fields -> rec[n]; true: rec[n] -> fields.
// recorder element idx: fp32, or fp16 when the grid was created with FDTD_FLAG_RECORDER_FP16
__device__ __forceinline__ void rec_store(float *rec, long long idx, float v, int half)
{
    if (half) reinterpret_cast<__half *>(rec)[idx] = __float2half_rn(v); else rec[idx] = v;
}
__device__ __forceinline__ float rec_load(const float *rec, long long idx, int half)
{
    return half ? __half2float(reinterpret_cast<const __half *>(rec)[idx]) : __ldg(rec + idx);
}

// PP=true (fused ping-pong path): fH/fE are the two field buffers A/B; step n read buffer n&1 (pre-step H)
// and wrote buffer (n+1)&1 (E'); for INJECT the target is buffer (n+1)&1 (the state the reverse step reads).
template <bool INJECT, bool PP>
__global__ void k_record(Dims G, RecLayout R, const float *__restrict__ fH, const float *__restrict__ fE,
                         float *__restrict__ fout, float *__restrict__ rec, const int *__restrict__ step)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= R.stride) return;
    if (PP) {
        const float *A = fH, *B = fE;
        const int par = (*step) & 1;
        fH = par ? B : A;
        fE = par ? A : B;
        fout = const_cast<float *>(fE);
    }
    // locate the segment
    int a = 0, side = 0, which = 0;
    long long local = -1;
#pragma unroll
    for (int aa = 0; aa < 3; ++aa)
#pragma unroll
        for (int ss = 0; ss < 2; ++ss)
#pragma unroll
            for (int ww = 0; ww < 2; ++ww) {
                const long long o = R.off[aa][ss][ww];
                if (t >= o && t < o + R.cells[aa]) { a = aa; side = ss; which = ww; local = t - o; }
            }
    if (local < 0) return;   // padding
    const int fa = R.fast[a], sl = R.slow[a];
    const int nf = G.hi[fa] - G.lo[fa];
    int pos[3];
    pos[a] = side ? G.hi[a] : G.lo[a] - 1;
    pos[fa] = G.lo[fa] + (int)(local % nf);
    pos[sl] = G.lo[sl] + (int)(local / nf);
    const int comp = (a + 1 + which) % 3;
    const long long p = lin(G, pos[0], pos[1], pos[2]);
    const long long r = (long long)(*step) * R.stride + t;
    if (!INJECT) {
        rec_store(rec, r, side ? __ldg(fE + comp * G.nc + p) : __ldg(fH + (3 + comp) * G.nc + p), R.half);
    } else {
        fout[(side ? comp : 3 + comp) * G.nc + p] = rec_load(rec, r, R.half);
    }
}

// Pipelined recorder of the fused path: runs beside forward step n and reads the buffer that step reads
// (n&1): pre-step H at lo-1 -> rec[n] (n < n_steps), E' at hi, written by step n-1, -> rec[n-1] (n >= 1).
// 128 threads x <= 32 registers and no shared memory, so a block fits beside a resident k_step CTA and shares its issue
// slots: the kernel is kept short in instructions (grid.y = the record's segment, 32-bit index arithmetic, PIPE_U elements
// per thread with their loads in flight together).
#ifndef FDTD_PIPE_U
#define FDTD_PIPE_U 2
#endif
constexpr int PIPE_U = FDTD_PIPE_U;

struct PipeSeg {               // segment blockIdx.y of a step's record
    long long base;            // volume offset (component included) of the segment's first face cell
    long long off;             // offset of the segment inside a step's record
    unsigned cells, nf;        // face cells; extent of the fast in-face axis
    long long sf, ss;          // volume strides of the fast / slow in-face axis
    int side;                  // 0: low face (H at lo-1), 1: high face (E' at hi)
};
struct PipeTable { PipeSeg s[12]; long long stride; int half; };

__global__ void __launch_bounds__(128, 16) k_record_pipe(const __grid_constant__ PipeTable T, const float *__restrict__ A,
                                                         const float *__restrict__ B, float *__restrict__ rec,
                                                         const int *__restrict__ step, int n_steps)
{
    const int n = *step;
    const PipeSeg &q = T.s[blockIdx.y];
    if (q.side ? n < 1 : n >= n_steps) return;
    const float *f = ((n & 1) ? B : A) + q.base;
    const unsigned l0 = blockIdx.x * (128u * PIPE_U) + threadIdx.x;
    float v[PIPE_U];
#pragma unroll
    for (int u = 0; u < PIPE_U; ++u) {
        const unsigned l = l0 + u * 128u;
        v[u] = l < q.cells ? __ldg(f + (l % q.nf) * q.sf + (l / q.nf) * q.ss) : 0.f;
    }
    const long long r0 = (long long)(q.side ? n - 1 : n) * T.stride + q.off;
#pragma unroll
    for (int u = 0; u < PIPE_U; ++u) {
        const unsigned l = l0 + u * 128u;
        if (l < q.cells) rec_store(rec, r0 + l, v[u], T.half);
    }
}

// Face injection of the fused reverse sweep, run beside adjoint step n: rec[n] -> buffer (n+1)&1, the volume
// the inverse step n reads (pre-step H at lo-1, E' at hi).  Sized like k_record_pipe to fit beside a k_step CTA.
__global__ void __launch_bounds__(128, 16) k_inject_pipe(const __grid_constant__ PipeTable T, float *__restrict__ A, float *__restrict__ B,
                                                         const float *__restrict__ rec, const int *__restrict__ step)
{
    const int n = *step;
    const PipeSeg &q = T.s[blockIdx.y];
    float *f = ((n & 1) ? A : B) + q.base;
    const unsigned l0 = blockIdx.x * (128u * PIPE_U) + threadIdx.x;
    const long long r0 = (long long)n * T.stride + q.off;
    float v[PIPE_U];
#pragma unroll
    for (int u = 0; u < PIPE_U; ++u) {
        const unsigned l = l0 + u * 128u;
        v[u] = l < q.cells ? rec_load(rec, r0 + l, T.half) : 0.f;
    }
#pragma unroll
    for (int u = 0; u < PIPE_U; ++u) {
        const unsigned l = l0 + u * 128u;
        if (l < q.cells) f[(l % q.nf) * q.sf + (l / q.nf) * q.ss] = v[u];
    }
}

__global__ void k_advance(int *step, int delta) { *step += delta; }
// the step counter lives in two slots that alternate between steps: nobody reads `out` during the step that writes it
__global__ void k_next_step(const int *in, int *out, int delta) { *out = *in + delta; }
__global__ void k_set_step(int *p, int v) { *p = v; }

// ------------------------------------------------------------------------------------------ B2 / B5
// Adjoint of the H update (FAMILY=1: reads lamH, updates lamE, psi_H cotangents) or of the E update
// (FAMILY=0: reads lamE, updates lamH, psi_E cotangents), in gather form:
//   w_c(q)  = sgn*S*med(q)*lam_c(q)          sgn = -1 (H update), +1 (E update)
//   g1_c(q) =  ik_a w + a_a (lpsi_c0 + w)    a = c+1 (tables of FAMILY at q_a)
//   g2_c(q) = -ik_b w + a_b (lpsi_c1 - w)    b = c+2
//   lpsi_c0 <- b_a (lpsi_c0 + w) ; lpsi_c1 <- b_b (lpsi_c1 - w)          (owner cell only)
//   FAMILY=1: lamE_t(p) -= [g1_{t+1}(p) - g1_{t+1}(p-e_{t+2})] + [g2_{t+2}(p) - g2_{t+2}(p-e_{t+1})]
//   FAMILY=0: lamH_t(p) -= [g1_{t+1}(p+e_{t+2}) - g1_{t+1}(p)] + [g2_{t+2}(p+e_{t+1}) - g2_{t+2}(p)]
// psi cotangents are ping-ponged (read set[n&1], write set[(n&1)^1]) because the neighbour's g is
// recomputed from its OLD psi cotangent.
template <int FAMILY>
struct AdjCtx {
    const Dims &G;
    const Tables &T;
    const float *lam_src;    // 3 volumes (lamH for FAMILY 1, lamE for FAMILY 0)
    const float *med;        // inv_mu (may be NULL) or inv_eps
    const PsiSet &lin_;      // old psi cotangents
    const float *sigma;      // FAMILY 0 only, lossy E update (N4): the bracket's cotangent is Cb S ie lamE'
    __device__ __forceinline__ float w(int c, long long q) const
    {
        const float m = med ? __ldg(med + ((!FAMILY && G.aniso) ? c * G.nc : 0) + q) : 1.f;
        float r = (FAMILY ? -G.S : G.S) * m * __ldg(lam_src + c * G.nc + q);
        if (!FAMILY && sigma) r /= 1.f + 0.5f * __ldg(sigma + q) * G.S * m;
        return r;
    }
    // g1 of component c at cell (i,j,k) (in range)
    __device__ __forceinline__ float g(int c, int s, int i, int j, int k, float *new_psi) const
    {
        const int ax = psi_axis(c, s);
        const int pa = ax == 0 ? i : (ax == 1 ? j : k);
        const long long q = lin(G, i, j, k);
        const float ww = w(c, q);
        const float sg = s ? -1.f : 1.f;
        float r = sg * __ldg(T.ik[FAMILY][ax] + pa) * ww;
        if (G.d > 0) {
            const long long si = psi_index(G, ax, i, j, k);
            if (si >= 0) {
                const float l = __ldg(lin_.p[c][s] + si) + sg * ww;
                r += __ldg(T.a[FAMILY][ax] + pa) * l;
                if (new_psi) *new_psi = __ldg(T.b[FAMILY][ax] + pa) * l;
            }
        }
        return r;
    }
};

template <int FAMILY, bool PER>
__global__ void __launch_bounds__(BX *BY) k_adjoint(Dims G, Tables T, float *__restrict__ lam,
                                                    const float *__restrict__ med, PsiSet set0, PsiSet set1,
                                                    const int *__restrict__ step, const float *__restrict__ sigma)
{
    CELL_IJK();
    const int par = (*step) & 1;
    const PsiSet &pin = par ? set1 : set0;
    const PsiSet &pout = par ? set0 : set1;
    const float *src = lam + (FAMILY ? 3 : 0) * G.nc;
    float *dst = lam + (FAMILY ? 0 : 3) * G.nc;
    AdjCtx<FAMILY> C{ G, T, src, med, pin, sigma };
    const int sgn = FAMILY ? -1 : +1;     // neighbour offset: p - e (H-update adjoint), p + e (E-update adjoint)
    // own-cell g values and psi-cotangent updates
    float g_own[3][2];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            float np_ = 0.f;
            bool has = false;
            if (G.d > 0) {
                const long long si = psi_index(G, psi_axis(c, s), i, j, k);
                has = si >= 0;
                g_own[c][s] = C.g(c, s, i, j, k, has ? &np_ : nullptr);
                if (has) pout.p[c][s][si] = np_;
            } else {
                g_own[c][s] = C.g(c, s, i, j, k, nullptr);
            }
        }
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        const int c1 = (t + 1) % 3, ax1 = (t + 2) % 3;   // g1 of component t+1, derivative axis t+2
        const int c2 = (t + 2) % 3, ax2 = (t + 1) % 3;   // g2 of component t+2, derivative axis t+1
        int q1[3] = { i, j, k }, q2[3] = { i, j, k };
        q1[ax1] += sgn;
        q2[ax2] += sgn;
        float n1 = 0.f, n2 = 0.f;
        {
            int qi = q1[0], qj = q1[1], qk = q1[2];
            bool ok = true;
            if (PER) {
                qi = qi < 0 ? qi + G.nx : (qi >= G.nx ? qi - G.nx : qi);
                qj = qj < 0 ? qj + G.ny : (qj >= G.ny ? qj - G.ny : qj);
                qk = qk < 0 ? qk + G.nz : (qk >= G.nz ? qk - G.nz : qk);
            } else {
                ok = qi >= 0 && qi < G.nx && qj >= 0 && qj < G.ny && qk >= 0 && qk < G.nz;
            }
            if (ok) n1 = C.g(c1, 0, qi, qj, qk, nullptr);
        }
        {
            int qi = q2[0], qj = q2[1], qk = q2[2];
            bool ok = true;
            if (PER) {
                qi = qi < 0 ? qi + G.nx : (qi >= G.nx ? qi - G.nx : qi);
                qj = qj < 0 ? qj + G.ny : (qj >= G.ny ? qj - G.ny : qj);
                qk = qk < 0 ? qk + G.nz : (qk >= G.nz ? qk - G.nz : qk);
            } else {
                ok = qi >= 0 && qi < G.nx && qj >= 0 && qj < G.ny && qk >= 0 && qk < G.nz;
            }
            if (ok) n2 = C.g(c2, 1, qi, qj, qk, nullptr);
        }
        // FAMILY=1: -(own - nbr) ; FAMILY=0: -(nbr - own)
        const float diff1 = FAMILY ? (g_own[c1][0] - n1) : (n1 - g_own[c1][0]);
        const float diff2 = FAMILY ? (g_own[c2][1] - n2) : (n2 - g_own[c2][1]);
        dst[t * G.nc + p] -= diff1 + diff2;
    }
}

// ------------------------------------------------------------------------------------------ B3
// inverse H step on I:  H = H' + S im curl+ E'   (sources already subtracted; the E' operand at
// index N_a-d was injected from the record)
// N4 (dL/d inv_mu): with lam and g_mu, g_mu -= S sum_c lamH'_c (curl+ E')_c, lamH' = the cotangent of the post-step H:
// the H part of `lam`, or of lam2 when the fused sweep's volume (n+1)&1 is the odd one; scaled: that part holds im lamH'.
template <bool PER>
__global__ void __launch_bounds__(BX *BY) k_inv_H(Dims G, float *__restrict__ f, const float *__restrict__ im,
                                                  const float *__restrict__ lam, const float *__restrict__ lam2,
                                                  const int *__restrict__ step, int scaled, float *__restrict__ g_mu)
{
    CELL_IJK();
    if (i < G.lo[0] || i >= G.hi[0] || j < G.lo[1] || j >= G.hi[1] || k < G.lo[2] || k >= G.hi[2]) return;
    const float m = im ? __ldg(im + p) : 1.f;
    const float sim = G.S * m;
    if (lam2 && ((*step + 1) & 1)) lam = lam2;
    float acc = 0.f;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        const float *Eb = f + b * G.nc, *Ea = f + a * G.nc;
        const float d1 = fetch<PER>(G, Eb, i + (a == 0), j + (a == 1), k + (a == 2)) - Eb[p];
        const float d2 = fetch<PER>(G, Ea, i + (b == 0), j + (b == 1), k + (b == 2)) - Ea[p];
        f[(3 + c) * G.nc + p] += sim * (d1 - d2);
        if (g_mu) acc = fmaf(lam[(3 + c) * G.nc + p], d1 - d2, acc);
    }
    if (g_mu) g_mu[p] -= G.S * (scaled ? acc / m : acc);
}

// ------------------------------------------------------------------------------------------ B4
// q = curl- H on I (operand at d-1 injected from the record); g += S sum_c lamE_c q_c on the
// gradient box; E = E' - S ie q.
template <bool PER>
__global__ void __launch_bounds__(BX *BY) k_inv_E_grad(Dims G, float *__restrict__ f, const float *__restrict__ ie,
                                                       const float *__restrict__ lam, float *__restrict__ g,
                                                       const float *__restrict__ lam2, const int *__restrict__ step)
{
    CELL_IJK();
    if (lam2 && ((*step) & 1)) lam = lam2;           // ping-pong cotangents of the fused path: lamE' of step n is in buffer n&1
    if (i < G.lo[0] || i >= G.hi[0] || j < G.lo[1] || j >= G.hi[1] || k < G.lo[2] || k >= G.hi[2]) return;
    const bool ing = i >= G.glo[0] && i < G.ghi[0] && j >= G.glo[1] && j < G.ghi[1] && k >= G.glo[2] && k < G.ghi[2];
    float acc = 0.f;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        const float *Hb = f + (3 + b) * G.nc, *Ha = f + (3 + a) * G.nc;
        const float d1 = Hb[p] - fetch<PER>(G, Hb, i - (a == 0), j - (a == 1), k - (a == 2));
        const float d2 = Ha[p] - fetch<PER>(G, Ha, i - (b == 0), j - (b == 1), k - (b == 2));
        const float q = d1 - d2;
        const float lq = __ldg(lam + c * G.nc + p) * q;
        acc += lq;
        if (G.aniso && ing) g[c * G.nc + p] += G.S * lq;                   // reading R30: one gradient volume per component
        f[c * G.nc + p] -= G.S * __ldg(ie + (G.aniso ? c * G.nc : 0) + p) * q;
    }
    if (!G.aniso && ing) g[p] += G.S * acc;
}

// ------------------------------------------------------------------------------------------ B6
__global__ void k_grad_rho(Dims G, const float *__restrict__ g, const float *__restrict__ ie, float delta_eps,
                           int lx, int ly, int lz, int bx, int by, int bz, float *__restrict__ out)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)bx * by * bz) return;
    const int i = (int)(t % bx), j = (int)((t / bx) % by), k = (int)(t / ((long long)bx * by));
    const long long p = lin(G, lx + i, ly + j, lz + k);
    const float v = __ldg(ie + p);
    out[t] = -__ldg(g + p) * delta_eps * v * v;
}

inline dim3 vol_grid(const Dims &G) { return dim3((G.nx + BX - 1) / BX, (G.ny + BY - 1) / BY, G.nz); }
inline dim3 vol_block() { return dim3(BX, BY, 1); }

}  // namespace

void launch_update_E(const Dims &G, const Tables &T, float *fields, const float *ie, PsiSet psiE, cudaStream_t st, const float *sigma)
{
    if (G.periodic) k_update_E<true><<<vol_grid(G), vol_block(), 0, st>>>(G, T, fields, ie, psiE, sigma);
    else            k_update_E<false><<<vol_grid(G), vol_block(), 0, st>>>(G, T, fields, ie, psiE, sigma);
}

void launch_update_H(const Dims &G, const Tables &T, float *fields, const float *im, PsiSet psiH, cudaStream_t st)
{
    if (G.periodic) k_update_H<true><<<vol_grid(G), vol_block(), 0, st>>>(G, T, fields, im, psiH);
    else            k_update_H<false><<<vol_grid(G), vol_block(), 0, st>>>(G, T, fields, im, psiH);
}

void launch_add_source(const Dims &G, float *fields, const SourceDev &s, const int *step, float sign, cudaStream_t st)
{
    const long long n = (long long)(s.hi[0] - s.lo[0]) * (s.hi[1] - s.lo[1]) * (s.hi[2] - s.lo[2]);
    k_add_source<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(G, fields, s, step, sign);
}

void launch_detector(const Dims &G, const float *fields, const DetectorDev &dt, const float *cs_table,
                     int total_freq, const int *step, cudaStream_t st)
{
    const long long n = (long long)(dt.hi[0] - dt.lo[0]) * (dt.hi[1] - dt.lo[1]) * (dt.hi[2] - dt.lo[2]);
    k_detector<false><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(G, const_cast<float *>(fields), dt, cs_table, total_freq, step, nullptr, 0, nullptr);
}

void launch_detector_adjoint(const Dims &G, float *lam, const DetectorDev &dt, const float *cs_table,
                             int total_freq, const int *step, cudaStream_t st)
{
    const long long n = (long long)(dt.hi[0] - dt.lo[0]) * (dt.hi[1] - dt.lo[1]) * (dt.hi[2] - dt.lo[2]);
    k_detector<true><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(G, lam, dt, cs_table, total_freq, step, nullptr, 0, nullptr);
}

// reverse step n of the fused path injects into the volume it is about to read: buffer (n+1)&1
void launch_detector_adjoint_pp(const Dims &G, float *lamA, float *lamB, const DetectorDev &dt, const float *cs_table,
                                int total_freq, const int *step, const float *im, cudaStream_t st)
{
    const long long n = (long long)(dt.hi[0] - dt.lo[0]) * (dt.hi[1] - dt.lo[1]) * (dt.hi[2] - dt.lo[2]);
    k_detector<true><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(G, lamA, dt, cs_table, total_freq, step, lamB, 1, im);
}

void launch_scale_H(const Dims &G, float *lam, const float *im, bool inverse, cudaStream_t st)
{
    const long long n = 3 * G.nc;
    k_scale_H<<<(unsigned)std::min<long long>((n + 255) / 256, 1 << 20), 256, 0, st>>>(lam + 3 * G.nc, im, G.nc, inverse);
}

void launch_record(const Dims &G, const RecLayout &R, const float *fields_H, const float *fields_E,
                   float *rec, const int *step, cudaStream_t st)
{
    if (R.stride == 0) return;
    k_record<false, false><<<(unsigned)((R.stride + 255) / 256), 256, 0, st>>>(G, R, fields_H, fields_E, nullptr, rec, step);
}

void launch_record_pp(const Dims &G, const RecLayout &R, const float *bufA, const float *bufB, float *rec,
                      const int *step, cudaStream_t st)
{
    if (R.stride == 0) return;
    k_record<false, true><<<(unsigned)((R.stride + 255) / 256), 256, 0, st>>>(G, R, bufA, bufB, nullptr, rec, step);
}

// grid of the pipe kernels: x = blocks over the largest face, y = the 12 segments of a step's record
static dim3 pipe_grid(const RecLayout &R)
{
    const long long c = std::max(R.cells[0], std::max(R.cells[1], R.cells[2]));
    return dim3((unsigned)((c + 128 * PIPE_U - 1) / (128 * PIPE_U)), 12, 1);
}
static PipeTable pipe_table(const Dims &G, const RecLayout &R)
{
    PipeTable T;
    const long long str[3] = { 1, G.nx, (long long)G.nx * G.ny };
    for (int seg = 0; seg < 12; ++seg) {
        const int a = seg >> 2, side = (seg >> 1) & 1, which = seg & 1;
        const int fa = R.fast[a], sl = R.slow[a], comp = (a + 1 + which) % 3;
        PipeSeg &q = T.s[seg];
        q.side = side;
        q.cells = (unsigned)R.cells[a];
        q.nf = (unsigned)(G.hi[fa] - G.lo[fa]);
        q.sf = str[fa]; q.ss = str[sl];
        q.base = (long long)(side ? comp : 3 + comp) * G.nc + (side ? G.hi[a] : G.lo[a] - 1) * str[a] + G.lo[fa] * str[fa] + G.lo[sl] * str[sl];
        q.off = R.off[a][side][which];
    }
    T.stride = R.stride; T.half = R.half;
    return T;
}

void launch_record_pipe(const Dims &G, const RecLayout &R, const float *bufA, const float *bufB, float *rec,
                        const int *step, int n_steps, cudaStream_t st)
{
    if (R.stride == 0) return;
    k_record_pipe<<<pipe_grid(R), 128, 0, st>>>(pipe_table(G, R), bufA, bufB, rec, step, n_steps);
}

void launch_inject_pipe(const Dims &G, const RecLayout &R, float *bufA, float *bufB, const float *rec,
                        const int *step, cudaStream_t st)
{
    if (R.stride == 0) return;
    k_inject_pipe<<<pipe_grid(R), 128, 0, st>>>(pipe_table(G, R), bufA, bufB, rec, step);
}

void launch_inject_pp(const Dims &G, const RecLayout &R, float *bufA, float *bufB, const float *rec,
                      const int *step, cudaStream_t st)
{
    if (R.stride == 0) return;
    k_record<true, true><<<(unsigned)((R.stride + 255) / 256), 256, 0, st>>>(G, R, bufA, bufB, nullptr, const_cast<float *>(rec), step);
}

void launch_inject(const Dims &G, const RecLayout &R, float *fields, const float *rec, const int *step, cudaStream_t st)
{
    if (R.stride == 0) return;
    k_record<true, false><<<(unsigned)((R.stride + 255) / 256), 256, 0, st>>>(G, R, nullptr, nullptr, fields, const_cast<float *>(rec), step);
}

void launch_advance(int *step, int delta, cudaStream_t st) { k_advance<<<1, 1, 0, st>>>(step, delta); }
void launch_next_step(const int *in, int *out, int delta, cudaStream_t st) { k_next_step<<<1, 1, 0, st>>>(in, out, delta); }
void launch_set_step(int *p, int v, cudaStream_t st) { k_set_step<<<1, 1, 0, st>>>(p, v); }

void launch_adj_H(const Dims &G, const Tables &T, float *lam, const float *im, PsiSet s0, PsiSet s1,
                  const int *step, cudaStream_t st)
{
    if (G.periodic) k_adjoint<1, true><<<vol_grid(G), vol_block(), 0, st>>>(G, T, lam, im, s0, s1, step, nullptr);
    else            k_adjoint<1, false><<<vol_grid(G), vol_block(), 0, st>>>(G, T, lam, im, s0, s1, step, nullptr);
}

void launch_adj_E(const Dims &G, const Tables &T, float *lam, const float *ie, PsiSet s0, PsiSet s1,
                  const int *step, cudaStream_t st, const float *sigma)
{
    if (G.periodic) k_adjoint<0, true><<<vol_grid(G), vol_block(), 0, st>>>(G, T, lam, ie, s0, s1, step, sigma);
    else            k_adjoint<0, false><<<vol_grid(G), vol_block(), 0, st>>>(G, T, lam, ie, s0, s1, step, sigma);
    // the cotangent of the pre-update E is Ca lamE' (the gather-form kernel reads its neighbours' lamE': scaled afterwards)
    if (sigma) k_lossy_scale_E<<<(unsigned)std::min<long long>((G.nc + 255) / 256, 1 << 20), 256, 0, st>>>(G, lam, ie, sigma);
}

void launch_grad_rho(const Dims &G, const float *g, const float *ie, float delta_eps, const int lo[3], const int hi[3],
                     float *out, cudaStream_t st)
{
    const int bx = hi[0] - lo[0], by = hi[1] - lo[1], bz = hi[2] - lo[2];
    const long long n = (long long)bx * by * bz;
    k_grad_rho<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(G, g, ie, delta_eps, lo[0], lo[1], lo[2], bx, by, bz, out);
}

void launch_inv_H(const Dims &G, float *fields, const float *im, cudaStream_t st, const float *lam, const float *lam2,
                  const int *step, bool scaled, float *g_mu)
{
    if (G.periodic) k_inv_H<true><<<vol_grid(G), vol_block(), 0, st>>>(G, fields, im, lam, lam2, step, scaled ? 1 : 0, g_mu);
    else            k_inv_H<false><<<vol_grid(G), vol_block(), 0, st>>>(G, fields, im, lam, lam2, step, scaled ? 1 : 0, g_mu);
}

// ------------------------------------------------------------------------------------------ checkpointed reverse sweep
// ("checkpointing": no inverse step.)  On the gradient box [glo, ghi) -- any box of the grid,
// PML cells included -- the replayed forward pass stores, per step, D_c = dE'_c / d inv_eps, and the adjoint sweep forms
// g += sum_c lamE'_c D_c.  Lossless: E' = E + S ie bracket + src, so D = (E' - E - src) / ie.  Lossy (reading R29):
// E' = Ca E + Cb S ie bracket + src, D = dCa E + F (E' - Ca E - src), F = (dCb ie + Cb) / (Cb ie),
// dCa = -sigma S Cb^2, dCb = -(sigma S / 2) Cb^2.  The slot of step n in the buffer is n % K (K = steps per segment).
// mode 0: state n in volume n&1 of (A, B), state n+1 in the other (the fused ping-pong);
// mode 1: before an in-place step, the slot takes E;  mode 2: after it, the slot becomes D.
__global__ void k_dE_store(Dims G, const float *__restrict__ A, const float *__restrict__ B, float *__restrict__ dE, int K, int mode,
                           const float *__restrict__ ie, const float *__restrict__ sigma, const int *__restrict__ step)
{
    const int bx = G.ghi[0] - G.glo[0], by = G.ghi[1] - G.glo[1], bz = G.ghi[2] - G.glo[2];
    const long long bc = (long long)bx * by * bz;
    const int n = *step;
    dE += (long long)(n % K) * 3 * bc;
    const float *En = A, *En1 = B;
    if (mode == 0 && (n & 1)) { En = B; En1 = A; }
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < bc; t += (long long)gridDim.x * blockDim.x) {
        const int i = G.glo[0] + (int)(t % bx), j = G.glo[1] + (int)((t / bx) % by), k = G.glo[2] + (int)(t / ((long long)bx * by));
        const long long p = lin(G, i, j, k);
        for (int c = 0; c < 3; ++c) {
            const float e = __ldg(ie + (G.aniso ? c * G.nc : 0) + p);
            const float hs = sigma ? 0.5f * __ldg(sigma + p) * G.S : 0.f, Cb = 1.f / (1.f + hs * e), Ca = (1.f - hs * e) * Cb;
            const float dCa = -2.f * hs * Cb * Cb, F = (-hs * Cb * Cb * e + Cb) / (Cb * e);
            float *o = dE + c * bc + t;
            if (mode == 0 && !sigma) *o = (En1[c * G.nc + p] - En[c * G.nc + p]) / e;
            else if (mode == 0) { const float E0 = En[c * G.nc + p]; *o = fmaf(dCa, E0, F * (En1[c * G.nc + p] - Ca * E0)); }
            else if (mode == 1) *o = En[c * G.nc + p];
            else { const float E0 = *o; *o = fmaf(dCa, E0, F * (En[c * G.nc + p] - Ca * E0)); }
        }
    }
}
// D_c -= F profile * waveform[n] where an E source of component c overlaps the box
__global__ void k_dE_source(Dims G, float *__restrict__ dE, int K, SourceDev s, const float *__restrict__ ie,
                            const float *__restrict__ sigma, const int *__restrict__ step)
{
    const int bx = s.hi[0] - s.lo[0], by = s.hi[1] - s.lo[1], bz = s.hi[2] - s.lo[2];
    const long long n_cells = (long long)bx * by * bz;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_cells) return;
    const int i = s.lo[0] + (int)(t % bx), j = s.lo[1] + (int)((t / bx) % by), k = s.lo[2] + (int)(t / ((long long)bx * by));
    if (i < G.glo[0] || i >= G.ghi[0] || j < G.glo[1] || j >= G.ghi[1] || k < G.glo[2] || k >= G.ghi[2]) return;
    const int gx = G.ghi[0] - G.glo[0], gy = G.ghi[1] - G.glo[1], gz = G.ghi[2] - G.glo[2];
    const long long bc = (long long)gx * gy * gz;
    const long long q = ((long long)(k - G.glo[2]) * gy + (j - G.glo[1])) * gx + (i - G.glo[0]);
    const int n = *step;
    const long long p = lin(G, i, j, k);
    const float e = __ldg(ie + (G.aniso ? s.comp * G.nc : 0) + p);
    const float hs = sigma ? 0.5f * __ldg(sigma + p) * G.S : 0.f, Cb = 1.f / (1.f + hs * e);
    const float F = (-hs * Cb * Cb * e + Cb) / (Cb * e);
    dE[(long long)(n % K) * 3 * bc + (long long)s.comp * bc + q] -= F * (s.profile ? __ldg(s.profile + t) : 1.f) * __ldg(s.waveform + n);
}
// g += sum_c lamE'_c D_c on the box; lamE' = the E part of the cotangents after B1 + B2 of reverse step n: volume n&1 of
// (lamA, lamB) after the fused adjoint step, lamA between the two adjoint kernels of the generic path
__global__ void k_grad_from_dE(Dims G, const float *__restrict__ lamA, const float *__restrict__ lamB, const float *__restrict__ dE, int K,
                               float *__restrict__ g, const int *__restrict__ step)
{
    const int bx = G.ghi[0] - G.glo[0], by = G.ghi[1] - G.glo[1], bz = G.ghi[2] - G.glo[2];
    const long long bc = (long long)bx * by * bz;
    const int n = *step;
    dE += (long long)(n % K) * 3 * bc;
    const float *lam = (lamB && (n & 1)) ? lamB : lamA;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < bc; t += (long long)gridDim.x * blockDim.x) {
        const int i = G.glo[0] + (int)(t % bx), j = G.glo[1] + (int)((t / bx) % by), k = G.glo[2] + (int)(t / ((long long)bx * by));
        const long long p = lin(G, i, j, k);
        float acc = 0.f;
        for (int c = 0; c < 3; ++c) {
            const float v = lam[c * G.nc + p] * dE[c * bc + t];
            if (G.aniso) g[c * G.nc + p] += v; else acc += v;
        }
        if (!G.aniso) g[p] += acc;
    }
}

void launch_dE_store(const Dims &G, const float *A, const float *B, float *dE, int K, int mode, const float *ie, const float *sigma,
                     const int *step, cudaStream_t st)
{
    const long long n = (long long)(G.ghi[0] - G.glo[0]) * (G.ghi[1] - G.glo[1]) * (G.ghi[2] - G.glo[2]);
    k_dE_store<<<(unsigned)std::min<long long>((n + 255) / 256, 1 << 16), 256, 0, st>>>(G, A, B, dE, K, mode, ie, sigma, step);
}
void launch_dE_source(const Dims &G, float *dE, int K, const SourceDev &s, const float *ie, const float *sigma, const int *step, cudaStream_t st)
{
    const long long n = (long long)(s.hi[0] - s.lo[0]) * (s.hi[1] - s.lo[1]) * (s.hi[2] - s.lo[2]);
    k_dE_source<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(G, dE, K, s, ie, sigma, step);
}
void launch_grad_from_dE(const Dims &G, const float *lamA, const float *lamB, const float *dE, int K, float *g,
                         const int *step, cudaStream_t st)
{
    const long long n = (long long)(G.ghi[0] - G.glo[0]) * (G.ghi[1] - G.glo[1]) * (G.ghi[2] - G.glo[2]);
    k_grad_from_dE<<<(unsigned)std::min<long long>((n + 255) / 256, 1 << 16), 256, 0, st>>>(G, lamA, lamB, dE, K, g, step);
}

void launch_inv_E_grad(const Dims &G, float *fields, const float *ie, const float *lam, float *g, cudaStream_t st)
{
    if (G.periodic) k_inv_E_grad<true><<<vol_grid(G), vol_block(), 0, st>>>(G, fields, ie, lam, g, nullptr, nullptr);
    else            k_inv_E_grad<false><<<vol_grid(G), vol_block(), 0, st>>>(G, fields, ie, lam, g, nullptr, nullptr);
}

void launch_inv_E_grad_pp(const Dims &G, float *fields, const float *ie, const float *lamA, const float *lamB,
                          const int *step, float *g, cudaStream_t st)
{
    k_inv_E_grad<false><<<vol_grid(G), vol_block(), 0, st>>>(G, fields, ie, lamA, g, lamB, step);
}

}  // namespace fdtd
