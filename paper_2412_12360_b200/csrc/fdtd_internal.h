// fdtd_internal.h -- private structures shared by the host API and the kernels.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/fdtd.h"

namespace fdtd {

// ----------------------------------------------------------------------------------------------
// Geometry shared by every kernel (passed by value).
// ----------------------------------------------------------------------------------------------
struct Dims {
    int nx, ny, nz;
    int d;            // CPML thickness
    int dpx;          // half-width of the x-slab psi storage (d rounded up to 4 when it fits)
    int periodic;
    float S;
    long long nc;     // cells
    int lo[3], hi[3]; // interior box I
    int glo[3], ghi[3]; // gradient box (already clipped to I)
    // z-slab sub-grid: the local planes are global planes [zoff, zoff + nz) of a grid of nzg
    // planes; zl / zh = how many of the first / last local planes lie in the global low / high z CPML slab (d / d on
    // an ordinary grid).  CPML tables are stored per local plane; the z-slab psi arrays keep 2 d planes.
    int zoff, nzg, zl, zh;
    int aniso;        // N4 (reading R30): inv_eps and dL/d inv_eps are [3][nc], one volume per E component
};

// slab-compact plane of local plane k in a z-slab psi array ([0, zl) low slab, [2 d - zh, 2 d) high slab), or -1
__host__ __device__ inline int zslab_pos(const Dims &G, int k)
{
    if (k < 0 || k >= G.nz) return -1;
    if (k < G.zl) return k;
    if (k >= G.nz - G.zh) return 2 * G.d - G.zh + (k - (G.nz - G.zh));
    return -1;
}

// CPML tables on the device: [family 0=E 1=H][axis] -> pointer to N_axis floats
struct Tables {
    const float *b[2][3];
    const float *a[2][3];
    const float *ik[2][3];
};

// psi arrays: [component c][s]; array (c,s) belongs to derivative axis (c+1+s)%3 and is stored
// slab-compact on the two slabs normal to that axis:
//   axis x: [nz][ny][2*dpx]   axis y: [nz][2*d][nx]   axis z: [2*d][ny][nx]
struct PsiSet {
    float *p[3][2];
};

__host__ __device__ inline int psi_axis(int c, int s) { return (c + 1 + s) % 3; }

__host__ __device__ inline long long psi_elems(const Dims &G, int axis)
{
    if (G.d == 0) return 0;
    if (axis == 0) return (long long)G.nz * G.ny * (2 * G.dpx);
    if (axis == 1) return (long long)G.nz * (2 * G.d) * G.nx;
    return (long long)(2 * G.d) * G.ny * G.nx;
}

// slab-compact index of cell (i,j,k) in a psi array of `axis`, or -1 if the cell is not in the PML
// slab of that axis.
__host__ __device__ inline long long psi_index(const Dims &G, int axis, int i, int j, int k)
{
    if (axis == 0) {
        int s;
        if (i < G.d) s = i; else if (i >= G.nx - G.d) s = i - (G.nx - 2 * G.dpx); else return -1;
        return ((long long)k * G.ny + j) * (2 * G.dpx) + s;
    } else if (axis == 1) {
        int s;
        if (j < G.d) s = j; else if (j >= G.ny - G.d) s = j - (G.ny - 2 * G.d); else return -1;
        return ((long long)k * (2 * G.d) + s) * G.nx + i;
    } else {
        const int s = zslab_pos(G, k);
        if (s < 0) return -1;
        return ((long long)s * G.ny + j) * G.nx + i;
    }
}

// ----------------------------------------------------------------------------------------------
// Interface recorder (reading R15).  One step's record = 12 segments:
// for axis a: [low H_{a+1}] [low H_{a+2}] [high E'_{a+1}] [high E'_{a+2}], each holding the face
// cells (other two indices over I; the lower-numbered of the two other axes is fastest), padded to
// a multiple of 4 floats.
// ----------------------------------------------------------------------------------------------
struct RecLayout {
    long long off[3][2][2];   // [axis][side 0=low,1=high][which]
    long long cells[3];       // face cells per axis
    int fast[3], slow[3];     // the two in-face axes
    long long stride;         // elements per step (multiple of 32)
    int half;                 // 1: elements are fp16 (FDTD_FLAG_RECORDER_FP16), 0: fp32
};

struct SourceDev {
    int comp;
    int lo[3], hi[3];
    const float *profile;
    const float *waveform;
};

struct DetectorDev {
    int mask, ncomp;
    int lo[3], hi[3];
    int n_freq;
    int cs_off;               // offset (in frequencies) into the per-step cos/sin table
    float *phasor;            // forward: accumulate into;  backward: cotangent (may be NULL)
};

// ----------------------------------------------------------------------------------------------
// Generic (one thread per cell) kernel launchers -- kernels_generic.cu
// All kernels read the current step index n from *step (device memory) so that the per-step
// launch sequence is identical for every n and can be replayed from a CUDA graph.
// ----------------------------------------------------------------------------------------------
// sigma: N4 (reading R29), normalised electric conductivity per voxel or NULL
void launch_update_E(const Dims &G, const Tables &T, float *fields, const float *ie, PsiSet psiE, cudaStream_t st,
                     const float *sigma = nullptr);
void launch_update_H(const Dims &G, const Tables &T, float *fields, const float *im, PsiSet psiH, cudaStream_t st);
void launch_add_source(const Dims &G, float *fields, const SourceDev &s, const int *step, float sign, cudaStream_t st);
void launch_detector(const Dims &G, const float *fields, const DetectorDev &dt, const float *cs_table,
                     int total_freq, const int *step, cudaStream_t st);
void launch_detector_adjoint(const Dims &G, float *lam, const DetectorDev &dt, const float *cs_table,
                             int total_freq, const int *step, cudaStream_t st);
// H source: fields that hold the pre-step H (low faces); E source: fields that hold the post-E-update E'
void launch_record(const Dims &G, const RecLayout &R, const float *fields_H, const float *fields_E,
                   float *rec, const int *step, cudaStream_t st);
// ping-pong variants for the fused path (buffers picked by step parity inside the kernel)
void launch_record_pp(const Dims &G, const RecLayout &R, const float *bufA, const float *bufB, float *rec,
                      const int *step, cudaStream_t st);
void launch_record_pipe(const Dims &G, const RecLayout &R, const float *bufA, const float *bufB, float *rec,
                        const int *step, int n_steps, cudaStream_t st);
void launch_inject_pipe(const Dims &G, const RecLayout &R, float *bufA, float *bufB, const float *rec,
                        const int *step, cudaStream_t st);
void launch_inject_pp(const Dims &G, const RecLayout &R, float *bufA, float *bufB, const float *rec,
                      const int *step, cudaStream_t st);
void launch_inject(const Dims &G, const RecLayout &R, float *fields, const float *rec, const int *step, cudaStream_t st);
void launch_advance(int *step, int delta, cudaStream_t st);
// two-slot step counter: step p reads slot p&1; one kernel of that step writes the other slot for the next step
void launch_next_step(const int *in, int *out, int delta, cudaStream_t st);
void launch_set_step(int *p, int v, cudaStream_t st);
// psi cotangents are ping-ponged by step parity: read set[n&1], write set[(n&1)^1]
void launch_adj_H(const Dims &G, const Tables &T, float *lam, const float *im, PsiSet set0, PsiSet set1,
                  const int *step, cudaStream_t st);
void launch_adj_E(const Dims &G, const Tables &T, float *lam, const float *ie, PsiSet set0, PsiSet set1,
                  const int *step, cudaStream_t st, const float *sigma = nullptr);
void launch_grad_rho(const Dims &G, const float *g, const float *ie, float delta_eps, const int lo[3], const int hi[3],
                     float *out, cudaStream_t st);
// N4: with g_mu, dL/d inv_mu is accumulated from the cotangent of the post-step H (the H part of lam, or of the
// fused sweep's volume (n+1)&1 of lam / lam2, which holds im lamH when `scaled`)
void launch_inv_H(const Dims &G, float *fields, const float *im, cudaStream_t st, const float *lam = nullptr,
                  const float *lam2 = nullptr, const int *step = nullptr, bool scaled = false, float *g_mu = nullptr);
void launch_inv_E_grad(const Dims &G, float *fields, const float *ie, const float *lam, float *g, cudaStream_t st);
// checkpointed reverse sweep (record = 3): D = dE'/d inv_eps per replayed step on the gradient box (slot n % K), g += sum_c lamE'_c D_c
void launch_dE_store(const Dims &G, const float *A, const float *B, float *dE, int K, int mode, const float *ie, const float *sigma,
                     const int *step, cudaStream_t st);
void launch_dE_source(const Dims &G, float *dE, int K, const SourceDev &s, const float *ie, const float *sigma, const int *step, cudaStream_t st);
void launch_grad_from_dE(const Dims &G, const float *lamA, const float *lamB, const float *dE, int K, float *g,
                         const int *step, cudaStream_t st);
// fused path: cotangent volumes are ping-ponged by step parity
void launch_inv_E_grad_pp(const Dims &G, float *fields, const float *ie, const float *lamA, const float *lamB,
                          const int *step, float *g, cudaStream_t st);
// im != NULL: the H part of the volumes holds im lamH, so H-component cotangents are scaled by im at their cell
void launch_detector_adjoint_pp(const Dims &G, float *lamA, float *lamB, const DetectorDev &dt, const float *cs_table,
                                int total_freq, const int *step, const float *im, cudaStream_t st);
// H part of a cotangent volume: lamH *= im (inverse = false) or lamH /= im (inverse = true)
void launch_scale_H(const Dims &G, float *lam, const float *im, bool inverse, cudaStream_t st);

// ----------------------------------------------------------------------------------------------
// N2: time-domain detectors, Poynting flux from phasors, TFSF plane source
// -- kernels_n2.cu.  A time-domain detector fires after step n when (n+1) % stride == 0 (record index
// (n+1)/stride - 1); the kernels read n from *step and return at once on the other steps, so the per-step launch
// sequence stays replayable.
// ----------------------------------------------------------------------------------------------
struct TimeDetDev {
    int kind;                 // 0 snapshot, 1 energy
    int mask, ncomp;
    int lo[3], hi[3];
    int stride;
    float *out;               // forward: written;  backward: cotangent (may be NULL)
};
struct ReduceScratch {        // block partials + ticket of the last-block-done reductions (grid owned)
    double *partial;          // [RED_BLOCKS]
    unsigned int *ticket;
};
constexpr int RED_BLOCKS = 1024;
// volA / volB: the state after step n sits in volA, or (fused ping-pong, volB != NULL) in the volume of parity
// (n + par_off) & 1 (0: volA)
void launch_time_detect(const Dims &G, const float *volA, const float *volB, int par_off, const float *ie, const float *im,
                        const TimeDetDev &td, const ReduceScratch &rs, const int *step, cudaStream_t st);
// transpose at reverse step n: cotangent volume lamA / lamB and primal volume fA / fB picked by parity like above;
// scaled_H: the H part of the cotangent volumes holds im lamH; g: dL/d inv_eps or NULL
void launch_time_detect_adjoint(const Dims &G, float *lamA, float *lamB, const float *fA, const float *fB, int par_off,
                                const float *ie, const float *im, bool scaled_H, const TimeDetDev &td, float *g,
                                const int *step, cudaStream_t st);
// flux_f = 1/2 sum Re(E_b conj(H_c) - E_c conj(H_b)) on the plane (reading R24); cw, sw = cos, sin(omega_f / 2)
void launch_flux(const DetectorDev &dt, const float *phasor, int axis, int interpolate, int f, float cw, float sw,
                 float *flux, const ReduceScratch &rs, cudaStream_t st);
void launch_flux_vjp(const DetectorDev &dt, const float *phasor, int axis, int interpolate, int f, float cw, float sw,
                     const float *dL_dflux, float *dL_dphasor, cudaStream_t st);
// auxiliary 1-D leapfrog of the TFSF plane source (reading R25); returns cudaErrorInvalidValue when n_steps is too large
cudaError_t launch_tfsf_aux(float S, float ie, float im, float sgn, float dir_sign, int n_steps, const float *base,
                            float *wE, float *wH, cudaStream_t st);

}  // namespace fdtd
