/*
 * fdtd.h -- C ABI of the B200-native FDTD hot path (arXiv 2412.12360, "FDTDX").
 *
 * What the library computes (citations: /root/reference/PAPER.md line numbers; the
 * discretisation choices the paper leaves open are the readings R1..R30 of DESIGN.md):
 *
 *   forward  : n_steps of the Yee-grid leapfrog (Eq. 1-2; Yee staggering L68):
 *              E update with per-voxel inverse permittivity and CPML psi_E recursion (L72),
 *              additive E sources (L72), [record interface values, L84], H update with per-voxel
 *              inverse permeability and CPML psi_H, additive H sources, running-DFT detectors
 *              (L68 "detector object"; interpolation off, L70).
 *   backward : the memory-efficient gradient of L84: for n = n_steps-1 .. 0 an inverse update
 *              reconstructs the interior fields of step n from those of step n+1 (the PML is not
 *              invertible, so the recorded PML/interior interface values are re-imposed), fused
 *              with the vector-Jacobian product (L78-84) that propagates the cotangents through
 *              the whole grid (adjoint CPML included) and accumulates dL/d(inv_eps) per voxel.
 *
 * Conventions
 *   grid nx*ny*nz cells, cell (i,j,k), x fastest: lin = (k*ny + j)*nx + i.  All volumes are fp32
 *   [nz][ny][nx].  `fields` is [6][nz][ny][nx], components Ex,Ey,Ez,Hx,Hy,Hz.  H is scaled by
 *   eta0, lengths by dx, times by dt: the only constant is the Courant number S = c dt/dx.
 *   For component c let a = c+1, b = c+2 (mod 3):
 *     E_c += S*ie*( ikE_a*dm_a H_b - ikE_b*dm_b H_a + psiE_c0 - psiE_c1 ),  dm_a F[p] = F[p]-F[p-e_a]
 *     H_c -= S*im*( ikH_a*dp_a E_b - ikH_b*dp_b E_a + psiH_c0 - psiH_c1 ),  dp_a F[p] = F[p+e_a]-F[p]
 *   (H from the just-updated E).  A neighbour outside the grid is the wrapped cell on a periodic
 *   grid and 0 otherwise.  One step n maps (E^n, H^{n+1/2}) to (E^{n+1}, H^{n+3/2}).
 *   Interior box I = [d, N-d) on every axis (d = pml_cells); whole grid when d == 0.
 *
 * Memory / ownership
 *   Every pointer marked DEVICE is caller-owned CUDA device memory (e.g. a PyTorch allocation),
 *   contiguous and 16-byte aligned; the library never frees or retains it beyond the call.
 *   Pointers marked HOST are ordinary host memory read during the call.  The grid object owns
 *   only scratch: CPML tables, psi slabs, cotangent fields, ping-pong copies, the recorder.
 *
 *   Everything the entry points need is allocated by fdtd_create_grid: psi slabs, the recorder and (record != 0)
 *   the cotangent volumes and their psi slabs, the fused path's ping-pong volumes, the DFT phase table for up to
 *   16 frequencies x max_steps, and with FDTD_FLAG_HOST_STAGING the staging buffers of the *_host entry points.
 *   Allocated on first use instead (cudaMalloc inside the call): the cotangent volumes when fdtd_backward runs
 *   on a grid created with record == 0 (adjoint sweep only), a larger phase table when a call passes more than 16
 *   frequencies in total, the *_host staging buffers without the flag (and those of inv_mu / dL_dfields, which
 *   are optional arguments, in any case).
 *
 * Execution
 *   All work is enqueued on `cuda_stream` (a cudaStream_t passed as void*, NULL = legacy default
 *   stream).  The device entry points never wait for kernels and copy nothing device->host.  They may wait for
 *   the host->device upload of a small host-built table of the PREVIOUS call on the same grid (the DFT phase
 *   table, the TMA descriptors: pinned staging that is about to be rewritten), which is over unless the calls
 *   follow each other within microseconds.  fdtd_create_grid is synchronous: on the fused path it also times
 *   the step kernels on scratch volumes (calibration of the work partition: ~30 launches per kernel, a
 *   temporary allocation of 7 volumes, cudaDeviceSynchronize).  The *_host entry points (below) copy
 *   host<->device and synchronise the stream.
 *
 * Kernel paths
 *   FDTD_PATH_AUTO picks the fused TMA kernels (one kernel per time step forward, adjoint step + inverse step
 *   per reverse time step) when ALL of these hold, else the generic one-thread-per-cell kernels:
 *     - not periodic; nx % 4 == 0; nx >= 2*roundup4(pml_cells); fewer than 2^31 - 4*nx*ny cells;
 *     - a compiled tile shape fits in shared memory and the driver provides cuTensorMapEncodeTiled.
 *   On a fused grid a single call still runs on the generic kernels when it passes more than 4 sources or
 *   more than 4 detectors (the fused kernels' parameter block has 4 slots each; under FDTD_PATH_FUSED such a
 *   call fails with EINVAL).  In fdtd_backward, detectors with a cotangent on an H component are injected
 *   by a small kernel per detector and step instead of inside the adjoint step kernel.  inv_mu, one inv_eps per
 *   component (FDTD_FLAG_ANISO_EPS) and a conductivity (fdtd_set_conductivity) are taken by both paths in both
 *   directions: the fused step kernels have a second instance that reads them at a thread's own cells.
 *   Results of the two paths agree to rounding (different summation order; the fused lossy step forms 1 / (1 + beta)
 *   with the hardware reciprocal, one unit in the last place).
 *
 * Errors
 *   Every function returns FDTD_OK (0) or a negative code; fdtd_last_error() returns a
 *   thread-local, never-NULL description of the last failure.  No exceptions, aborts or prints.
 */
#ifndef FDTD_B200_H
#define FDTD_B200_H

#include <stdint.h>
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define FDTD_API __attribute__((visibility("default")))
#else
#define FDTD_API
#endif

#define FDTD_OK        0
#define FDTD_EINVAL   -1   /* bad dims / Courant / boxes / NULL required pointer / n_steps > max_steps */
#define FDTD_ENOMEM   -2   /* device allocation failed (recorder, scratch)                           */
#define FDTD_ECUDA    -3   /* CUDA runtime / driver error; message holds cudaGetErrorString           */
#define FDTD_ESTATE   -4   /* backward on a CPML grid without a matching recorded forward              */

/* kernel path selection (fdtd_grid_desc.path) */
#define FDTD_PATH_AUTO     0   /* fused TMA kernels when the grid qualifies, else generic            */
#define FDTD_PATH_GENERIC  1   /* one-thread-per-cell kernels (periodic grids, odd sizes, debugging)  */
#define FDTD_PATH_FUSED    2   /* fused kernels; create_grid fails with EINVAL if not applicable      */

/* fdtd_grid_desc.flags */
#define FDTD_FLAG_HOST_STAGING  1   /* allocate the staging buffers of fdtd_forward_host / fdtd_backward_host
                                       (fields, inv_eps, and the gradient when record != 0) in fdtd_create_grid */

#define FDTD_FLAG_RECORDER_FP16  2   /* SURVEY 8(f) N1, reduced-precision recorder: the interface values are stored as
                                       fp16 (round to nearest) instead of fp32, halving the recorder (C3: 2.97 -> 1.49 GB,
                                       C4: 117 -> 58 GB).  An approximation, off by default: the reconstructed fields carry
                                       the rounding (2^-11 relative per recorded value); the gradient error this costs is
                                       measured in tests/test_gpu_parity.py and stated in DESIGN.md.                       */

#define FDTD_FLAG_ANISO_EPS  4       /* SURVEY 8(f) N4, reading R30: inv_eps is [3][nz][ny][nx], one volume per E component (E_c is
                                       updated with inv_eps[c] at its own staggered position: what sub-pixel smoothing of an
                                       interface produces), and dL_dinv_eps is [3][nz][ny][nx] likewise.  Both kernel paths;
                                       not with fdtd_grad_rho, the energy detector or the *_host entry points.               */

typedef struct fdtd_grid fdtd_grid;      /* opaque */

/* Grid descriptor.  A zero in any CPML constant selects its default (reading R8). */
typedef struct {
    int32_t nx, ny, nz;        /* cells per axis, each >= 1                                          */
    float   courant;           /* S = c*dt/dx, 0 < S < 1/sqrt(3) (stability for ie*im <= 1 everywhere;
                                  keeping S*sqrt(max ie*im) < 1/sqrt(3) is the caller's job)         */
    int32_t periodic;          /* 1: periodic box (pml_cells must be 0); 0: zero outside the grid    */
    int32_t pml_cells;         /* d >= 0; if d > 0 then 2*d + 2 <= min(nx,ny,nz)                     */
    float   pml_m;             /* polynomial grading order of sigma and kappa      (default 3)      */
    float   pml_sigma_scale;   /* sigma~_max = scale/sqrt(pml_eps_bg)              (default 0.8*(m+1)) */
    float   pml_kappa_max;     /* kappa at full depth                              (default 1)      */
    float   pml_alpha_max;     /* alpha~ at the interface, graded to 0 at full depth (default 0)    */
    float   pml_alpha_m;       /* grading order of alpha                           (default 1)      */
    float   pml_eps_bg;        /* background relative permittivity used in sigma~_max (default 1)   */
    int32_t max_steps;         /* upper bound of n_steps; sizes the recorder when record != 0       */
    int32_t record;            /* 0: forward only; 1: record the PML/interior interface every step; */
                               /* 2: record the faces of the gradient box instead (pml_cells > 0):  */
                               /*    fdtd_backward then reconstructs the fields on that box only;   */
                               /* 3: checkpointed reverse sweep: the  */
                               /*    whole state every checkpoint_every steps, no inverse step -- see */
                               /*    "Checkpointed reverse sweep" below                              */
    int32_t grad_lo[3];        /* half-open (i,j,k) box on which dL_dinv_eps is wanted;             */
    int32_t grad_hi[3];        /*   all zero => the whole interior I.  Always clipped to I.         */
    int32_t path;              /* FDTD_PATH_*                                                       */
    int32_t flags;             /* FDTD_FLAG_* bits                                                  */
    /* z-slab sub-grid (one simulation over several GPUs).  z_global == 0:
     * an ordinary grid.  Otherwise this grid holds the planes [z_offset, z_offset + nz) of a grid of z_global planes:
     * z_ghost_lo (0 or 1) ghost plane below and z_ghost_hi (0 or 1) above the planes it owns; the CPML tables, the
     * interior box and the recorder faces follow the GLOBAL position (an internal cut is recorded like a PML face, so
     * the reverse sweep's inverse step needs no exchange).  See "Domain decomposition" below. */
    int32_t z_global, z_offset, z_ghost_lo, z_ghost_hi;
    int32_t checkpoint_every;  /* record == 3: steps between checkpoints; 0 => about sqrt(max_steps)    */
    int32_t reserved[1];       /* must be zero                                                      */
} fdtd_grid_desc;

/* Additive source patch (reading R10/R11): during step n,
 * F_c[box] += profile[cell] * waveform[n], after the update of F's family (E or H).
 * A one-directional TFSF plane is one E patch plus one H patch. */
typedef struct {
    int32_t component;         /* 0..5 = Ex,Ey,Ez,Hx,Hy,Hz                                          */
    int32_t lo[3], hi[3];      /* half-open box in (i,j,k), inside the grid, non-empty              */
    const float *profile;      /* DEVICE, box-shaped [k][j][i]; NULL => 1.0                         */
    const float *waveform;     /* DEVICE, length >= n_steps                                         */
} fdtd_source;

/* Running-DFT detector (reading R13): after step n,
 * P_f[c][cell] += F_c[cell] * exp(-i*omega_f*(n+1)) for every component c in component_mask. */
typedef struct {
    int32_t component_mask;    /* bit c set => component c is accumulated                            */
    int32_t lo[3], hi[3];      /* half-open box in (i,j,k), inside the grid, non-empty              */
    int32_t n_freq;            /* >= 1                                                              */
    const float *omega;        /* HOST, n_freq angular frequencies in rad per step                  */
    float *phasor;             /* DEVICE, [n_freq][n_comp_set][box cells][2] (re,im), box cells
                                  ordered [k][j][i]; accumulated INTO (caller zeroes).  Ignored by
                                  fdtd_backward.                                                    */
} fdtd_detector;

/* Creates a grid: validates the descriptor, builds the CPML tables (fp64 on the host, stored
 * fp32), allocates psi slabs and, when record != 0, the recorder for max_steps steps.
 * Errors: EINVAL (see above), ENOMEM, ECUDA.  *out is NULL on failure. */
FDTD_API int fdtd_create_grid(const fdtd_grid_desc *desc, fdtd_grid **out);

/* Runs n_steps forward steps (0 <= n_steps <= max_steps) from the state in `fields`
 * (DEVICE, [6][nz][ny][nx]; in: state 0, out: state n_steps), with psi = 0 at entry (R21).
 * inv_eps: DEVICE [nz][ny][nx]; inv_mu: DEVICE [nz][ny][nx] or NULL (= 1).
 * src/det: HOST arrays of n_src / n_det descriptors (may be NULL when the count is 0).
 * With record != 0 the interface values of steps 0..n_steps-1 are stored in the grid. */
FDTD_API int fdtd_forward(fdtd_grid *grid, float *fields, const float *inv_eps, const float *inv_mu,
                 const fdtd_source *src, int32_t n_src,
                 const fdtd_detector *det, int32_t n_det,
                 int32_t n_steps, void *cuda_stream);

/* Time-reversed gradient of a scalar loss L(fields_n, phasors).
 * fields      : DEVICE, in: state n_steps as left by fdtd_forward; out: reconstructed state 0
 *               on I (cells outside I are unspecified).
 * src, det    : the descriptors of the forward call (sources are subtracted in the inverse step;
 *               detectors give geometry and omega).
 * dL_dphasor  : HOST array of n_det DEVICE pointers, each laid out like the detector's phasor
 *               (dL/dRe, dL/dIm); the array or any entry may be NULL (= zero cotangent).
 * dL_dfields  : DEVICE [6][nz][ny][nx] cotangent of state n_steps, or NULL (= 0).
 * dL_dinv_eps : DEVICE [nz][ny][nx], OUT; zero-filled by the library, non-zero only on
 *               I intersected with the grad box (R17).  inv_mu and source gradients are not computed.
 *               NULL (then dL_dfields0 is required) = adjoint sweep only: the cotangent of state 0 does not
 *               depend on the primal fields (the steps are linear in the fields), so nothing is reconstructed,
 *               `fields` is not touched and no recorded forward is needed.
 * dL_dfields0 : DEVICE [6][nz][ny][nx] OUT cotangent of state 0, or NULL.
 * Errors: ESTATE if dL_dinv_eps is wanted, pml_cells > 0 and the last fdtd_forward on this grid did not record
 *         exactly n_steps steps. */
FDTD_API int fdtd_backward(fdtd_grid *grid, float *fields, const float *inv_eps, const float *inv_mu,
                  const fdtd_source *src, int32_t n_src,
                  const fdtd_detector *det, int32_t n_det,
                  const float *const *dL_dphasor, const float *dL_dfields,
                  int32_t n_steps, float *dL_dinv_eps, float *dL_dfields0,
                  void *cuda_stream);

/* N4: fdtd_backward that also returns dL/d inv_mu (Eq. 1: the H update depends on
 * inv_mu at its own cell), dL_dinv_mu[p] = sum_n sum_c lamH'_c[p] * (-S (curl+ E')_c[p]) with lamH' the cotangent of
 * the post-step H.  DEVICE [nz][ny][nx], OUT, zero-filled by the library, non-zero only on the reconstruction box
 * (like dL_dinv_eps it needs the reconstructed fields, so dL_dinv_eps must be requested too).  NULL: fdtd_backward.
 * On the fused path the fused inverse step forms it (lamH' read at a thread's own cells); the inverse step of step n then has to
 * run before adjoint step n-1, so the two are launched one after the other instead of side by side. */
FDTD_API int fdtd_backward_mu(fdtd_grid *grid, float *fields, const float *inv_eps, const float *inv_mu,
                     const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                     const float *const *dL_dphasor, const float *dL_dfields,
                     int32_t n_steps, float *dL_dinv_eps, float *dL_dinv_mu, float *dL_dfields0, void *cuda_stream);

/* Checkpointed reverse sweep (record == 3, "checkpointing" as the alternative to time reversal).
 * fdtd_forward stores the whole state (fields and CPML psi) every checkpoint_every steps.  fdtd_backward then works segment by
 * segment from the last one: it restores the segment's checkpoint, runs the segment's forward steps again keeping
 * dE = E' - E (sources subtracted) on the gradient box for each of them, and runs the segment's adjoint steps with
 *   dL_dinv_eps[cell] += sum_c lamE'_c * dE_c / inv_eps      (= S lamE' . bracket of the E update: exact, no inverse step).
 * Nothing is reconstructed backwards in time, so: the gradient box (grad_lo / grad_hi; all zero = the whole grid) may
 * include PML cells, `fields` is scratch for the replay (unspecified on return), and the method does not rely on the update
 * being invertible.  Costs one
 * more forward pass; memory (max_steps / K) * (6 volumes + psi) + K * 3 * box cells floats (K = checkpoint_every).
 * Same result as the time-reversed sweep on the interior to its reconstruction rounding; equals the plain reverse-mode
 * derivative (the oracle's tape mode) on every cell.  Not available with time-domain detectors, range calls or sub-grids. */

/* N4, lossy media ("reversible ... for lossless materials"; reading R29): a normalised electric
 * conductivity per voxel, sigma~ = sigma eta0 dx (DEVICE [nz][ny][nx], caller-owned, must stay valid while it is set; NULL
 * removes it).  The E update becomes the semi-implicit lossy Yee update
 *   beta = sigma~ S inv_eps / 2,   E'_c = (1 - beta)/(1 + beta) E_c + 1/(1 + beta) S inv_eps bracket_c .
 * Such a step cannot be inverted stably, so the grid must have record == 0 (forward, adjoint sweep only) or record == 3 (the
 * checkpointed reverse sweep, which then delivers dL_dinv_eps); ESTATE otherwise.  Both kernel paths take it (the fused step
 * kernels read sigma~ at a thread's own cells).  On a fused record == 3 grid the first call that sets a conductivity allocates
 * three scratch volumes (the adjoint step leaves lamE' there before scaling it by (1 - beta)/(1 + beta)); ENOMEM if that fails. */
FDTD_API int fdtd_set_conductivity(fdtd_grid *grid, const float *sigma);

/* B6, chain rule to design parameters (once per gradient, not per step): for a design box whose
 * permittivity is eps = eps_bg + delta_eps*rho (reading R20),
 *   dL_drho[cell] = dL_dinv_eps[cell] * d(1/eps)/drho = -dL_dinv_eps[cell] * delta_eps * inv_eps[cell]^2.
 * dL_dinv_eps, inv_eps: DEVICE volumes; dL_drho: DEVICE, box-shaped [k][j][i], OUT. */
FDTD_API int fdtd_grad_rho(fdtd_grid *grid, const float *dL_dinv_eps, const float *inv_eps, float delta_eps,
                           const int32_t lo[3], const int32_t hi[3], float *dL_drho, void *cuda_stream);

/* ------------------------------------------------------------------------------------------
 * N2 -- the paper's source / detector set beyond the running DFT.
 *
 * Time-domain detectors ("access to intermediate fields, energy, Poynting flux"; L70: the six
 * components are taken at the same index, no Yee co-location, the paper's default; reading R23).
 * A detector fires after step n when (n+1) % stride == 0, record index q = (n+1)/stride - 1, on the state
 * (E^{n+1}, H^{n+3/2}) -- the time stamp of the DFT detectors:
 *   FDTD_TD_SNAPSHOT: out[q][ci][cell] = F_c[cell] for every component c of component_mask (ci counts the set bits);
 *   FDTD_TD_ENERGY  : out[q] = sum_cells 1/2 (sum_c E_c^2 / inv_eps + H_c^2 / inv_mu)   (eta0-normalised H).
 * out: DEVICE, snapshot [n_steps/stride][n_comp][box cells ordered k,j,i], energy [n_steps/stride]; written, not
 * accumulated.  In fdtd_backward_td the matching cotangent dL/d out has the same layout; the energy detector's
 * transpose reads the reconstructed primal fields, so its box must lie inside the reconstruction box (the
 * interior I, or the gradient box with record == 2) and dL_dinv_eps must be requested; it also adds the explicit
 * dependence on inv_eps, dL/d out[q] * (-1/2) sum_c E_c^2 / inv_eps^2, to dL_dinv_eps. */
#define FDTD_TD_SNAPSHOT 0
#define FDTD_TD_ENERGY   1
typedef struct {
    int32_t kind;              /* FDTD_TD_*                                                          */
    int32_t component_mask;    /* snapshot: bit c set => component c; energy: ignored               */
    int32_t lo[3], hi[3];      /* half-open box in (i,j,k), inside the grid, non-empty              */
    int32_t stride;            /* >= 1                                                              */
    float  *out;               /* DEVICE (see above).  Ignored by fdtd_backward_td.                 */
} fdtd_time_detector;

/* fdtd_forward / fdtd_backward with time-domain detectors (td: HOST array of n_td descriptors; dL_dtd: HOST array
 * of n_td DEVICE pointers, the array or any entry may be NULL).  With n_td == 0 they are fdtd_forward /
 * fdtd_backward.  Each detector adds one small kernel launch per time step. */
FDTD_API int fdtd_forward_td(fdtd_grid *grid, float *fields, const float *inv_eps, const float *inv_mu,
                    const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                    const fdtd_time_detector *td, int32_t n_td, int32_t n_steps, void *cuda_stream);
FDTD_API int fdtd_backward_td(fdtd_grid *grid, float *fields, const float *inv_eps, const float *inv_mu,
                     const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                     const float *const *dL_dphasor,
                     const fdtd_time_detector *td, int32_t n_td, const float *const *dL_dtd,
                     const float *dL_dfields, int32_t n_steps, float *dL_dinv_eps, float *dL_dfields0,
                     void *cuda_stream);

/* Poynting flux through a plane from the phasors of a DFT detector (Fig. 5 "fraction of
 * Poynting flux"; L70 Yee interpolation, off by default; reading R24).  The detector box is a slab normal to
 * `axis` a whose component_mask holds the four tangential components E_b, E_c, H_b, H_c (b = a+1, c = a+2 mod 3):
 *   flux[f] = 1/2 sum_cells Re( E_b conj(H_c) - E_c conj(H_b) )          (normal +e_a)
 * interpolate == 0: slab one plane thick, the phasors as accumulated (same index, same phase stamp);
 * interpolate == 1: slab two planes thick (p-1, p along a); E from plane p, H co-located with it in space,
 *   (H[p-1] + H[p])/2, and in time, multiplied by exp(-i omega_f / 2) (H is stamped half a step late).
 * det: HOST descriptor (geometry, mask, n_freq, omega; its phasor field is ignored); phasor: DEVICE, laid out as
 * fdtd_detector.phasor; flux: DEVICE [n_freq], written.  fdtd_flux_vjp writes dL_dphasor (DEVICE, same layout as
 * phasor, zero where the flux does not depend on it) from dL_dflux (DEVICE [n_freq]); pass it to fdtd_backward.
 * Errors: EINVAL if the mask lacks a tangential component or the slab thickness does not match. */
FDTD_API int fdtd_flux(fdtd_grid *grid, const fdtd_detector *det, const float *phasor, int32_t axis, int32_t interpolate,
              float *flux, void *cuda_stream);
FDTD_API int fdtd_flux_vjp(fdtd_grid *grid, const fdtd_detector *det, const float *phasor, int32_t axis, int32_t interpolate,
                  const float *dL_dflux, float *dL_dphasor, void *cuda_stream);

/* fdtd_flux for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): same flux, same arguments without the grid (whose only part in fdtd_flux is the reduction scratch
 * that fdtd_create_grid allocated).  This entry point calls no cudaMalloc / cudaFree and no allocating library routine: its
 * scratch (one block partial per 2048 plane cells + a ticket, 16.25 KB) is a file-scope `static __device__` array of the
 * library, held by every GPU that loads the library until the process exits.  Hence the limit: the plane may have at most
 * FDTD_FLUX_STATIC_MAX_CELLS cells (e.g. 2048 x 2048); beyond it EINVAL, use fdtd_flux.  The detector box is taken as it is
 * (no grid to check it against: lo >= 0, hi > lo).  Work: one 256-byte memset and n_freq kernels on cuda_stream; the first
 * call on a device also resolves the array's device address (cudaGetSymbolAddress), so make that call outside a capture.
 * All calls share the array and it keeps the last call's contents: what must start at zero is cleared on cuda_stream at
 * the start of every call, but calls that overlap on the GPU (other streams, other threads) race on it -- serialise them.
 * The sum over the plane is taken in a fixed order (deterministic); it differs from fdtd_flux's by rounding only.
 * det: HOST; phasor: DEVICE; flux: DEVICE [n_freq], written.  Errors: EINVAL as fdtd_flux, and for a plane beyond the limit. */
#define FDTD_FLUX_STATIC_MAX_CELLS 4194304
FDTD_API int fdtd_flux_static(const fdtd_detector *det, const float *phasor, int32_t axis, int32_t interpolate, float *flux,
                     void *cuda_stream);

/* One-directional plane source = Total-Field/Scattered-Field interface (reading R25).
 * A plane wave travelling along `axis` a in direction dir = +1 / -1, E polarised along pol = b != a, its H along the
 * third axis c, in a medium that is uniform (eps_r, mu_r) on the planes the interface touches.  The incident wave is
 * generated on an auxiliary 1-D grid with the 3-D grid's own update (same S, same medium, hard source
 * e[0] = base[n]), so it carries the grid's numerical dispersion and the field behind the interface cancels to
 * rounding.  Outputs the waveforms of the two additive patches (fdtd_source) that realise the interface at plane p0:
 *   E_b on plane p0, waveform wE;   H_c (component *h_component) on plane p0 + *h_plane_offset, waveform wH
 * (total-field side = the side the wave travels to; the caller supplies the transverse profile).
 * base, wE, wH: DEVICE, n_steps floats each; one kernel on cuda_stream, no grid needed.
 * Errors: EINVAL for bad axis / pol / dir or n_steps > 50000 (the auxiliary grid lives in shared memory). */
FDTD_API int fdtd_tfsf_plane(float courant, float eps_r, float mu_r, int32_t axis, int32_t pol, int32_t dir, int32_t n_steps,
                    const float *base, float *wE, float *wH, int32_t *h_component, int32_t *h_plane_offset,
                    void *cuda_stream);

/* ------------------------------------------------------------------------------------------
 * N3 -- domain decomposition along z (2.3 B cells over 4 GPUs).
 *
 * One simulation of z_global planes is cut into slabs of xy planes; each slab is a grid of its own (one per GPU /
 * process) created with z_global / z_offset / z_ghost_lo / z_ghost_hi.  A slab owns the planes
 * [z_offset + z_ghost_lo, z_offset + nz - z_ghost_hi) and carries one ghost plane on every side that is a cut:
 *   ghost below (local plane 0)     : holds the H-type components of the lower neighbour's top plane, imported;
 *   ghost above (local plane nz - 1): a replica of the upper neighbour's bottom plane -- its E-type components are
 *                                     updated here redundantly (bit-identical arithmetic), its H-type components are
 *                                     imported.  Everything else computed on ghost planes is overwritten or unused.
 * Protocol: advance all slabs by one step (fdtd_forward_range(n, n+1)), then every slab exports its lowest and its
 * highest owned plane (fdtd_halo_export: the three H-type components, [3][ny][nx]) and imports its neighbours'
 * (fdtd_halo_import); one exchange per full step, 3 nx ny floats per neighbour and direction.  The adjoint sweep
 * (fdtd_backward_range(n+1, n)) exchanges the H-type cotangents the same way (which = 1).  The primal inverse step of
 * the reverse sweep needs NO exchange: the interior box of a slab is the global interior restricted to its own
 * planes, and a cut is recorded like a PML face (tangential H of the ghost plane below before the step, tangential E'
 * of the ghost plane above after the E update), so every slab reconstructs its own planes from its own record.
 * Inputs per slab: inv_eps / inv_mu / dL_dfields are the local planes (ghosts included) of the global volumes;
 * sources are clipped to the local planes (ghosts included: the replica needs them); detectors are clipped to the
 * owned planes in fdtd_forward_range and to the local planes (with the matching slice of the cotangent) in
 * fdtd_backward_range.  All slabs must run the same kernel path.  On owned planes the fields, the phasors and the
 * cotangents are bit-identical to the undivided grid; dL_dinv_eps agrees to the rounding of the time reversal (next
 * to a cut the inverse step reads the recorded value where the undivided grid reads its reconstructed neighbour:
 * a few 1e-8 of the maximum; tests/test_gpu_subgrid.py).  Time-domain detectors are not available on range calls.
 *
 * fdtd_forward_range: steps n_begin .. n_end-1 of a run of n_total steps (n_begin == 0 starts a run: psi = 0; later
 *   calls must continue where the previous one ended, else ESTATE).  Between the calls of a sequence `fields` may be
 *   stale (the fused path keeps state n in its own second volume when n is odd); the call with n_end == n_total
 *   leaves state n_total in `fields`.  fdtd_forward is fdtd_forward_range(0, n_steps, n_steps).
 * fdtd_backward_range: reverse steps n_hi-1 .. n_lo (n_hi == n_total starts: B0 seeds from dL_dfields, zeroes
 *   dL_dinv_eps; n_lo == 0 ends: dL_dfields0 is written).  The same pointers must be passed to every call of a sequence.
 * fdtd_halo_export / fdtd_halo_import: which = 0 the fields holding state n (after fdtd_forward_range(.., n, ..)),
 *   which = 1 the cotangents after reverse step n (after fdtd_backward_range(.., n, ..)); side 0 = low end, 1 = high
 *   end; out / in: DEVICE [3][ny][nx].  Plane copies on cuda_stream.  The seed of the reverse sweep needs no exchange:
 *   dL_dfields is given on the local planes, ghosts included. */
FDTD_API int fdtd_forward_range(fdtd_grid *grid, float *fields, const float *inv_eps, const float *inv_mu,
                       const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                       int32_t n_begin, int32_t n_end, int32_t n_total, void *cuda_stream);
FDTD_API int fdtd_backward_range(fdtd_grid *grid, float *fields, const float *inv_eps, const float *inv_mu,
                        const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                        const float *const *dL_dphasor, const float *dL_dfields,
                        int32_t n_hi, int32_t n_lo, int32_t n_total, float *dL_dinv_eps, float *dL_dfields0,
                        void *cuda_stream);
FDTD_API int fdtd_halo_export(fdtd_grid *grid, float *fields, int32_t which, int32_t n, int32_t side, float *out, void *cuda_stream);
FDTD_API int fdtd_halo_import(fdtd_grid *grid, float *fields, int32_t which, int32_t n, int32_t side, const float *in, void *cuda_stream);

/* Peer stores: the exchange fused into the step kernel.  With a neighbour
 * attached, the fused step kernel that produces the H-type components of a slab's lowest / highest owned plane stores
 * them a second time, straight into the ghost plane of the neighbour's volume (same-process pointers, peer-mapped
 * pointers of another GPU, or pointers opened from another process's handle: plain stores over NVLink), and leaves the
 * H-type components of its own ghost plane on that side to the neighbour's kernel.  No plane copies, no
 * fdtd_halo_export / _import: what is left of the exchange is ordering -- all slabs finish step n before any starts
 * step n+1 (one stream in one process; a neighbour token or barrier across processes).  Fields, phasors and
 * cotangents stay bit-identical to the undivided grid (tests/test_gpu_subgrid.py).
 *
 * fdtd_halo_volumes: the two volumes of this grid's ping-pong that hold state n (n even: *vol0, n odd: *vol1);
 *   which = 0 the primal fields (`fields` is the pointer the range calls are given, *vol0 == fields), which = 1 the
 *   cotangents (allocated here if no reverse sweep ran yet).  DEVICE pointers, [6][nz][ny][nx], owned by the caller
 *   (fields) / the grid (the rest); they stay valid until fdtd_destroy.  ESTATE on a grid that runs the generic kernels.
 * fdtd_halo_attach: side 0 = the neighbour below, 1 = above; peer_vol0 / peer_vol1 = that neighbour's
 *   fdtd_halo_volumes of the same `which`, peer_nz its local plane count (ghosts included).  Both NULL detaches.  The
 *   pointers are kept as given: the neighbour's volumes (and an IPC mapping of them) must stay valid until this grid is
 *   detached or destroyed, and nothing checks that they are what they claim to be.  The
 *   grid must have a cut on that side and run the fused kernels (ESTATE otherwise); the neighbour must attach this
 *   grid in turn (a ghost plane on an attached side is written by the neighbour only).  While a neighbour is attached
 *   without flags (below) a range call must advance exactly one step (EINVAL otherwise) and the caller orders the steps
 *   of the slabs as stated above; a call that would run on the generic kernels (more than 4 sources / detectors) returns ESTATE.
 * fdtd_ipc_export / fdtd_ipc_open / fdtd_ipc_close: cudaIpcGetMemHandle / OpenMemHandle / CloseMemHandle behind this ABI,
 *   so that ranks can hand their volumes to each other without a CUDA binding of their own.  handle: HOST, 64 bytes;
 *   offset: the pointer's offset inside the allocation the handle names (a caching allocator hands out interior
 *   pointers).  fdtd_ipc_open returns the pointer itself (base + offset), valid in the calling process until
 *   fdtd_ipc_close(ptr, offset).  Volumes obtained from cudaMalloc (PyTorch's default allocator, this library) qualify;
 *   stream-ordered pools and expandable segments do not (ECUDA). */
/* Device-side ordering (csrc/halo_sync.cu): with flags attached on every attached side the slabs order their steps
 * themselves -- before a step a one-thread kernel waits (ld.acquire.sys) until the slab's own flags show the state it is
 * about to read, after a step another publishes the state reached in the neighbours' flags (st.release.sys) -- both as
 * graph nodes beside the step kernel, so a range call may advance ANY number of steps and replays without the host; no
 * token, no NCCL on the data path.  A wait passes when the flag shows the state wanted or the next one in the direction
 * of time (a neighbour may be one state ahead, never two), so the value a previous run left behind does not pass: runs
 * have at least 3 steps (EINVAL otherwise).  The slabs must then run concurrently (one GPU each): on ONE device the
 * calls have to be issued step by step in slab order on one stream, so that every wait finds its flag already set.
 * fdtd_halo_flags: this grid's two flags of `which` (DEVICE, int32[2]: [0] written by the neighbour below, [1] by the
 *   neighbour above), allocated by the first call; owned by the grid.
 * fdtd_halo_attach_flags: peer_flags = the fdtd_halo_flags pointer of the neighbour on `side` (same-process pointer or
 *   opened from its IPC handle); needs fdtd_halo_attach on that side first and this grid's own fdtd_halo_flags (ESTATE
 *   otherwise); NULL detaches the flag (fdtd_halo_attach(NULL, NULL) detaches both).
 * fdtd_halo_sync_error: a wait gives up after FDTD_HALO_TIMEOUT_MS (environment, default 10000) instead of hanging the
 *   device and raises a flag; this call reads and clears it (synchronous copy; *timed_out = 0: all waits were met,
 *   else 1 + the state index that never came).  The results of such a run are invalid. */
FDTD_API int fdtd_halo_flags(fdtd_grid *grid, int32_t which, int32_t **flags);
FDTD_API int fdtd_halo_attach_flags(fdtd_grid *grid, int32_t which, int32_t side, int32_t *peer_flags);
FDTD_API int fdtd_halo_sync_error(fdtd_grid *grid, int32_t *timed_out);
FDTD_API int fdtd_halo_volumes(fdtd_grid *grid, float *fields, int32_t which, float **vol0, float **vol1);
FDTD_API int fdtd_halo_attach(fdtd_grid *grid, int32_t which, int32_t side, float *peer_vol0, float *peer_vol1, int32_t peer_nz);
FDTD_API int fdtd_ipc_export(const void *dev_ptr, uint8_t handle[64], int64_t *offset);
FDTD_API int fdtd_ipc_open(const uint8_t handle[64], int64_t offset, void **dev_ptr);
FDTD_API int fdtd_ipc_close(void *dev_ptr, int64_t offset);

/* Frees the grid and everything it owns (synchronises the device first).  NULL is a no-op. */
FDTD_API int fdtd_destroy(fdtd_grid *grid);

/* Thread-local description of the last error on this thread ("" if none).  Never NULL. */
FDTD_API const char *fdtd_last_error(void);

/* Introspection for benchmarks and tests (no device work). */
typedef struct {
    int32_t path;                    /* FDTD_PATH_GENERIC or FDTD_PATH_FUSED actually in use          */
    int32_t tile_x, tile_y, tile_z;  /* fused path: cells per tile and z-chunk length (0 otherwise)  */
    int64_t kernel_launches;         /* kernels launched by this grid so far (graph nodes * replays) */
    int64_t recorder_bytes;          /* bytes of the interface recorder                              */
    int64_t scratch_bytes;           /* all other device bytes owned by the grid                     */
    int64_t record_floats_per_step;  /* recorder stride in floats                                    */
    int64_t pipelined_inverse_ctas;  /* CTAs of the inverse step in the pipelined reverse sweep; 0: sequential */
    int64_t fused_step_launches;     /* launches of the fused step kernel (forward + adjoint) so far         */
    int64_t fused_inverse_launches;  /* launches of the fused inverse step kernel so far                     */
    int64_t partition;               /* fused path: FDTD_PARTITION_* of the step kernels' work split         */
} fdtd_grid_info;
#define FDTD_PARTITION_NONE        0   /* generic path                                                    */
#define FDTD_PARTITION_CONTIGUOUS  1   /* the (column, plane) sequence cut into contiguous runs           */
#define FDTD_PARTITION_LOCKSTEP    2   /* columns of one cost class get identical cuts */
#define FDTD_PARTITION_WAVES       3   /* whole columns dealt out in waves, the rest cut to level the CTAs */
FDTD_API int fdtd_get_info(const fdtd_grid *grid, fdtd_grid_info *info);

/* Per-kernel timing for roofline reports.  While profiling is enabled the per-step kernels are
 * launched directly (no CUDA graph) and every launch of a step kernel is bracketed by CUDA events
 * recorded on the launch stream.  fdtd_get_profile synchronises those events and returns, per kernel
 * class, the number of launches and their summed device time since profiling was enabled (or since
 * the last fdtd_get_profile, which resets the counters). */
#define FDTD_PROF_CLASSES 16
typedef struct {
    int32_t n_classes;                          /* number of valid entries below                       */
    int32_t reserved;
    char    name[FDTD_PROF_CLASSES][32];        /* kernel class names, e.g. "fused_forward_step"       */
    int64_t launches[FDTD_PROF_CLASSES];
    double  total_ms[FDTD_PROF_CLASSES];
} fdtd_profile;
FDTD_API int fdtd_set_profiling(fdtd_grid *grid, int32_t enable);
FDTD_API int fdtd_get_profile(fdtd_grid *grid, fdtd_profile *out);

/* Host-only introspection of the fused step kernels' work partition (no device work, no
 * grid needed): the (tile column, plane) sequence of an nx x ny x nz grid with d CPML cells, tiles of
 * tile_x x tile_y cells, split into n_cta runs of equal model cost (a plane of a tile costs 1, + wy if the tile
 * has rows in a y slab, + wz if the plane is in a z slab).  lockstep != 0: the lock-step split (columns of one
 * cost class get identical cuts); 0: the plain contiguous split.  Writes up to `cap` segments as
 * {cta, i0, j0, k0, k1} (cells [i0, i0+tile_x) x [j0, j0+tile_y) clipped to the grid, planes [k0, k1)) into
 * `segments` (HOST, caller-owned, 5 int32 each), in marching order per CTA, and returns the number of segments
 * of the partition (which may exceed cap), or a negative FDTD_E* code for bad arguments. */
FDTD_API int fdtd_debug_partition(int32_t nx, int32_t ny, int32_t nz, int32_t d, int32_t tile_x, int32_t tile_y,
                         int32_t n_cta, double wy, double wz, int32_t lockstep, int32_t *segments, int32_t cap);

/* Bandwidth probe for the roofline discussion (bench.py --probe; not on the hot path): moves the step kernel's bytes -- 7 volumes
 * read, 6 written, float4 per thread -- without its arithmetic.  pattern 0: grid-stride streaming with `blocks` x `threads`, `runs` passes over the volumes per launch;
 * pattern 1: the step kernel's traversal, a block per (tile column of tile_y whole-x rows, run of nz / runs planes), `unroll`
 * (1, 2, 4) planes in flight per iteration; pattern 2: pattern 1 on ping-pong volumes, the way a time step hands its results to
 * the next (launch r reads the six volumes launch r-1 wrote plus the seventh of `in`; plain copies); pattern 3: pattern 2 with
 * the marching direction alternating from launch to launch.  in: DEVICE 7 * nx*ny*nz floats (patterns 2, 3 also WRITE its first
 * six volumes, with the values they held), out: DEVICE 6 * nx*ny*nz floats.  Synchronous: times
 * `reps` launches with CUDA events after 3 warm-up launches; *gbs = 13 volumes * reps / time in GB/s. */
FDTD_API int fdtd_probe_bandwidth(int32_t pattern, int32_t nx, int32_t ny, int32_t nz, int32_t tile_y, int32_t runs, int32_t unroll,
                         int32_t blocks, int32_t threads, int32_t reps, const float *in, float *out, double *gbs,
                         void *cuda_stream);

/* Library version string, e.g. "fdtd-b200 0.1 sm_100a". */
FDTD_API const char *fdtd_version(void);

/* ------------------------------------------------------------------------------------------
 * Host-buffer entry points: same computation, every array argument (and every pointer inside
 * the descriptors) is HOST memory; the library stages them through device buffers it owns,
 * runs the device path on `cuda_stream`, copies the results back and synchronises the stream
 * before returning.  Used for the end-to-end measurement.
 *   fdtd_forward_host : h_fields in/out (NULL => start from all-zero fields and leave the final
 *                       state on the device inside the grid); phasors are copied in before and
 *                       out after the run.
 *   fdtd_backward_host: h_fields NULL => use the state the last fdtd_forward_host left in the grid;
 *                       otherwise in: state n, out: reconstructed state 0.  h_dL_dphasor is a HOST
 *                       array of HOST pointers.  h_dL_dinv_eps is written; h_dL_dfields0 may be NULL.
 * ------------------------------------------------------------------------------------------ */
FDTD_API int fdtd_forward_host(fdtd_grid *grid, float *h_fields, const float *h_inv_eps, const float *h_inv_mu,
                      const fdtd_source *h_src, int32_t n_src,
                      const fdtd_detector *h_det, int32_t n_det,
                      int32_t n_steps, void *cuda_stream);
FDTD_API int fdtd_backward_host(fdtd_grid *grid, float *h_fields, const float *h_inv_eps, const float *h_inv_mu,
                       const fdtd_source *h_src, int32_t n_src,
                       const fdtd_detector *h_det, int32_t n_det,
                       const float *const *h_dL_dphasor, const float *h_dL_dfields,
                       int32_t n_steps, float *h_dL_dinv_eps, float *h_dL_dfields0,
                       void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* FDTD_B200_H */
