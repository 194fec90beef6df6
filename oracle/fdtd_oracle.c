/*
 * fdtd_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU statement of the hot path of
 * arXiv 2412.12360 ("FDTDX"): Yee-grid FDTD time stepping with CPML, additive
 * sources, DFT detectors, PML-interface recording, and the time-reversed
 * gradient (inverse update + vector-Jacobian product).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may build, load or call this file.  It shares no code,
 * header, table generator or constant with paper_2412_12360_b200/csrc.
 *
 * What the paper fixes:
 *   Eq. 1-2 (L64-66)  dH/dt = -(1/mu) curl E ;  dE/dt = (1/eps) curl H
 *   L68               Yee staggering, "curl updates ... used in every time step"
 *   L72               convolutional PML (Roden-Gedney, ref. 7); sources
 *   L68/L70           detectors, interpolation disabled by default
 *   L80               "chain of function calls, each call updates either the
 *                      electric or magnetic field"
 *   L84               time reversibility; PML not invertible; "field values at
 *                      the boundary between the PML and the inner simulation
 *                      volume ... saved for every time step"
 * Everything below that level (index convention, normalisation, CPML grading,
 * DFT phase stamp, what the recorder stores) is silent in the paper; the
 * readings R1..R30 are listed in DESIGN.md section 3 and followed literally here.
 *
 * Conventions:
 *   grid nx*ny*nz, x fastest: lin = (k*ny + j)*nx + i
 *   fields = [6][nz][ny][nx], components Ex,Ey,Ez,Hx,Hy,Hz
 *   cyclic triple for component c: a = c+1, b = c+2 (mod 3);
 *      (curl F)_c = d_a F_b - d_b F_a
 *   dm_a F[p] = F[p] - F[p - e_a]   (in the E update, acting on H)
 *   dp_a F[p] = F[p + e_a] - F[p]   (in the H update, acting on E)
 *   out-of-range operand: wrapped if periodic, 0 otherwise
 *   one step n: E update (from old H), E sources, H update (from new E),
 *               H sources, detectors with phase omega*(n+1)
 *   S = c dt/dx (Courant number); H is scaled by eta0.
 *
 * Compiled twice: -DREAL=double (parity reference) and -DREAL=float (timed
 * CPU baseline).  No tiling, no fusion, no reordering; OpenMP (optional, only
 * with -fopenmp) splits the outermost k loop of loops whose iterations are
 * independent.
 *
 * Parity pins (tests/test_oracle_pins.py): exact discrete plane-wave
 * eigenmode / dispersion relation, exact discrete energy invariant, discrete
 * Gauss law, forward-N/inverse-N recovery, tape == reversible gradient,
 * gradient vs central finite differences, adjoint dot-product identity,
 * CPML vs big-box, late-time decay, linearity/null tests, the paper's
 * Table 2 step counts (Courant convention); CPML coefficients a, b against
 * the zero-frequency limit and the low-frequency response of ref. 7's
 * stretch factor; the rho chain rule (B6) against a central finite
 * difference of the loss with respect to rho.
 * NEXT rows (tests/test_oracle_pins_n2.py): flux and energy of the exact
 * eigenmode in closed form, detector transposes and flux VJP against finite
 * differences, one-directionality of the TFSF plane source (N2); dL/d inv_mu,
 * the lossy update (closed-form eigenvalue of a plane wave in a conductive
 * box) and one inv_eps per E component (exact eigenmode of a diagonal-
 * anisotropic box) with their gradients against finite differences (N4).
 * Parity unpinned: agreement with the paper's own FDTDX outputs (no numbers,
 * code, geometry or data are available) and the specific CPML constants /
 * DFT normalisation FDTDX uses.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stddef.h>
#if defined(__x86_64__) || defined(__i386__)
#include <xmmintrin.h>
#endif
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef REAL
#define REAL double
#endif

typedef struct {
    int nx, ny, nz;
    int periodic;          /* 1: periodic box (d must be 0); 0: zero outside   */
    int d;                 /* CPML thickness in cells                          */
    double S;              /* Courant number c dt/dx                           */
    double m;              /* grading order of sigma and kappa                 */
    double sigma_max;      /* sigma~_max = sigma eta0 dx at full depth         */
    double kappa_max;
    double alpha_max;      /* alpha~ at the PML/interior interface             */
    double alpha_m;        /* grading order of alpha                           */
} orc_desc;

typedef struct {           /* additive patch F_c[box] += profile*waveform[n]  */
    int comp;              /* 0..5                                             */
    int lo[3], hi[3];      /* half-open box (i,j,k)                            */
    const REAL *profile;   /* box-shaped [k][j][i], or NULL => 1               */
    const REAL *waveform;  /* length >= n_steps                                */
} orc_source;

typedef struct {           /* running DFT on a box                             */
    int mask;              /* bit c set => component c accumulated             */
    int lo[3], hi[3];
    int n_freq;
    const double *omega;   /* rad per step                                     */
    REAL *phasor;          /* [n_freq][n_comp_set][box cells][2] (re,im)       */
} orc_detector;

typedef struct {
    orc_desc D;
    size_t nc;                               /* cells                          */
    REAL *bE[3], *aE[3], *ikE[3];            /* CPML tables, E positions x = p    */
    REAL *bH[3], *aH[3], *ikH[3];            /* CPML tables, H positions x = p+1/2 */
    REAL *psiE[3][2], *psiH[3][2];           /* primal psi, full volumes       */
    REAL *lpsiE[3][2], *lpsiH[3][2];         /* cotangents of psi              */
    REAL *tmp[3][2];                         /* scratch volumes for the adjoint */
    const REAL *sigma;                       /* N4: normalised electric conductivity per voxel, or NULL (lossless) */
    int aniso;                               /* N4: 1 = inv_eps (and its gradient) are three volumes, one per E component */
} orc_state;

/* N4 (SURVEY 8(f) N4 "per-component inv_eps (3 volumes / sub-pixel averaging)"), reading R30: with aniso set, inv_eps is      */
/* [3][cells] and E_c is updated with inv_eps[c] at its own (staggered) position -- what sub-pixel smoothing of an interface     */
/* produces -- instead of the one value per voxel of reading R6; the gradient is then [3][cells] as well.                        */
#define IEC(c, p) ie[(st->aniso ? (size_t)(c) * nc : 0) + (p)]

#define NX (D->nx)
#define NY (D->ny)
#define NZ (D->nz)
#define IDX(i, j, k) (((size_t)(k) * NY + (j)) * NX + (i))

/* ------------------------------------------------------------------------ */
/* helpers                                                                  */
/* ------------------------------------------------------------------------ */

/* value of volume F at (i,j,k); out of range: wrapped if periodic, else 0 (R7) */
static inline REAL at(const orc_desc *D, const REAL *F, int i, int j, int k)
{
    if (D->periodic) {
        i = (i % NX + NX) % NX;
        j = (j % NY + NY) % NY;
        k = (k % NZ + NZ) % NZ;
    } else if (i < 0 || i >= NX || j < 0 || j >= NY || k < 0 || k >= NZ) {
        return (REAL)0;
    }
    return F[IDX(i, j, k)];
}

static inline int dimlen(const orc_desc *D, int axis)
{
    return axis == 0 ? NX : (axis == 1 ? NY : NZ);
}

/* interior box I = [d, N_a - d) on every axis (whole grid if d == 0) */
static inline int lo_I(const orc_desc *D, int axis) { (void)axis; return D->d; }
static inline int hi_I(const orc_desc *D, int axis) { return dimlen(D, axis) - D->d; }

void orc_set_ftz(int on)
{
#if defined(__x86_64__) || defined(__i386__)
#ifdef _OPENMP
#pragma omp parallel
#endif
    {
        unsigned csr = _mm_getcsr();
        if (on) csr |= 0x8040u; else csr &= ~0x8040u;   /* FTZ | DAZ */
        _mm_setcsr(csr);
    }
#else
    (void)on;
#endif
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* threads the OpenMP loops use from now on (bench.py times the oracle with all cores and with 1 thread) */
void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_sizeof_real(void) { return (int)sizeof(REAL); }

/* ------------------------------------------------------------------------ */
/* CPML tables (PAPER.md L72 -> ref. 7; constants: DESIGN.md R8)            */
/*   depth rho(x) = max(0, d - x, x - (N - d)),  r = rho/d                  */
/*   sigma = sigma_max r^m ; kappa = 1 + (kappa_max-1) r^m ;                */
/*   alpha = alpha_max (1-r)^alpha_m  (inside the PML, 0 outside)           */
/*   b = exp(-(sigma/kappa + alpha) S)                                      */
/*   a = sigma / (kappa (sigma + kappa alpha)) (b - 1)   (0 where sigma=0)  */
/*   ik = 1/kappa                                                           */
/* half = 0: E tables at x = p ; half = 1: H tables at x = p + 1/2          */
/* ------------------------------------------------------------------------ */
void orc_cpml_table(const orc_desc *D, int axis, int half,
                    double *b, double *a, double *ik)
{
    int n = dimlen(D, axis);
    for (int p = 0; p < n; ++p) {
        double x = (double)p + (half ? 0.5 : 0.0);
        double rho = 0.0;
        if (D->d > 0) {
            double r1 = (double)D->d - x;
            double r2 = x - (double)(n - D->d);
            if (r1 > rho) rho = r1;
            if (r2 > rho) rho = r2;
        }
        if (rho <= 0.0) { b[p] = 1.0; a[p] = 0.0; ik[p] = 1.0; continue; }
        double r = rho / (double)D->d;
        double sig = D->sigma_max * pow(r, D->m);
        double kap = 1.0 + (D->kappa_max - 1.0) * pow(r, D->m);
        double alp = D->alpha_max * pow(1.0 - r, D->alpha_m);
        double bb = exp(-(sig / kap + alp) * D->S);
        double aa = 0.0;
        if (sig > 0.0) aa = sig / (kap * (sig + kap * alp)) * (bb - 1.0);
        b[p] = bb; a[p] = aa; ik[p] = 1.0 / kap;
    }
}

/* ------------------------------------------------------------------------ */
/* state                                                                    */
/* ------------------------------------------------------------------------ */
static REAL *zalloc(size_t n) { return (REAL *)calloc(n ? n : 1, sizeof(REAL)); }

void orc_destroy(orc_state *st)
{
    if (!st) return;
    for (int a = 0; a < 3; ++a) {
        free(st->bE[a]); free(st->aE[a]); free(st->ikE[a]);
        free(st->bH[a]); free(st->aH[a]); free(st->ikH[a]);
        for (int s = 0; s < 2; ++s) {
            free(st->psiE[a][s]); free(st->psiH[a][s]);
            free(st->lpsiE[a][s]); free(st->lpsiH[a][s]);
            free(st->tmp[a][s]);
        }
    }
    free(st);
}

orc_state *orc_create(const orc_desc *desc)
{
    if (desc->nx < 1 || desc->ny < 1 || desc->nz < 1) return NULL;
    if (desc->periodic && desc->d != 0) return NULL;
    if (desc->d < 0) return NULL;
    orc_state *st = (orc_state *)calloc(1, sizeof(orc_state));
    if (!st) return NULL;
    st->D = *desc;
    const orc_desc *D = &st->D;
    st->nc = (size_t)NX * NY * NZ;
    for (int a = 0; a < 3; ++a) {
        int n = dimlen(D, a);
        double *b = (double *)malloc(sizeof(double) * n);
        double *aa = (double *)malloc(sizeof(double) * n);
        double *ik = (double *)malloc(sizeof(double) * n);
        for (int half = 0; half < 2; ++half) {
            orc_cpml_table(D, a, half, b, aa, ik);
            REAL *tb = zalloc(n), *ta = zalloc(n), *tk = zalloc(n);
            for (int p = 0; p < n; ++p) { tb[p] = (REAL)b[p]; ta[p] = (REAL)aa[p]; tk[p] = (REAL)ik[p]; }
            if (half == 0) { st->bE[a] = tb; st->aE[a] = ta; st->ikE[a] = tk; }
            else           { st->bH[a] = tb; st->aH[a] = ta; st->ikH[a] = tk; }
        }
        free(b); free(aa); free(ik);
        for (int s = 0; s < 2; ++s) {
            st->psiE[a][s] = zalloc(st->nc);  st->psiH[a][s] = zalloc(st->nc);
            st->lpsiE[a][s] = zalloc(st->nc); st->lpsiH[a][s] = zalloc(st->nc);
            st->tmp[a][s] = zalloc(st->nc);
        }
    }
    return st;
}

/* accessors so tests can read / set psi and its cotangent */
REAL *orc_psi(orc_state *st, int is_H, int c, int s)  { return is_H ? st->psiH[c][s] : st->psiE[c][s]; }
REAL *orc_lpsi(orc_state *st, int is_H, int c, int s) { return is_H ? st->lpsiH[c][s] : st->lpsiE[c][s]; }

void orc_zero_psi(orc_state *st)
{
    for (int c = 0; c < 3; ++c) for (int s = 0; s < 2; ++s) {
        memset(st->psiE[c][s], 0, st->nc * sizeof(REAL));
        memset(st->psiH[c][s], 0, st->nc * sizeof(REAL));
    }
}
void orc_zero_lpsi(orc_state *st)
{
    for (int c = 0; c < 3; ++c) for (int s = 0; s < 2; ++s) {
        memset(st->lpsiE[c][s], 0, st->nc * sizeof(REAL));
        memset(st->lpsiH[c][s], 0, st->nc * sizeof(REAL));
    }
}

/* ------------------------------------------------------------------------ */
/* N4 (SURVEY 8(f) N4 "conductive ... media where time reversal fails"; "reversible ... for lossless  */
/* materials", L82 checkpointing as the alternative).  Reading R29: an electric conductivity sigma per voxel,        */
/* normalised like the CPML's (sigma~ = sigma eta0 dx), enters Eq. 2 as  eps dE/dt = curl H - sigma E  and is         */
/* discretised semi-implicitly (sigma E at the half step = sigma (E' + E)/2), the standard lossy Yee update:          */
/*   beta = sigma~ S ie / 2,  Ca = (1 - beta)/(1 + beta),  Cb = 1/(1 + beta),   E'_c = Ca E_c + Cb S ie bracket_c     */
/* (the same ie and sigma~ for the three components stored at the voxel, like R6).  sigma = NULL: Ca = Cb = 1.        */
/* The inverse step is not defined for it (orc_backward refuses); gradients come from tape mode.                      */
/* ------------------------------------------------------------------------ */
void orc_set_sigma(orc_state *st, const REAL *sigma) { st->sigma = sigma; }
void orc_set_aniso(orc_state *st, int aniso) { st->aniso = aniso ? 1 : 0; }

/* ------------------------------------------------------------------------ */
/* O1: E update (Eq. 2 discretised on the Yee grid; CPML psi_E recursion)   */
/*   d1 = dm_a H_b, d2 = dm_b H_a                                           */
/*   psiE_c0 = bE_a psiE_c0 + aE_a d1 ; psiE_c1 = bE_b psiE_c1 + aE_b d2    */
/*   E_c += S ie (ikE_a d1 - ikE_b d2 + psiE_c0 - psiE_c1)                  */
/* bracket (optional, [3][cells]) receives the bracketed term: dE_c/d(ie)=S*bracket */
/* ------------------------------------------------------------------------ */
void orc_step_E(orc_state *st, REAL *fields, const REAL *ie, REAL *bracket)
{
    const orc_desc *D = &st->D;
    const REAL S = (REAL)D->S;
    const size_t nc = st->nc;
    REAL *E[3] = { fields, fields + nc, fields + 2 * nc };
    const REAL *H[3] = { fields + 3 * nc, fields + 4 * nc, fields + 5 * nc };
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = 0; k < NZ; ++k)
        for (int j = 0; j < NY; ++j)
            for (int i = 0; i < NX; ++i) {
                const size_t p = IDX(i, j, k);
                const int pos[3] = { i, j, k };
                for (int c = 0; c < 3; ++c) {
                    const int a = (c + 1) % 3, b = (c + 2) % 3;
                    int ea[3] = { 0, 0, 0 }, eb[3] = { 0, 0, 0 };
                    ea[a] = 1; eb[b] = 1;
                    REAL d1 = H[b][p] - at(D, H[b], i - ea[0], j - ea[1], k - ea[2]);
                    REAL d2 = H[a][p] - at(D, H[a], i - eb[0], j - eb[1], k - eb[2]);
                    REAL p0 = st->bE[a][pos[a]] * st->psiE[c][0][p] + st->aE[a][pos[a]] * d1;
                    REAL p1 = st->bE[b][pos[b]] * st->psiE[c][1][p] + st->aE[b][pos[b]] * d2;
                    st->psiE[c][0][p] = p0;
                    st->psiE[c][1][p] = p1;
                    REAL br = st->ikE[a][pos[a]] * d1 - st->ikE[b][pos[b]] * d2 + p0 - p1;
                    if (!st->sigma) {
                        if (bracket) bracket[(size_t)c * nc + p] = br;
                        E[c][p] += S * IEC(c, p) * br;
                    } else {
                        /* lossy update; `bracket` keeps its meaning dE'_c/d(ie) = S * bracket:                      */
                        /*   dCa/d ie = -sigma S / (1+beta)^2,  dCb/d ie = -(sigma S / 2) / (1+beta)^2               */
                        const REAL hs = (REAL)0.5 * st->sigma[p] * S, beta = hs * IEC(c, p);
                        const REAL Ca = ((REAL)1 - beta) / ((REAL)1 + beta), Cb = (REAL)1 / ((REAL)1 + beta);
                        const REAL dCa = (REAL)-2 * hs * Cb * Cb, dCb = -hs * Cb * Cb;
                        if (bracket) bracket[(size_t)c * nc + p] = (dCa * E[c][p] + (dCb * IEC(c, p) + Cb) * S * br) / S;
                        E[c][p] = Ca * E[c][p] + Cb * S * IEC(c, p) * br;
                    }
                }
            }
}

/* ------------------------------------------------------------------------ */
/* O3: H update (Eq. 1 discretised; note the minus sign)                    */
/*   d1 = dp_a E_b, d2 = dp_b E_a  on the just-updated E                    */
/*   H_c -= S im (ikH_a d1 - ikH_b d2 + psiH_c0 - psiH_c1)                  */
/* im == NULL means inv_mu = 1                                              */
/* ------------------------------------------------------------------------ */
void orc_step_H(orc_state *st, REAL *fields, const REAL *im)
{
    const orc_desc *D = &st->D;
    const REAL S = (REAL)D->S;
    const size_t nc = st->nc;
    const REAL *E[3] = { fields, fields + nc, fields + 2 * nc };
    REAL *H[3] = { fields + 3 * nc, fields + 4 * nc, fields + 5 * nc };
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = 0; k < NZ; ++k)
        for (int j = 0; j < NY; ++j)
            for (int i = 0; i < NX; ++i) {
                const size_t p = IDX(i, j, k);
                const int pos[3] = { i, j, k };
                for (int c = 0; c < 3; ++c) {
                    const int a = (c + 1) % 3, b = (c + 2) % 3;
                    int ea[3] = { 0, 0, 0 }, eb[3] = { 0, 0, 0 };
                    ea[a] = 1; eb[b] = 1;
                    REAL d1 = at(D, E[b], i + ea[0], j + ea[1], k + ea[2]) - E[b][p];
                    REAL d2 = at(D, E[a], i + eb[0], j + eb[1], k + eb[2]) - E[a][p];
                    REAL p0 = st->bH[a][pos[a]] * st->psiH[c][0][p] + st->aH[a][pos[a]] * d1;
                    REAL p1 = st->bH[b][pos[b]] * st->psiH[c][1][p] + st->aH[b][pos[b]] * d2;
                    st->psiH[c][0][p] = p0;
                    st->psiH[c][1][p] = p1;
                    REAL br = st->ikH[a][pos[a]] * d1 - st->ikH[b][pos[b]] * d2 + p0 - p1;
                    H[c][p] -= S * (im ? im[p] : (REAL)1) * br;
                }
            }
}

/* ------------------------------------------------------------------------ */
/* O2 / O4: additive sources of one field family (E: comp 0..2, H: 3..5)    */
/* sign = +1 in the forward step, -1 in the inverse step                    */
/* ------------------------------------------------------------------------ */
static void add_sources(const orc_desc *D, REAL *fields, size_t nc,
                        const orc_source *src, int n_src, int n, int family_H, REAL sign)
{
    for (int s = 0; s < n_src; ++s) {
        const orc_source *q = &src[s];
        if ((q->comp >= 3) != (family_H != 0)) continue;
        REAL *F = fields + (size_t)q->comp * nc;
        const REAL w = q->waveform[n];
        const int bx = q->hi[0] - q->lo[0], by = q->hi[1] - q->lo[1];
        for (int k = q->lo[2]; k < q->hi[2]; ++k)
            for (int j = q->lo[1]; j < q->hi[1]; ++j)
                for (int i = q->lo[0]; i < q->hi[0]; ++i) {
                    size_t c = ((size_t)(k - q->lo[2]) * by + (j - q->lo[1])) * bx + (i - q->lo[0]);
                    REAL prof = q->profile ? q->profile[c] : (REAL)1;
                    F[IDX(i, j, k)] += sign * prof * w;
                }
    }
}

static int popcount6(int m) { int n = 0; for (int c = 0; c < 6; ++c) n += (m >> c) & 1; return n; }

/* O5: detectors  P_f[c][cell] += F_c[cell] (cos phi - i sin phi), phi = omega_f (n+1)  (R13) */
static void detect(const orc_desc *D, const REAL *fields, size_t nc,
                   const orc_detector *det, int n_det, int n)
{
    for (int s = 0; s < n_det; ++s) {
        const orc_detector *q = &det[s];
        const int bx = q->hi[0] - q->lo[0], by = q->hi[1] - q->lo[1], bz = q->hi[2] - q->lo[2];
        const size_t bc = (size_t)bx * by * bz;
        const int ncomp = popcount6(q->mask);
        for (int f = 0; f < q->n_freq; ++f) {
            const double phi = q->omega[f] * (double)(n + 1);
            const REAL cs = (REAL)cos(phi), sn = (REAL)sin(phi);
            int ci = 0;
            for (int c = 0; c < 6; ++c) {
                if (!((q->mask >> c) & 1)) continue;
                const REAL *F = fields + (size_t)c * nc;
                REAL *P = q->phasor + ((size_t)f * ncomp + ci) * bc * 2;
                for (int k = q->lo[2]; k < q->hi[2]; ++k)
                    for (int j = q->lo[1]; j < q->hi[1]; ++j)
                        for (int i = q->lo[0]; i < q->hi[0]; ++i) {
                            size_t cell = ((size_t)(k - q->lo[2]) * by + (j - q->lo[1])) * bx + (i - q->lo[0]);
                            REAL v = F[IDX(i, j, k)];
                            P[2 * cell]     += v * cs;
                            P[2 * cell + 1] -= v * sn;
                        }
                ++ci;
            }
        }
    }
}

/* B1: transpose of detect():  lam F_c[cell] += Gr cos phi - Gi sin phi */
static void detect_adjoint(const orc_desc *D, REAL *lam, size_t nc,
                           const orc_detector *det, int n_det,
                           const REAL *const *dL_dphasor, int n)
{
    if (!dL_dphasor) return;
    for (int s = 0; s < n_det; ++s) {
        const orc_detector *q = &det[s];
        const REAL *G = dL_dphasor[s];
        if (!G) continue;
        const int bx = q->hi[0] - q->lo[0], by = q->hi[1] - q->lo[1], bz = q->hi[2] - q->lo[2];
        const size_t bc = (size_t)bx * by * bz;
        const int ncomp = popcount6(q->mask);
        for (int f = 0; f < q->n_freq; ++f) {
            const double phi = q->omega[f] * (double)(n + 1);
            const REAL cs = (REAL)cos(phi), sn = (REAL)sin(phi);
            int ci = 0;
            for (int c = 0; c < 6; ++c) {
                if (!((q->mask >> c) & 1)) continue;
                REAL *L = lam + (size_t)c * nc;
                const REAL *Gp = G + ((size_t)f * ncomp + ci) * bc * 2;
                for (int k = q->lo[2]; k < q->hi[2]; ++k)
                    for (int j = q->lo[1]; j < q->hi[1]; ++j)
                        for (int i = q->lo[0]; i < q->hi[0]; ++i) {
                            size_t cell = ((size_t)(k - q->lo[2]) * by + (j - q->lo[1])) * bx + (i - q->lo[0]);
                            L[IDX(i, j, k)] += Gp[2 * cell] * cs - Gp[2 * cell + 1] * sn;
                        }
                ++ci;
            }
        }
    }
}

/* ------------------------------------------------------------------------ */
/* Recorder (reading R15): per step, for each axis a,          */
/*   low face : H_b, H_c (b=a+1, c=a+2) at index d-1 on axis a, BEFORE step n */
/*   high face: E'_b, E'_c at index N_a-d on axis a, after O1/O2 of step n   */
/* the two other indices run over I.  Layout of one step's record:          */
/*   for a in 0..2: [low: comp b cells, comp c cells][high: comp b, comp c] */
/* with face cells ordered (slower other axis, faster other axis).          */
/* ------------------------------------------------------------------------ */
static size_t face_cells(const orc_desc *D, int a)
{
    int u = (a + 1) % 3, v = (a + 2) % 3;
    if (D->d == 0) return 0;
    return (size_t)(hi_I(D, u) - lo_I(D, u)) * (size_t)(hi_I(D, v) - lo_I(D, v));
}

size_t orc_record_stride(const orc_desc *D)
{
    size_t n = 0;
    for (int a = 0; a < 3; ++a) n += 4 * face_cells(D, a);
    return n;
}

/* offset (in REALs) inside one step's record of (axis a, side 0=low/1=high, which 0/1) */
static size_t rec_offset(const orc_desc *D, int a, int side, int which)
{
    size_t off = 0;
    for (int q = 0; q < a; ++q) off += 4 * face_cells(D, q);
    return off + (size_t)(2 * side + which) * face_cells(D, a);
}

/* index of a face cell; pos[] is the full (i,j,k); axis a is ignored.
   face cells are ordered with the higher-numbered of the two other axes slowest */
static size_t face_index(const orc_desc *D, int a, const int pos[3])
{
    int u = (a + 1) % 3, v = (a + 2) % 3;
    if (u > v) { int t = u; u = v; v = t; }          /* u < v : v slowest */
    return (size_t)(pos[v] - lo_I(D, v)) * (size_t)(hi_I(D, u) - lo_I(D, u)) + (size_t)(pos[u] - lo_I(D, u));
}

static void record_faces(const orc_desc *D, const REAL *fields, size_t nc, REAL *rec, int side)
{
    if (D->d == 0) return;
    for (int a = 0; a < 3; ++a) {
        const int fixed = side ? hi_I(D, a) : lo_I(D, a) - 1;
        for (int which = 0; which < 2; ++which) {
            const int comp = (a + 1 + which) % 3;                 /* tangential component */
            const REAL *F = fields + (size_t)(side ? comp : 3 + comp) * nc;   /* E' high, H low */
            REAL *out = rec + rec_offset(D, a, side, which);
            int pos[3];
            for (pos[2] = (a == 2 ? fixed : lo_I(D, 2)); pos[2] < (a == 2 ? fixed + 1 : hi_I(D, 2)); ++pos[2])
                for (pos[1] = (a == 1 ? fixed : lo_I(D, 1)); pos[1] < (a == 1 ? fixed + 1 : hi_I(D, 1)); ++pos[1])
                    for (pos[0] = (a == 0 ? fixed : lo_I(D, 0)); pos[0] < (a == 0 ? fixed + 1 : hi_I(D, 0)); ++pos[0])
                        out[face_index(D, a, pos)] = F[IDX(pos[0], pos[1], pos[2])];
        }
    }
}

/* ------------------------------------------------------------------------ */
/* N2 ("access to intermediate fields, energy,     */
/* Poynting flux", L70 interpolation off by default): time-domain detectors. */
/* Reading R23: a time-domain detector fires after step n when               */
/* (n+1) % stride == 0, record index q = (n+1)/stride - 1, on the state      */
/* (E^{n+1}, H^{n+3/2}) -- the same time stamp as the DFT detectors (R13):   */
/*   kind 0 SNAPSHOT: out[q][ci][cell] = F_c[cell] for every c in mask       */
/*   kind 1 ENERGY  : out[q] = sum_cells 1/2 (sum_c E_c^2/ie + H_c^2/im)     */
/*                    (eta0-normalised H, energy in units of eps0 dx^3; the   */
/*                    six components are taken at the same index, no          */
/*                    co-location, as the paper's default)                    */
/* ------------------------------------------------------------------------ */
typedef struct {
    int kind;              /* 0 snapshot, 1 energy                             */
    int mask;              /* snapshot: components; energy: ignored            */
    int lo[3], hi[3];
    int stride;            /* >= 1                                             */
    REAL *out;             /* snapshot [n_rec][n_comp][cells]; energy [n_rec]  */
} orc_tdetector;

static void time_detect(const orc_desc *D, const REAL *fields, size_t nc, const REAL *ie, const REAL *im,
                        const orc_tdetector *td, int n_td, int n)
{
    for (int s = 0; s < n_td; ++s) {
        const orc_tdetector *q = &td[s];
        if ((n + 1) % q->stride != 0) continue;
        const size_t rec_i = (size_t)((n + 1) / q->stride - 1);
        const int bx = q->hi[0] - q->lo[0], by = q->hi[1] - q->lo[1], bz = q->hi[2] - q->lo[2];
        const size_t bc = (size_t)bx * by * bz;
        if (q->kind == 0) {
            const int ncomp = popcount6(q->mask);
            int ci = 0;
            for (int c = 0; c < 6; ++c) {
                if (!((q->mask >> c) & 1)) continue;
                REAL *out = q->out + (rec_i * ncomp + ci) * bc;
                for (int k = q->lo[2]; k < q->hi[2]; ++k)
                    for (int j = q->lo[1]; j < q->hi[1]; ++j)
                        for (int i = q->lo[0]; i < q->hi[0]; ++i)
                            out[((size_t)(k - q->lo[2]) * by + (j - q->lo[1])) * bx + (i - q->lo[0])] = fields[(size_t)c * nc + IDX(i, j, k)];
                ++ci;
            }
        } else {
            double acc = 0.0;
            for (int k = q->lo[2]; k < q->hi[2]; ++k)
                for (int j = q->lo[1]; j < q->hi[1]; ++j)
                    for (int i = q->lo[0]; i < q->hi[0]; ++i) {
                        const size_t p = IDX(i, j, k);
                        double e2 = 0.0, h2 = 0.0;
                        for (int c = 0; c < 3; ++c) {
                            e2 += (double)fields[(size_t)c * nc + p] * fields[(size_t)c * nc + p];
                            h2 += (double)fields[(size_t)(3 + c) * nc + p] * fields[(size_t)(3 + c) * nc + p];
                        }
                        acc += 0.5 * (e2 / (double)ie[p] + h2 / (im ? (double)im[p] : 1.0));
                    }
            q->out[rec_i] = (REAL)acc;
        }
    }
}

/* transpose of time_detect at reverse step n, with G = dL/d out:                               */
/*   snapshot: lam F_c[cell] += G[q][ci][cell]                                                  */
/*   energy  : lam E_c += G[q] E_c/ie ; lam H_c += G[q] H_c/im  (primal state after step n: the  */
/*             detector box must lie inside the reconstruction box I), and the explicit          */
/*             dependence on ie:  g[cell] += G[q] * (-1/2) sum_c E_c^2 / ie^2                     */
static void time_detect_adjoint(const orc_desc *D, REAL *lam, const REAL *fields, size_t nc, const REAL *ie, const REAL *im,
                                const orc_tdetector *td, int n_td, const REAL *const *dL_dout, REAL *g, int n)
{
    if (!dL_dout) return;
    for (int s = 0; s < n_td; ++s) {
        const orc_tdetector *q = &td[s];
        const REAL *G = dL_dout[s];
        if (!G || (n + 1) % q->stride != 0) continue;
        const size_t rec_i = (size_t)((n + 1) / q->stride - 1);
        const int bx = q->hi[0] - q->lo[0], by = q->hi[1] - q->lo[1], bz = q->hi[2] - q->lo[2];
        const size_t bc = (size_t)bx * by * bz;
        if (q->kind == 0) {
            const int ncomp = popcount6(q->mask);
            int ci = 0;
            for (int c = 0; c < 6; ++c) {
                if (!((q->mask >> c) & 1)) continue;
                const REAL *Gp = G + (rec_i * ncomp + ci) * bc;
                for (int k = q->lo[2]; k < q->hi[2]; ++k)
                    for (int j = q->lo[1]; j < q->hi[1]; ++j)
                        for (int i = q->lo[0]; i < q->hi[0]; ++i)
                            lam[(size_t)c * nc + IDX(i, j, k)] += Gp[((size_t)(k - q->lo[2]) * by + (j - q->lo[1])) * bx + (i - q->lo[0])];
                ++ci;
            }
        } else {
            const REAL Gq = G[rec_i];
            for (int k = q->lo[2]; k < q->hi[2]; ++k)
                for (int j = q->lo[1]; j < q->hi[1]; ++j)
                    for (int i = q->lo[0]; i < q->hi[0]; ++i) {
                        const size_t p = IDX(i, j, k);
                        REAL e2 = (REAL)0;
                        for (int c = 0; c < 3; ++c) {
                            const REAL E = fields[(size_t)c * nc + p], H = fields[(size_t)(3 + c) * nc + p];
                            lam[(size_t)c * nc + p] += Gq * E / ie[p];
                            lam[(size_t)(3 + c) * nc + p] += Gq * H / (im ? im[p] : (REAL)1);
                            e2 += E * E;
                        }
                        if (g) g[p] += Gq * (REAL)(-0.5) * e2 / (ie[p] * ie[p]);
                    }
        }
    }
}

/* ------------------------------------------------------------------------ */
/* forward driver: n_steps of  [O0r] O1 O2 [O2r] O3 O4 O5 [time detectors]  */
/* rec   : NULL or n_steps * orc_record_stride() REALs                      */
/* tape  : NULL or n_steps * 3 * cells REALs (bracket of every E update)    */
/* psi is NOT reset here (callers use orc_zero_psi; R21)                    */
/* ------------------------------------------------------------------------ */
int orc_forward_td(orc_state *st, REAL *fields, const REAL *ie, const REAL *im,
                   const orc_source *src, int n_src, const orc_detector *det, int n_det,
                   const orc_tdetector *td, int n_td,
                   int n_steps, REAL *rec, REAL *tape)
{
    const orc_desc *D = &st->D;
    const size_t nc = st->nc;
    const size_t rs = orc_record_stride(D);
    for (int s = 0; s < n_td; ++s) if (st->aniso && td[s].kind == 1) return -1;    /* the energy detector is stated for one inv_eps per voxel */
    for (int n = 0; n < n_steps; ++n) {
        if (rec) record_faces(D, fields, nc, rec + (size_t)n * rs, 0);           /* O0r */
        orc_step_E(st, fields, ie, tape ? tape + (size_t)n * 3 * nc : NULL);     /* O1  */
        add_sources(D, fields, nc, src, n_src, n, 0, (REAL)1);                   /* O2  */
        if (rec) record_faces(D, fields, nc, rec + (size_t)n * rs, 1);           /* O2r */
        orc_step_H(st, fields, im);                                              /* O3  */
        add_sources(D, fields, nc, src, n_src, n, 1, (REAL)1);                   /* O4  */
        detect(D, fields, nc, det, n_det, n);                                    /* O5  */
        time_detect(D, fields, nc, ie, im, td, n_td, n);                         /* N2  */
    }
    return 0;
}

int orc_forward(orc_state *st, REAL *fields, const REAL *ie, const REAL *im,
                const orc_source *src, int n_src, const orc_detector *det, int n_det,
                int n_steps, REAL *rec, REAL *tape)
{
    return orc_forward_td(st, fields, ie, im, src, n_src, det, n_det, NULL, 0, n_steps, rec, tape);
}

/* ------------------------------------------------------------------------ */
/* B2: adjoint of O3 (H update incl. psi_H recursion), whole grid.          */
/* Reverse-mode of                                                          */
/*   p0' = bH_a p0 + aH_a d1 ; p1' = bH_b p1 + aH_b d2                       */
/*   H_c' = H_c - S im (ikH_a d1 - ikH_b d2 + p0' - p1')                     */
/*   d1 = dp_a E_b ; d2 = dp_b E_a                                          */
/* with w = -S im lamH_c:  lp0 += w ; lp1 -= w ;                            */
/*   g1 = ikH_a w + aH_a lp0 ; g2 = -ikH_b w + aH_b lp1 ;                   */
/*   lp0 <- bH_a lp0 ; lp1 <- bH_b lp1 ;                                    */
/*   lamE_b += (dp_a)^T g1 = -dm_a g1 ; lamE_a += (dp_b)^T g2 = -dm_b g2    */
/* lamH passes through unchanged.  Two passes (compute g, then difference)  */
/* so that no loop iteration writes another iteration's cells.              */
/* ------------------------------------------------------------------------ */
void orc_adj_H(orc_state *st, REAL *lam, const REAL *im)
{
    const orc_desc *D = &st->D;
    const REAL S = (REAL)D->S;
    const size_t nc = st->nc;
    REAL *lE[3] = { lam, lam + nc, lam + 2 * nc };
    const REAL *lH[3] = { lam + 3 * nc, lam + 4 * nc, lam + 5 * nc };
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = 0; k < NZ; ++k)
        for (int j = 0; j < NY; ++j)
            for (int i = 0; i < NX; ++i) {
                const size_t p = IDX(i, j, k);
                const int pos[3] = { i, j, k };
                for (int c = 0; c < 3; ++c) {
                    const int a = (c + 1) % 3, b = (c + 2) % 3;
                    REAL w = -S * (im ? im[p] : (REAL)1) * lH[c][p];
                    REAL l0 = st->lpsiH[c][0][p] + w;
                    REAL l1 = st->lpsiH[c][1][p] - w;
                    st->tmp[c][0][p] = st->ikH[a][pos[a]] * w + st->aH[a][pos[a]] * l0;    /* g1 */
                    st->tmp[c][1][p] = -st->ikH[b][pos[b]] * w + st->aH[b][pos[b]] * l1;   /* g2 */
                    st->lpsiH[c][0][p] = st->bH[a][pos[a]] * l0;
                    st->lpsiH[c][1][p] = st->bH[b][pos[b]] * l1;
                }
            }
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = 0; k < NZ; ++k)
        for (int j = 0; j < NY; ++j)
            for (int i = 0; i < NX; ++i) {
                const size_t p = IDX(i, j, k);
                for (int c = 0; c < 3; ++c) {
                    const int a = (c + 1) % 3, b = (c + 2) % 3;
                    int ea[3] = { 0, 0, 0 }, eb[3] = { 0, 0, 0 };
                    ea[a] = 1; eb[b] = 1;
                    /* component c's g1 feeds lamE_b, its g2 feeds lamE_a */
                    lE[b][p] -= st->tmp[c][0][p] - at(D, st->tmp[c][0], i - ea[0], j - ea[1], k - ea[2]);
                    lE[a][p] -= st->tmp[c][1][p] - at(D, st->tmp[c][1], i - eb[0], j - eb[1], k - eb[2]);
                }
            }
}

/* ------------------------------------------------------------------------ */
/* B5: adjoint of O1 (E update incl. psi_E recursion), whole grid.          */
/*   with w = +S ie lamE_c: same pattern, E tables;                         */
/*   lamH_b += (dm_a)^T g1 = -dp_a g1 ; lamH_a += (dm_b)^T g2 = -dp_b g2    */
/* ------------------------------------------------------------------------ */
void orc_adj_E(orc_state *st, REAL *lam, const REAL *ie)
{
    const orc_desc *D = &st->D;
    const REAL S = (REAL)D->S;
    const size_t nc = st->nc;
    REAL *lE[3] = { lam, lam + nc, lam + 2 * nc };
    REAL *lH[3] = { lam + 3 * nc, lam + 4 * nc, lam + 5 * nc };
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = 0; k < NZ; ++k)
        for (int j = 0; j < NY; ++j)
            for (int i = 0; i < NX; ++i) {
                const size_t p = IDX(i, j, k);
                const int pos[3] = { i, j, k };
                /* N4, lossy update E' = Ca E + Cb S ie bracket: the bracket's cotangent is Cb S ie lamE', and E's is Ca lamE' */
                for (int c = 0; c < 3; ++c) {
                    const int a = (c + 1) % 3, b = (c + 2) % 3;
                    const REAL beta = st->sigma ? (REAL)0.5 * st->sigma[p] * S * IEC(c, p) : (REAL)0;
                    const REAL Ca = ((REAL)1 - beta) / ((REAL)1 + beta), Cb = (REAL)1 / ((REAL)1 + beta);
                    REAL w = (st->sigma ? Cb : (REAL)1) * S * IEC(c, p) * lE[c][p];
                    if (st->sigma) lE[c][p] *= Ca;
                    REAL l0 = st->lpsiE[c][0][p] + w;
                    REAL l1 = st->lpsiE[c][1][p] - w;
                    st->tmp[c][0][p] = st->ikE[a][pos[a]] * w + st->aE[a][pos[a]] * l0;
                    st->tmp[c][1][p] = -st->ikE[b][pos[b]] * w + st->aE[b][pos[b]] * l1;
                    st->lpsiE[c][0][p] = st->bE[a][pos[a]] * l0;
                    st->lpsiE[c][1][p] = st->bE[b][pos[b]] * l1;
                }
            }
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = 0; k < NZ; ++k)
        for (int j = 0; j < NY; ++j)
            for (int i = 0; i < NX; ++i) {
                const size_t p = IDX(i, j, k);
                for (int c = 0; c < 3; ++c) {
                    const int a = (c + 1) % 3, b = (c + 2) % 3;
                    int ea[3] = { 0, 0, 0 }, eb[3] = { 0, 0, 0 };
                    ea[a] = 1; eb[b] = 1;
                    lH[b][p] -= at(D, st->tmp[c][0], i + ea[0], j + ea[1], k + ea[2]) - st->tmp[c][0][p];
                    lH[a][p] -= at(D, st->tmp[c][1], i + eb[0], j + eb[1], k + eb[2]) - st->tmp[c][1][p];
                }
            }
}

/* ------------------------------------------------------------------------ */
/* O6c: inverse H step on the interior box I ("the inverse     */
/* function of the FDTD update"):  H = H' + S im curl+ E'                    */
/* An E' operand one cell outside I on the high side (index N_a - d) is not  */
/* read from the volume but from this step's record (rec_n); on a periodic   */
/* grid I is the whole box and operands wrap.  H sources are subtracted by   */
/* the caller before this function.                                          */
/* ------------------------------------------------------------------------ */
static REAL E_plus(const orc_desc *D, const REAL *const E[3], const REAL *rec_n,
                   int comp, int axis, int i, int j, int k)
{
    int pos[3] = { i, j, k };
    pos[axis] += 1;
    if (D->d > 0 && pos[axis] == hi_I(D, axis)) {
        int which = (comp - axis - 1 + 3) % 3;               /* 0: comp = axis+1, 1: comp = axis+2 */
        return rec_n[rec_offset(D, axis, 1, which) + face_index(D, axis, pos)];
    }
    return at(D, E[comp], pos[0], pos[1], pos[2]);
}

/* N4 ("dL/d inv_mu"; Eq. 1): the H update H'_c = H_c - S im C_c(E') depends on im   */
/* at its own cell only, so  dL/d im[p] = sum_n sum_c lamH'_c[p] * (-S C_c(E')[p]),  lamH' = cotangent of the       */
/* post-step H (the cotangent as it stands after B1, before B5).  Like dL/d inv_eps it is formed on the interior I  */
/* only (reading R17), where C = curl+ E' has no psi term and the primal fields are reconstructed.  Same loop as     */
/* orc_inv_H with the accumulation added; lam = NULL or g_mu = NULL: orc_inv_H itself.                               */
void orc_inv_H_grad(orc_state *st, REAL *fields, const REAL *im, const REAL *rec_n, const REAL *lam, REAL *g_mu)
{
    const orc_desc *D = &st->D;
    const REAL S = (REAL)D->S;
    const size_t nc = st->nc;
    const REAL *E[3] = { fields, fields + nc, fields + 2 * nc };
    REAL *H[3] = { fields + 3 * nc, fields + 4 * nc, fields + 5 * nc };
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = lo_I(D, 2); k < hi_I(D, 2); ++k)
        for (int j = lo_I(D, 1); j < hi_I(D, 1); ++j)
            for (int i = lo_I(D, 0); i < hi_I(D, 0); ++i) {
                const size_t p = IDX(i, j, k);
                REAL acc = (REAL)0;
                for (int c = 0; c < 3; ++c) {
                    const int a = (c + 1) % 3, b = (c + 2) % 3;
                    REAL d1 = E_plus(D, E, rec_n, b, a, i, j, k) - E[b][p];
                    REAL d2 = E_plus(D, E, rec_n, a, b, i, j, k) - E[a][p];
                    if (lam && g_mu) acc += lam[(size_t)(3 + c) * nc + p] * (d1 - d2);
                    H[c][p] += S * (im ? im[p] : (REAL)1) * (d1 - d2);
                }
                if (lam && g_mu) g_mu[p] -= S * acc;
            }
}

void orc_inv_H(orc_state *st, REAL *fields, const REAL *im, const REAL *rec_n)
{
    const orc_desc *D = &st->D;
    const REAL S = (REAL)D->S;
    const size_t nc = st->nc;
    const REAL *E[3] = { fields, fields + nc, fields + 2 * nc };
    REAL *H[3] = { fields + 3 * nc, fields + 4 * nc, fields + 5 * nc };
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = lo_I(D, 2); k < hi_I(D, 2); ++k)
        for (int j = lo_I(D, 1); j < hi_I(D, 1); ++j)
            for (int i = lo_I(D, 0); i < hi_I(D, 0); ++i) {
                const size_t p = IDX(i, j, k);
                for (int c = 0; c < 3; ++c) {
                    const int a = (c + 1) % 3, b = (c + 2) % 3;
                    REAL d1 = E_plus(D, E, rec_n, b, a, i, j, k) - E[b][p];
                    REAL d2 = E_plus(D, E, rec_n, a, b, i, j, k) - E[a][p];
                    H[c][p] += S * (im ? im[p] : (REAL)1) * (d1 - d2);
                }
            }
}

/* ------------------------------------------------------------------------ */
/* O7a: q = curl- H on I (an H operand at index d-1 comes from the record),  */
/*      g += S sum_c lamE_c q_c   (VJP wrt inv_eps; lamE is the cotangent of */
/*      the post-update E'),  E = E' - S ie q   (inverse E step).            */
/* E sources are subtracted by the caller before this function.             */
/* ------------------------------------------------------------------------ */
static REAL H_minus(const orc_desc *D, const REAL *const H[3], const REAL *rec_n,
                    int comp, int axis, int i, int j, int k)
{
    int pos[3] = { i, j, k };
    pos[axis] -= 1;
    if (D->d > 0 && pos[axis] == lo_I(D, axis) - 1) {
        int which = (comp - axis - 1 + 3) % 3;
        return rec_n[rec_offset(D, axis, 0, which) + face_index(D, axis, pos)];
    }
    return at(D, H[comp], pos[0], pos[1], pos[2]);
}

void orc_inv_E_grad(orc_state *st, REAL *fields, const REAL *ie, const REAL *lam,
                    REAL *g, const REAL *rec_n)
{
    const orc_desc *D = &st->D;
    const REAL S = (REAL)D->S;
    const size_t nc = st->nc;
    REAL *E[3] = { fields, fields + nc, fields + 2 * nc };
    const REAL *H[3] = { fields + 3 * nc, fields + 4 * nc, fields + 5 * nc };
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = lo_I(D, 2); k < hi_I(D, 2); ++k)
        for (int j = lo_I(D, 1); j < hi_I(D, 1); ++j)
            for (int i = lo_I(D, 0); i < hi_I(D, 0); ++i) {
                const size_t p = IDX(i, j, k);
                REAL acc = (REAL)0;
                for (int c = 0; c < 3; ++c) {
                    const int a = (c + 1) % 3, b = (c + 2) % 3;
                    REAL d1 = H[b][p] - H_minus(D, H, rec_n, b, a, i, j, k);
                    REAL d2 = H[a][p] - H_minus(D, H, rec_n, a, b, i, j, k);
                    REAL q = d1 - d2;
                    if (lam) acc += lam[(size_t)c * nc + p] * q;
                    if (lam && g && st->aniso) g[(size_t)c * nc + p] += S * lam[(size_t)c * nc + p] * q;
                    E[c][p] -= S * IEC(c, p) * q;
                }
                if (g && !st->aniso) g[p] += S * acc;
            }
}

/* ------------------------------------------------------------------------ */
/* reverse driver (time-reversed gradient):                    */
/* for n = n_steps-1 .. 0:  B1, [O4^T: nothing], B2, primal -srcH, O6c,      */
/*                          O7a (after -srcE), B5                            */
/* fields: in = state n_steps (valid on I), out = reconstructed state 0 on I */
/* g (cells) and dL_dfields0 (6*cells, may be NULL) are outputs.             */
/* ------------------------------------------------------------------------ */
int orc_backward_mu(orc_state *st, REAL *fields, const REAL *ie, const REAL *im,
                    const orc_source *src, int n_src, const orc_detector *det, int n_det,
                    const REAL *const *dL_dphasor,
                    const orc_tdetector *td, int n_td, const REAL *const *dL_dtd,
                    const REAL *dL_dfields,
                    int n_steps, const REAL *rec, REAL *g, REAL *dL_dfields0, REAL *g_mu);

int orc_backward_td(orc_state *st, REAL *fields, const REAL *ie, const REAL *im,
                    const orc_source *src, int n_src, const orc_detector *det, int n_det,
                    const REAL *const *dL_dphasor,
                    const orc_tdetector *td, int n_td, const REAL *const *dL_dtd,
                    const REAL *dL_dfields,
                    int n_steps, const REAL *rec, REAL *g, REAL *dL_dfields0)
{
    return orc_backward_mu(st, fields, ie, im, src, n_src, det, n_det, dL_dphasor, td, n_td, dL_dtd, dL_dfields,
                           n_steps, rec, g, dL_dfields0, NULL);
}

/* the reverse driver; g_mu (cells, may be NULL): dL/d inv_mu on I (N4) */
int orc_backward_mu(orc_state *st, REAL *fields, const REAL *ie, const REAL *im,
                    const orc_source *src, int n_src, const orc_detector *det, int n_det,
                    const REAL *const *dL_dphasor,
                    const orc_tdetector *td, int n_td, const REAL *const *dL_dtd,
                    const REAL *dL_dfields,
                    int n_steps, const REAL *rec, REAL *g, REAL *dL_dfields0, REAL *g_mu)
{
    const orc_desc *D = &st->D;
    const size_t nc = st->nc;
    const size_t rs = orc_record_stride(D);
    if (D->d > 0 && !rec) return -4;
    if (st->sigma) return -4;                 /* the inverse step is for lossless media */
    REAL *lam = zalloc(6 * nc);
    if (!lam) return -2;
    if (dL_dfields) memcpy(lam, dL_dfields, 6 * nc * sizeof(REAL));      /* B0 */
    orc_zero_lpsi(st);
    memset(g, 0, (st->aniso ? 3 : 1) * nc * sizeof(REAL));
    if (g_mu) memset(g_mu, 0, nc * sizeof(REAL));
    for (int n = n_steps - 1; n >= 0; --n) {
        const REAL *rec_n = rec ? rec + (size_t)n * rs : NULL;
        time_detect_adjoint(D, lam, fields, nc, ie, im, td, n_td, dL_dtd, g, n);   /* N2^T (primal state after step n) */
        detect_adjoint(D, lam, nc, det, n_det, dL_dphasor, n);           /* B1  */
        orc_adj_H(st, lam, im);                                          /* B2  */
        add_sources(D, fields, nc, src, n_src, n, 1, (REAL)-1);          /* undo O4 */
        orc_inv_H_grad(st, fields, im, rec_n, lam, g_mu);                /* O6c (+ N4: dL/d inv_mu) */
        add_sources(D, fields, nc, src, n_src, n, 0, (REAL)-1);          /* undo O2 */
        orc_inv_E_grad(st, fields, ie, lam, g, rec_n);                   /* O7a */
        orc_adj_E(st, lam, ie);                                          /* B5  */
    }
    if (dL_dfields0) memcpy(dL_dfields0, lam, 6 * nc * sizeof(REAL));
    free(lam);
    return 0;
}

int orc_backward(orc_state *st, REAL *fields, const REAL *ie, const REAL *im,
                 const orc_source *src, int n_src, const orc_detector *det, int n_det,
                 const REAL *const *dL_dphasor, const REAL *dL_dfields,
                 int n_steps, const REAL *rec, REAL *g, REAL *dL_dfields0)
{
    return orc_backward_td(st, fields, ie, im, src, n_src, det, n_det, dL_dphasor, NULL, 0, NULL, dL_dfields,
                           n_steps, rec, g, dL_dfields0);
}

/* ------------------------------------------------------------------------ */
/* tape-mode gradient (the plain definition: reverse-mode derivative of the  */
/* forward program with every E-update bracket stored):                      */
/*   g += S sum_c lamE'_c * bracket_n,c    on ALL cells (PML included)       */
/* ------------------------------------------------------------------------ */
int orc_backward_tape(orc_state *st, const REAL *ie, const REAL *im,
                      const orc_detector *det, int n_det,
                      const REAL *const *dL_dphasor, const REAL *dL_dfields,
                      int n_steps, const REAL *tape, REAL *g, REAL *dL_dfields0)
{
    const orc_desc *D = &st->D;
    const size_t nc = st->nc;
    const REAL S = (REAL)D->S;
    REAL *lam = zalloc(6 * nc);
    if (!lam) return -2;
    if (dL_dfields) memcpy(lam, dL_dfields, 6 * nc * sizeof(REAL));
    orc_zero_lpsi(st);
    memset(g, 0, (st->aniso ? 3 : 1) * nc * sizeof(REAL));
    for (int n = n_steps - 1; n >= 0; --n) {
        const REAL *br = tape + (size_t)n * 3 * nc;
        detect_adjoint(D, lam, nc, det, n_det, dL_dphasor, n);
        orc_adj_H(st, lam, im);
        for (int c = 0; c < 3; ++c)
            for (size_t p = 0; p < nc; ++p)
                g[(st->aniso ? (size_t)c * nc : 0) + p] += S * lam[(size_t)c * nc + p] * br[(size_t)c * nc + p];
        orc_adj_E(st, lam, ie);
    }
    if (dL_dfields0) memcpy(dL_dfields0, lam, 6 * nc * sizeof(REAL));
    free(lam);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* B6: chain rule to the design parameters (reading R20).    */
/* On a design box the permittivity is eps = eps_bg + delta_eps * rho, the   */
/* solver's input is ie = 1/eps, hence                                       */
/*   d(ie)/d(rho) = -delta_eps / eps^2 = -delta_eps * ie^2                   */
/*   dL/drho[cell] = g[cell] * d(ie)/d(rho)[cell],   g = dL/d(inv_eps).      */
/* out is box-shaped [k][j][i].  Pinned by a central finite difference of L  */
/* with respect to rho (tests/test_oracle_pins.py), not by this formula.     */
/* ------------------------------------------------------------------------ */
void orc_grad_rho(const orc_desc *D, const REAL *g, const REAL *ie, double delta_eps,
                  const int lo[3], const int hi[3], REAL *out)
{
    const int bx = hi[0] - lo[0], by = hi[1] - lo[1];
    for (int k = lo[2]; k < hi[2]; ++k)
        for (int j = lo[1]; j < hi[1]; ++j)
            for (int i = lo[0]; i < hi[0]; ++i) {
                const size_t p = IDX(i, j, k);
                const size_t c = ((size_t)(k - lo[2]) * by + (j - lo[1])) * bx + (i - lo[0]);
                const REAL dinv = -(REAL)delta_eps * ie[p] * ie[p];
                out[c] = g[p] * dinv;
            }
}

/* ------------------------------------------------------------------------ */
/* N2: Poynting flux through a plane from the DFT phasors (PAPER.md L68      */
/* "Poynting flux", L148 Fig. 5 "fraction of Poynting flux"; L70 "Yee        */
/* interpolation", off by default).  Reading R24:                            */
/* the detector box is a slab normal to `axis` a whose mask holds the four   */
/* tangential components E_b, E_c, H_b, H_c (b = a+1, c = a+2 mod 3); for    */
/* every frequency                                                           */
/*   flux_f = 1/2 sum_cells Re( E_b conj(H_c) - E_c conj(H_b) )     (n = +e_a)*/
/* interpolate = 0: slab one plane thick, phasors multiplied as accumulated  */
/*   (same index, same phase stamp w (n+1): the paper's default);            */
/* interpolate = 1: slab two planes thick (indices p-1, p along a); E from   */
/*   plane p; H co-located with it in space, Hbar = (H[p-1] + H[p])/2 (H_c   */
/*   sits half a cell above E_b along a and at the same in-plane position),  */
/*   and in time, H~ = exp(-i w/2) Hbar (H is stamped half a step late).     */
/* ------------------------------------------------------------------------ */
static int comp_slot(int mask, int comp)
{
    int ci = 0;
    for (int c = 0; c < comp; ++c) ci += (mask >> c) & 1;
    return ci;
}

/* flux[n_freq] out; vjp: dL_dflux[n_freq] in, dL_dphasor (laid out like phasor) written */
static int flux_impl(const orc_detector *q, const REAL *phasor, int axis, int interpolate,
                     REAL *flux, const REAL *dL_dflux, REAL *dL_dphasor)
{
    const int a = axis, b = (a + 1) % 3, c = (a + 2) % 3;
    const int need = (1 << b) | (1 << c) | (1 << (3 + b)) | (1 << (3 + c));
    if ((q->mask & need) != need) return -1;
    const int ext[3] = { q->hi[0] - q->lo[0], q->hi[1] - q->lo[1], q->hi[2] - q->lo[2] };
    if (ext[a] != (interpolate ? 2 : 1)) return -1;
    const size_t bc = (size_t)ext[0] * ext[1] * ext[2];
    const int ncomp = popcount6(q->mask);
    const int sEb = comp_slot(q->mask, b), sEc = comp_slot(q->mask, c);
    const int sHb = comp_slot(q->mask, 3 + b), sHc = comp_slot(q->mask, 3 + c);
    const int t1 = ext[a] - 1;                       /* plane of E (and of the upper H) inside the box */
    if (dL_dphasor) memset(dL_dphasor, 0, (size_t)q->n_freq * ncomp * bc * 2 * sizeof(REAL));
    for (int f = 0; f < q->n_freq; ++f) {
        const double cw = interpolate ? cos(0.5 * q->omega[f]) : 1.0, sw = interpolate ? sin(0.5 * q->omega[f]) : 0.0;
        const REAL *P = phasor + (size_t)f * ncomp * bc * 2;
        REAL *dP = dL_dphasor ? dL_dphasor + (size_t)f * ncomp * bc * 2 : NULL;
        double acc = 0.0;
        int pos[3];
        for (pos[2] = 0; pos[2] < ext[2]; ++pos[2])
            for (pos[1] = 0; pos[1] < ext[1]; ++pos[1])
                for (pos[0] = 0; pos[0] < ext[0]; ++pos[0]) {
                    if (pos[a] != t1) continue;
                    const size_t cell = ((size_t)pos[2] * ext[1] + pos[1]) * ext[0] + pos[0];
                    int pm[3] = { pos[0], pos[1], pos[2] };
                    pm[a] -= 1;
                    const size_t cellm = interpolate ? ((size_t)pm[2] * ext[1] + pm[1]) * ext[0] + pm[0] : cell;
                    /* pair 0: E_b with H_c (sign +), pair 1: E_c with H_b (sign -) */
                    for (int pr = 0; pr < 2; ++pr) {
                        const int sE = pr ? sEc : sEb, sH = pr ? sHb : sHc;
                        const double sg = pr ? -1.0 : 1.0;
                        const REAL *E = P + ((size_t)sE * bc + cell) * 2;
                        const REAL *H1 = P + ((size_t)sH * bc + cell) * 2, *H0 = P + ((size_t)sH * bc + cellm) * 2;
                        const double hr = interpolate ? 0.5 * ((double)H0[0] + H1[0]) : (double)H1[0];
                        const double hi = interpolate ? 0.5 * ((double)H0[1] + H1[1]) : (double)H1[1];
                        const double tr = hr * cw + hi * sw, ti = hi * cw - hr * sw;      /* H~ = exp(-i w/2) Hbar */
                        acc += sg * 0.5 * ((double)E[0] * tr + (double)E[1] * ti);
                        if (dP) {
                            const double G = sg * 0.5 * (double)dL_dflux[f];
                            REAL *dE = dP + ((size_t)sE * bc + cell) * 2;
                            dE[0] += (REAL)(G * tr); dE[1] += (REAL)(G * ti);
                            const double dtr = G * (double)E[0], dti = G * (double)E[1];
                            const double dhr = dtr * cw - dti * sw, dhi = dtr * sw + dti * cw;
                            REAL *d1 = dP + ((size_t)sH * bc + cell) * 2;
                            if (interpolate) {
                                REAL *d0 = dP + ((size_t)sH * bc + cellm) * 2;
                                d1[0] += (REAL)(0.5 * dhr); d1[1] += (REAL)(0.5 * dhi);
                                d0[0] += (REAL)(0.5 * dhr); d0[1] += (REAL)(0.5 * dhi);
                            } else {
                                d1[0] += (REAL)dhr; d1[1] += (REAL)dhi;
                            }
                        }
                    }
                }
        if (flux) flux[f] = (REAL)acc;
    }
    return 0;
}

int orc_flux(const orc_detector *q, const REAL *phasor, int axis, int interpolate, REAL *flux)
{
    return flux_impl(q, phasor, axis, interpolate, flux, NULL, NULL);
}

int orc_flux_vjp(const orc_detector *q, const REAL *phasor, int axis, int interpolate,
                 const REAL *dL_dflux, REAL *dL_dphasor)
{
    return flux_impl(q, phasor, axis, interpolate, NULL, dL_dflux, dL_dphasor);
}

/* ------------------------------------------------------------------------ */
/* N2: one-directional plane source = Total-Field/Scattered-Field interface  */
/* ("Total-Field Scattered-Field", L130).  Reading R25.         */
/* A plane wave travelling along axis a (dir = +1 / -1), E polarised along   */
/* `pol` = b != a, its H along the third axis c, in a medium that is uniform */
/* (eps_r, mu_r) on the planes the interface touches.  With                  */
/*   sgn = +1 if a == b+1 (mod 3), -1 if a == b+2                            */
/* the updates of 8.0 restricted to this wave are the 1-D leapfrog           */
/*   e[m] += sgn S ie (h[m] - h[m-1]) ;  h[m] += sgn S im (e[m+1] - e[m]).   */
/* The incident wave is generated on an auxiliary 1-D grid of exactly that   */
/* form (same S, same medium, hard source e[0] = base[n], long enough that   */
/* its far wall is out of causal reach), so it carries the 3-D grid's own    */
/* numerical dispersion and the field behind the interface cancels to        */
/* rounding.  Interface at plane p0 (aux node m0 = 2), total-field side =    */
/* the side the wave travels to.  The two additive patches (R10/R11) are     */
/*   E_b on plane p0            : wE[n] = -sgn S ie h_aux^{n+1/2}[m0-1]      */
/*   H_c on plane p0-1 (dir +1) : wH[n] = -sgn S im e_aux^{n+1}[m0]          */
/*   H_c on plane p0   (dir -1) : wH[n] = +sgn S im e_aux^{n+1}[m0]          */
/* (for dir = -1 the aux axis is the mirror image; mirroring flips h).       */
/* Returns the H component (3 + c) and writes *h_plane_offset = -1 or 0.     */
/* ------------------------------------------------------------------------ */
int orc_tfsf_plane(double S, double eps_r, double mu_r, int axis, int pol, int dir,
                   int n_steps, const double *base, double *wE, double *wH, int *h_plane_offset)
{
    if (axis < 0 || axis > 2 || pol < 0 || pol > 2 || pol == axis || (dir != 1 && dir != -1)) return -1;
    const int a = axis, b = pol, c = 3 - a - b;
    const double sgn = (a == (b + 1) % 3) ? 1.0 : -1.0;
    const double ie = 1.0 / eps_r, im = 1.0 / mu_r;
    const int m0 = 2, L = m0 + n_steps / 2 + 16;
    double *e = (double *)calloc((size_t)L + 1, sizeof(double)), *h = (double *)calloc((size_t)L + 1, sizeof(double));
    if (!e || !h) { free(e); free(h); return -2; }
    for (int n = 0; n < n_steps; ++n) {
        wE[n] = -sgn * S * ie * h[m0 - 1];
        for (int m = L - 1; m >= 1; --m) e[m] += sgn * S * ie * (h[m] - h[m - 1]);
        e[0] = base[n];
        wH[n] = (dir > 0 ? -1.0 : 1.0) * sgn * S * im * e[m0];
        for (int m = 0; m < L - 1; ++m) h[m] += sgn * S * im * (e[m + 1] - e[m]);
    }
    free(e); free(h);
    if (h_plane_offset) *h_plane_offset = dir > 0 ? -1 : 0;
    return 3 + c;
}
