// fdtd_api.cu -- the C ABI of include/fdtd.h: validation, the grid object, host orchestration.
// Every step of the path runs in the kernels of kernels_generic.cu / kernels_step.cu; this
// file only owns memory, builds tables and enqueues launches (through CUDA graphs).
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>
#include <new>

#include "fdtd_internal.h"
#include "fdtd_grid.h"

using namespace fdtd;

namespace {

thread_local std::string g_err;

int fail(int code, const std::string &msg)
{
    g_err = msg;
    return code;
}

}  // namespace
int fdtd_fail(int code, const std::string &msg) { return fail(code, msg); }
namespace {

int cuda_fail(cudaError_t e, const char *what)
{
    // clear the sticky-less error state so later calls report their own errors
    (void)cudaGetLastError();
    return fail(e == cudaErrorMemoryAllocation ? FDTD_ENOMEM : FDTD_ECUDA,
                std::string(what) + ": " + cudaGetErrorString(e));
}

#define CK(call)                                                       \
    do {                                                               \
        cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call);          \
    } while (0)

int dim_of(const Dims &G, int a) { return a == 0 ? G.nx : (a == 1 ? G.ny : G.nz); }

// CPML tables (PAPER.md L72 -> ref. 7; constants: reading R8), fp64 on the host.
//   depth rho(x) = max(0, d - x, x - (N - d)), r = rho/d
//   sigma = sigma_max r^m, kappa = 1 + (kappa_max - 1) r^m, alpha = alpha_max (1 - r)^m_alpha
//   b = exp(-(sigma/kappa + alpha) S), a = sigma (b - 1) / (kappa (sigma + kappa alpha)), ik = 1/kappa
void make_table(int n, int d, int half, double S, double m, double smax, double kmax, double amax,
                double am, float *b, float *a, float *ik)
{
    for (int p = 0; p < n; ++p) {
        const double x = p + (half ? 0.5 : 0.0);
        double rho = 0.0;
        if (d > 0) rho = std::max(0.0, std::max((double)d - x, x - (double)(n - d)));
        if (rho <= 0.0) { b[p] = 1.f; a[p] = 0.f; ik[p] = 1.f; continue; }
        const double r = rho / d;
        const double rm = std::pow(r, m);
        const double sig = smax * rm, kap = 1.0 + (kmax - 1.0) * rm, alp = amax * std::pow(1.0 - r, am);
        const double bb = std::exp(-(sig / kap + alp) * S);
        const double aa = sig > 0.0 ? sig * (bb - 1.0) / (kap * (sig + kap * alp)) : 0.0;
        b[p] = (float)bb; a[p] = (float)aa; ik[p] = (float)(1.0 / kap);
    }
}

void make_rec_layout(const Dims &G, RecLayout &R)
{
    std::memset(&R, 0, sizeof(R));
    if (G.d == 0) return;
    long long off = 0;
    for (int a = 0; a < 3; ++a) {
        int u = (a + 1) % 3, v = (a + 2) % 3;
        if (u > v) std::swap(u, v);
        R.fast[a] = u; R.slow[a] = v;
        R.cells[a] = (long long)(G.hi[u] - G.lo[u]) * (G.hi[v] - G.lo[v]);
        const long long seg = (R.cells[a] + 3) / 4 * 4;
        for (int side = 0; side < 2; ++side)
            for (int which = 0; which < 2; ++which) { R.off[a][side][which] = off; off += seg; }
    }
    R.stride = (off + 31) / 32 * 32;
}

bool box_ok(const Dims &G, const int32_t lo[3], const int32_t hi[3])
{
    for (int a = 0; a < 3; ++a)
        if (lo[a] < 0 || hi[a] > dim_of(G, a) || lo[a] >= hi[a]) return false;
    return true;
}

int popcount6(int m) { int n = 0; for (int c = 0; c < 6; ++c) n += (m >> c) & 1; return n; }

constexpr int CS_PREALLOC_FREQ = 16;     // frequencies (summed over the detectors) the (cos, sin) table is sized for at create time

}  // namespace

// ================================================================================================
// grid lifetime
// ================================================================================================
int fdtd_grid::alloc(void **p, size_t bytes, bool recorder)
{
    *p = nullptr;
    if (bytes == 0) return FDTD_OK;
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        char buf[160];
        std::snprintf(buf, sizeof buf, "cudaMalloc(%zu bytes) failed: %s", bytes, cudaGetErrorString(e));
        return fail(FDTD_ENOMEM, buf);
    }
    owned.push_back(*p);
    if (recorder) recorder_bytes += (long long)bytes; else scratch_bytes += (long long)bytes;
    return FDTD_OK;
}

int fdtd_grid::alloc_psi(PsiSet &s)
{
    for (int c = 0; c < 3; ++c)
        for (int q = 0; q < 2; ++q) {
            const size_t bytes = (size_t)psi_elems(G, psi_axis(c, q)) * sizeof(float);
            int rc = alloc((void **)&s.p[c][q], bytes);
            if (rc) return rc;
        }
    return FDTD_OK;
}

int fdtd_grid::zero_psi(const PsiSet &s, cudaStream_t st)
{
    for (int c = 0; c < 3; ++c)
        for (int q = 0; q < 2; ++q) {
            const size_t bytes = (size_t)psi_elems(G, psi_axis(c, q)) * sizeof(float);
            if (bytes) CK(cudaMemsetAsync(s.p[c][q], 0, bytes, st));
        }
    return FDTD_OK;
}

void fdtd_grid::drop_graphs()
{
    for (GraphCache *gc : { &fwd_graph, &bwd_graph }) {
        if (gc->done) { cudaEventSynchronize(gc->done); }
        if (gc->exec_main) cudaGraphExecDestroy(gc->exec_main);
        for (int q = 0; q < 2; ++q) if (gc->exec_tail[q]) { cudaGraphExecDestroy(gc->exec_tail[q]); gc->exec_tail[q] = nullptr; }
        gc->exec_main = nullptr;
        gc->key.clear();
    }
}

extern "C" int fdtd_create_grid(const fdtd_grid_desc *desc, fdtd_grid **out)
{
    if (out) *out = nullptr;
    if (!desc || !out) return fail(FDTD_EINVAL, "fdtd_create_grid: NULL argument");
    if (desc->nx < 1 || desc->ny < 1 || desc->nz < 1) return fail(FDTD_EINVAL, "grid dims must be >= 1");
    if ((long long)desc->nx * desc->ny * desc->nz > (1LL << 40)) return fail(FDTD_EINVAL, "grid too large");
    if (!(desc->courant > 0.f) || !(desc->courant < 0.57735027f))
        return fail(FDTD_EINVAL, "courant must satisfy 0 < S < 1/sqrt(3)");
    if (desc->pml_cells < 0) return fail(FDTD_EINVAL, "pml_cells must be >= 0");
    if (desc->periodic && desc->pml_cells != 0) return fail(FDTD_EINVAL, "a periodic grid cannot have a PML");
    const bool sub = desc->z_global != 0;
    if (sub) {
        if (desc->periodic) return fail(FDTD_EINVAL, "a z-slab sub-grid cannot be periodic");
        if (desc->z_ghost_lo < 0 || desc->z_ghost_lo > 1 || desc->z_ghost_hi < 0 || desc->z_ghost_hi > 1)
            return fail(FDTD_EINVAL, "z_ghost_lo / z_ghost_hi must be 0 or 1");
        if (desc->z_offset < 0 || desc->z_offset + desc->nz > desc->z_global || desc->nz - desc->z_ghost_lo - desc->z_ghost_hi < 1)
            return fail(FDTD_EINVAL, "sub-grid planes [z_offset, z_offset + nz) must lie inside [0, z_global) and own at least one plane");
        if ((desc->z_ghost_lo == 0) != (desc->z_offset == 0) || (desc->z_ghost_hi == 0) != (desc->z_offset + desc->nz == desc->z_global))
            return fail(FDTD_EINVAL, "a sub-grid has a ghost plane exactly where it does not touch the end of the global grid");
    } else if (desc->z_offset || desc->z_ghost_lo || desc->z_ghost_hi) {
        return fail(FDTD_EINVAL, "z_offset / z_ghost_* need z_global");
    }
    const int nz_full = sub ? desc->z_global : desc->nz;
    const int mn = std::min(desc->nx, std::min(desc->ny, nz_full));
    if (desc->pml_cells > 0 && 2 * desc->pml_cells + 2 > mn)
        return fail(FDTD_EINVAL, "need 2*pml_cells + 2 <= min(nx,ny,nz)");
    if (desc->max_steps < 0) return fail(FDTD_EINVAL, "max_steps must be >= 0");
    if (desc->record < 0 || desc->record > 3) return fail(FDTD_EINVAL, "record must be 0, 1, 2 or 3");
    if (desc->checkpoint_every < 0) return fail(FDTD_EINVAL, "checkpoint_every must be >= 0");
    if (desc->record == 3 && desc->z_global) return fail(FDTD_EINVAL, "the checkpointed reverse sweep is not available on a z-slab sub-grid");
    if (desc->path < 0 || desc->path > 2) return fail(FDTD_EINVAL, "unknown path");
    if (desc->reserved[0]) return fail(FDTD_EINVAL, "reserved fields must be zero");
    if (desc->flags & ~(FDTD_FLAG_HOST_STAGING | FDTD_FLAG_RECORDER_FP16 | FDTD_FLAG_ANISO_EPS)) return fail(FDTD_EINVAL, "unknown bit in flags");
    if ((desc->flags & FDTD_FLAG_ANISO_EPS) && (desc->flags & FDTD_FLAG_HOST_STAGING))
        return fail(FDTD_EINVAL, "the host-buffer entry points take one inv_eps volume (no FDTD_FLAG_ANISO_EPS)");
    if (desc->pml_m < 0 || desc->pml_sigma_scale < 0 || desc->pml_kappa_max < 0 || desc->pml_alpha_max < 0 ||
        desc->pml_alpha_m < 0 || desc->pml_eps_bg < 0)
        return fail(FDTD_EINVAL, "CPML constants must be >= 0");
    if (desc->pml_kappa_max != 0.f && desc->pml_kappa_max < 1.f) return fail(FDTD_EINVAL, "pml_kappa_max must be >= 1");

    fdtd_grid *g = new (std::nothrow) fdtd_grid();
    if (!g) return fail(FDTD_ENOMEM, "host allocation failed");
    g->desc = *desc;
    Dims &G = g->G;
    G.nx = desc->nx; G.ny = desc->ny; G.nz = desc->nz;
    G.d = desc->pml_cells;
    G.periodic = desc->periodic ? 1 : 0;
    G.S = desc->courant;
    G.nc = (long long)G.nx * G.ny * G.nz;
    const int dp4 = (G.d + 3) / 4 * 4;
    G.dpx = (G.nx % 4 == 0 && G.nx >= 2 * dp4) ? dp4 : G.d;
    for (int a = 0; a < 3; ++a) { G.lo[a] = G.d; G.hi[a] = dim_of(G, a) - G.d; }
    G.aniso = (desc->flags & FDTD_FLAG_ANISO_EPS) ? 1 : 0;
    G.zoff = sub ? desc->z_offset : 0; G.nzg = nz_full;
    G.zl = std::min(G.nz, std::max(0, G.d - G.zoff));
    G.zh = std::min(G.nz, std::max(0, G.zoff + G.nz - (G.nzg - G.d)));
    if (sub) {
        // interior box along z: the global interior restricted to the planes this sub-grid owns (local indices)
        const int own_lo = G.zoff + desc->z_ghost_lo, own_hi = G.zoff + G.nz - desc->z_ghost_hi;
        G.lo[2] = std::max(G.d, own_lo) - G.zoff;
        G.hi[2] = std::min(G.nzg - G.d, own_hi) - G.zoff;
        if (G.hi[2] <= G.lo[2]) { delete g; return fail(FDTD_EINVAL, "a sub-grid must own at least one plane of the interior"); }
    }
    bool all_zero = true;
    for (int a = 0; a < 3; ++a) if (desc->grad_lo[a] || desc->grad_hi[a]) all_zero = false;
    for (int a = 0; a < 3; ++a) {
        if (all_zero) { G.glo[a] = G.lo[a]; G.ghi[a] = G.hi[a]; }
        else {
            if (desc->grad_lo[a] < 0 || desc->grad_hi[a] > dim_of(G, a) || desc->grad_lo[a] >= desc->grad_hi[a]) {
                delete g;
                return fail(FDTD_EINVAL, "grad box outside the grid or empty");
            }
            G.glo[a] = std::max(desc->grad_lo[a], G.lo[a]);
            G.ghi[a] = std::max(G.glo[a], std::min(desc->grad_hi[a], G.hi[a]));
        }
    }
    // record == 3 (checkpointed reverse sweep): no inverse step, so the gradient box is any box of the grid, PML included
    if (desc->record == 3)
        for (int a = 0; a < 3; ++a) {
            G.glo[a] = all_zero ? 0 : desc->grad_lo[a];
            G.ghi[a] = all_zero ? dim_of(G, a) : desc->grad_hi[a];
        }
    // record == 2 (NEXT N1, design-box recorder): the reconstruction box shrinks from the interior I to the
    // gradient box -- the faces recorded, the inverse step and the reconstructed fields all follow G.lo / G.hi
    if (desc->record == 2 && G.d > 0) {
        for (int a = 0; a < 3; ++a) {
            if (G.ghi[a] <= G.glo[a]) { delete g; return fail(FDTD_EINVAL, "record=2 needs a non-empty gradient box inside the interior"); }
            G.lo[a] = G.glo[a]; G.hi[a] = G.ghi[a];
        }
    }
    make_rec_layout(G, g->R);
    g->R.half = (desc->flags & FDTD_FLAG_RECORDER_FP16) ? 1 : 0;

    int rc = FDTD_OK;
    auto bail = [&](int code) { std::string keep = g_err; fdtd_destroy(g); g_err = keep; return code; };

    // CPML tables
    {
        const double m = desc->pml_m > 0 ? desc->pml_m : 3.0;
        const double ss = desc->pml_sigma_scale > 0 ? desc->pml_sigma_scale : 0.8 * (m + 1.0);
        const double km = desc->pml_kappa_max > 0 ? desc->pml_kappa_max : 1.0;
        const double am = desc->pml_alpha_m > 0 ? desc->pml_alpha_m : 1.0;
        const double eb = desc->pml_eps_bg > 0 ? desc->pml_eps_bg : 1.0;
        const double smax = ss / std::sqrt(eb);
        // every table is padded to a multiple of 4 floats plus 4 tail entries (b=1, a=0, ik=1) so that the
        // fused kernels can read float4s and index N (the first cell outside the grid)
        auto padded = [](int n) { return (n + 4 + 3) / 4 * 4; };
        const int tot = 6 * (padded(G.nx) + padded(G.ny) + padded(G.nz));
        std::vector<float> h(tot);
        float *dev = nullptr;
        if ((rc = g->alloc((void **)&dev, tot * sizeof(float)))) return bail(rc);
        int off = 0;
        for (int fam = 0; fam < 2; ++fam)
            for (int a = 0; a < 3; ++a) {
                const int n = dim_of(G, a), np = padded(n);
                for (int q = 0; q < np; ++q) { h[off + q] = 1.f; h[off + np + q] = 0.f; h[off + 2 * np + q] = 1.f; }
                if (a == 2 && sub) {      // the planes [zoff, zoff + nz) of the global table
                    std::vector<float> tb(G.nzg), ta(G.nzg), tk(G.nzg);
                    make_table(G.nzg, G.d, fam, (double)G.S, m, smax, km, (double)desc->pml_alpha_max, am, tb.data(), ta.data(), tk.data());
                    for (int q = 0; q < n; ++q) { h[off + q] = tb[G.zoff + q]; h[off + np + q] = ta[G.zoff + q]; h[off + 2 * np + q] = tk[G.zoff + q]; }
                } else
                make_table(n, G.d, fam, (double)G.S, m, smax, km, (double)desc->pml_alpha_max, am,
                           &h[off], &h[off + np], &h[off + 2 * np]);
                g->T.b[fam][a] = dev + off; g->T.a[fam][a] = dev + off + np; g->T.ik[fam][a] = dev + off + 2 * np;
                off += 3 * np;
            }
        cudaError_t e = cudaMemcpy(dev, h.data(), tot * sizeof(float), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) return bail(cuda_fail(e, "upload CPML tables"));
        g->h_tables = h;
    }
    if ((rc = g->alloc((void **)&g->d_step, 64))) return bail(rc);
    if ((rc = g->alloc((void **)&g->red.partial, RED_BLOCKS * sizeof(double))) || (rc = g->alloc((void **)&g->red.ticket, 64))) return bail(rc);
    if (cudaMemset(g->red.ticket, 0, 64) != cudaSuccess) return bail(cuda_fail(cudaGetLastError(), "cudaMemset"));
    if ((rc = g->alloc_psi(g->psiE[0])) || (rc = g->alloc_psi(g->psiH[0]))) return bail(rc);
    if ((desc->record == 1 || desc->record == 2) && G.d > 0 && desc->max_steps > 0) {
        const size_t bytes = (size_t)g->R.stride * (g->R.half ? 2 : sizeof(float)) * (size_t)desc->max_steps;
        if ((rc = g->alloc((void **)&g->rec, bytes, true))) return bail(rc);
    }
    if (desc->record == 3 && desc->max_steps > 0) {
        // checkpoints of the whole state (6 volumes + the 12 psi arrays) every K steps, and dE = E' - E on the gradient box
        // for the K steps of one segment; K defaults to ~sqrt(max_steps), which minimises their sum for a box of the grid's size
        g->ck_every = desc->checkpoint_every > 0 ? desc->checkpoint_every : std::max(1, (int)std::lround(std::sqrt((double)desc->max_steps)));
        g->ck_count = (desc->max_steps + g->ck_every - 1) / g->ck_every;
        size_t psi_floats = 0;
        for (int c = 0; c < 3; ++c) for (int q = 0; q < 2; ++q) psi_floats += (size_t)psi_elems(G, psi_axis(c, q));
        g->ck_stride = 6 * (size_t)G.nc + 2 * psi_floats;
        const size_t box = (size_t)(G.ghi[0] - G.glo[0]) * (G.ghi[1] - G.glo[1]) * (G.ghi[2] - G.glo[2]);
        if ((rc = g->alloc((void **)&g->ckpt, g->ck_stride * g->ck_count * sizeof(float), true))) return bail(rc);
        if ((rc = g->alloc((void **)&g->dE, 3 * box * (size_t)g->ck_every * sizeof(float), true))) return bail(rc);
    }
    {
        cudaError_t e = cudaStreamCreateWithFlags(&g->cap_stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) return bail(cuda_fail(e, "cudaStreamCreate"));
        e = cudaEventCreateWithFlags(&g->fwd_graph.done, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g->bwd_graph.done, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g->table_done, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g->fork_ev, cudaEventDisableTiming);
        for (int q = 0; q < 2 && e == cudaSuccess; ++q) {
            e = cudaStreamCreateWithFlags(&g->side_stream[q], cudaStreamNonBlocking);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g->join_ev[q], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) return bail(cuda_fail(e, "cudaEventCreate"));
    }
    g->path = FDTD_PATH_GENERIC;
    rc = fused_setup(g);          // may switch g->path to FDTD_PATH_FUSED (kernels_step.cu)
    if (rc) return bail(rc);
    if (desc->path == FDTD_PATH_FUSED && g->path != FDTD_PATH_FUSED)
        return bail(fail(FDTD_EINVAL, "FDTD_PATH_FUSED requested but the grid does not qualify: " + g->fused_why_not));
    // everything the entry points need is allocated here (include/fdtd.h "Memory / ownership"): a recording grid will
    // run fdtd_backward, so its cotangent volumes exist from the start; the (cos, sin) table is sized for
    // CS_PREALLOC_FREQ frequencies; the staging buffers of the *_host entry points when the flag asks for them
    if (desc->record && (rc = g->ensure_backward_buffers())) return bail(rc);
    if (desc->max_steps > 0 && (rc = g->reserve_cs_table((size_t)desc->max_steps * CS_PREALLOC_FREQ * 2))) return bail(rc);
    if ((desc->flags & FDTD_FLAG_HOST_STAGING) && (rc = g->ensure_host_buffers(false, desc->record != 0))) return bail(rc);
    *out = g;
    return FDTD_OK;
}

extern "C" int fdtd_destroy(fdtd_grid *g)
{
    if (!g) return FDTD_OK;
    cudaDeviceSynchronize();
    g->drop_graphs();
    fused_teardown(g);
    for (void *p : g->owned) cudaFree(p);
    if (g->h_cs) cudaFreeHost(g->h_cs);
    if (g->cap_stream) cudaStreamDestroy(g->cap_stream);
    if (g->fwd_graph.done) cudaEventDestroy(g->fwd_graph.done);
    if (g->bwd_graph.done) cudaEventDestroy(g->bwd_graph.done);
    if (g->table_done) cudaEventDestroy(g->table_done);
    if (g->fork_ev) cudaEventDestroy(g->fork_ev);
    for (int q = 0; q < 2; ++q) {
        if (g->side_stream[q]) cudaStreamDestroy(g->side_stream[q]);
        if (g->join_ev[q]) cudaEventDestroy(g->join_ev[q]);
    }
    for (auto &sp : g->prof_spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
    for (cudaEvent_t e : g->prof_pool) cudaEventDestroy(e);
    (void)cudaGetLastError();
    delete g;
    return FDTD_OK;
}

extern "C" const char *fdtd_last_error(void) { return g_err.c_str(); }
extern "C" const char *fdtd_version(void) { return "fdtd-b200 0.1 sm_100a"; }

cudaEvent_t fdtd_grid::prof_begin(cudaStream_t st)
{
    if (!profiling || prof_capturing) return nullptr;
    cudaEvent_t a = nullptr;
    if (!prof_pool.empty()) { a = prof_pool.back(); prof_pool.pop_back(); }
    else if (cudaEventCreate(&a) != cudaSuccess) return nullptr;
    cudaEventRecord(a, st);
    return a;
}

void fdtd_grid::prof_end(int cls, cudaEvent_t a, cudaStream_t st)
{
    cudaEvent_t b = nullptr;
    if (!prof_pool.empty()) { b = prof_pool.back(); prof_pool.pop_back(); }
    else if (cudaEventCreate(&b) != cudaSuccess) { prof_pool.push_back(a); return; }
    cudaEventRecord(b, st);
    prof_spans.push_back({ cls, a, b });
}

extern "C" int fdtd_set_profiling(fdtd_grid *g, int32_t enable)
{
    if (!g) return fail(FDTD_EINVAL, "fdtd_set_profiling: NULL grid");
    g->profiling = enable != 0;
    return FDTD_OK;
}

extern "C" int fdtd_get_profile(fdtd_grid *g, fdtd_profile *out)
{
    if (!g || !out) return fail(FDTD_EINVAL, "fdtd_get_profile: NULL argument");
    static const char *names[fdtd_grid::PC_COUNT] = { "update_E", "update_H", "adjoint_H", "inverse_H", "inverse_E_grad",
        "adjoint_E", "fused_forward_step", "fused_adjoint_step", "fused_inverse_step", "record_faces", "inject_faces", "source_detector", "other" };
    for (auto &sp : g->prof_spans) {
        cudaError_t e = cudaEventSynchronize(sp.b);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, sp.a, sp.b);
        if (e != cudaSuccess) return cuda_fail(e, "fdtd_get_profile");
        g->prof_ms[sp.cls] += ms;
        g->prof_launches[sp.cls] += 1;
        g->prof_pool.push_back(sp.a);
        g->prof_pool.push_back(sp.b);
    }
    g->prof_spans.clear();
    std::memset(out, 0, sizeof(*out));
    out->n_classes = fdtd_grid::PC_COUNT;
    for (int c = 0; c < fdtd_grid::PC_COUNT; ++c) {
        std::snprintf(out->name[c], sizeof out->name[c], "%s", names[c]);
        out->launches[c] = g->prof_launches[c];
        out->total_ms[c] = g->prof_ms[c];
        g->prof_launches[c] = 0;
        g->prof_ms[c] = 0.0;
    }
    return FDTD_OK;
}

extern "C" int fdtd_get_info(const fdtd_grid *g, fdtd_grid_info *info)
{
    if (!g || !info) return fail(FDTD_EINVAL, "fdtd_get_info: NULL argument");
    std::memset(info, 0, sizeof(*info));
    info->path = g->path;
    info->tile_x = g->tile_x; info->tile_y = g->tile_y; info->tile_z = g->tile_z;
    info->kernel_launches = g->kernel_launches;
    info->recorder_bytes = g->recorder_bytes;
    info->scratch_bytes = g->scratch_bytes;
    info->record_floats_per_step = g->R.stride;
    info->pipelined_inverse_ctas = g->pipelined_inverse_ctas;
    info->fused_step_launches = g->fused_step_launches;
    info->fused_inverse_launches = g->fused_inverse_launches;
    info->partition = g->path == FDTD_PATH_FUSED ? g->partition : FDTD_PARTITION_NONE;
    return FDTD_OK;
}

// ================================================================================================
// argument checking and descriptor translation
// ================================================================================================
namespace {

int check_common(fdtd_grid *g, const float *fields, const float *inv_eps, const fdtd_source *src, int n_src,
                 const fdtd_detector *det, int n_det, int n_steps, const char *who)
{
    if (!g) return fail(FDTD_EINVAL, std::string(who) + ": NULL grid");
    if (!fields || !inv_eps) return fail(FDTD_EINVAL, std::string(who) + ": fields and inv_eps are required");
    if (n_steps < 0 || n_steps > g->desc.max_steps) return fail(FDTD_EINVAL, std::string(who) + ": need 0 <= n_steps <= max_steps");
    if (n_src < 0 || n_det < 0 || (n_src && !src) || (n_det && !det))
        return fail(FDTD_EINVAL, std::string(who) + ": bad source/detector array");
    for (int s = 0; s < n_src; ++s) {
        if (src[s].component < 0 || src[s].component > 5) return fail(FDTD_EINVAL, "source component must be 0..5");
        if (!box_ok(g->G, src[s].lo, src[s].hi)) return fail(FDTD_EINVAL, "source box outside the grid or empty");
        if (!src[s].waveform) return fail(FDTD_EINVAL, "source waveform is NULL");
    }
    for (int s = 0; s < n_det; ++s) {
        if (det[s].component_mask <= 0 || det[s].component_mask > 63) return fail(FDTD_EINVAL, "detector component_mask must be 1..63");
        if (!box_ok(g->G, det[s].lo, det[s].hi)) return fail(FDTD_EINVAL, "detector box outside the grid or empty");
        if (det[s].n_freq < 1 || !det[s].omega) return fail(FDTD_EINVAL, "detector needs n_freq >= 1 and omega");
    }
    return FDTD_OK;
}

void translate(const fdtd_source *src, int n_src, std::vector<SourceDev> &out)
{
    out.resize(n_src);
    for (int s = 0; s < n_src; ++s) {
        out[s].comp = src[s].component;
        for (int a = 0; a < 3; ++a) { out[s].lo[a] = src[s].lo[a]; out[s].hi[a] = src[s].hi[a]; }
        out[s].profile = src[s].profile;
        out[s].waveform = src[s].waveform;
    }
}

int translate(const fdtd_detector *det, int n_det, std::vector<DetectorDev> &out)
{
    out.resize(n_det);
    int tot = 0;
    for (int s = 0; s < n_det; ++s) {
        out[s].mask = det[s].component_mask;
        out[s].ncomp = popcount6(det[s].component_mask);
        for (int a = 0; a < 3; ++a) { out[s].lo[a] = det[s].lo[a]; out[s].hi[a] = det[s].hi[a]; }
        out[s].n_freq = det[s].n_freq;
        out[s].cs_off = tot;
        out[s].phasor = det[s].phasor;
        tot += det[s].n_freq;
    }
    return tot;
}

int translate_td(fdtd_grid *g, const fdtd_time_detector *td, int n_td, int n_steps, std::vector<TimeDetDev> &out, const char *who)
{
    out.clear();
    if (n_td < 0 || (n_td && !td)) return fail(FDTD_EINVAL, std::string(who) + ": bad time-detector array");
    out.resize(n_td);
    for (int s = 0; s < n_td; ++s) {
        if (td[s].kind != FDTD_TD_SNAPSHOT && td[s].kind != FDTD_TD_ENERGY) return fail(FDTD_EINVAL, "time detector kind must be FDTD_TD_SNAPSHOT or FDTD_TD_ENERGY");
        if (td[s].kind == FDTD_TD_SNAPSHOT && (td[s].component_mask <= 0 || td[s].component_mask > 63))
            return fail(FDTD_EINVAL, "snapshot detector component_mask must be 1..63");
        if (!box_ok(g->G, td[s].lo, td[s].hi)) return fail(FDTD_EINVAL, "time detector box outside the grid or empty");
        if (td[s].stride < 1) return fail(FDTD_EINVAL, "time detector stride must be >= 1");
        if (td[s].kind == FDTD_TD_ENERGY && g->G.aniso) return fail(FDTD_EINVAL, "the energy detector is stated for one inv_eps per voxel (no FDTD_FLAG_ANISO_EPS)");
        out[s].kind = td[s].kind;
        out[s].mask = td[s].kind == FDTD_TD_SNAPSHOT ? td[s].component_mask : 0;
        out[s].ncomp = popcount6(out[s].mask);
        for (int a = 0; a < 3; ++a) { out[s].lo[a] = td[s].lo[a]; out[s].hi[a] = td[s].hi[a]; }
        out[s].stride = td[s].stride;
        out[s].out = td[s].out;
    }
    (void)n_steps;
    return FDTD_OK;
}

}  // namespace

// device + pinned host capacity of the (cos, sin) table; earlier uploads have to be finished before the old buffers go
int fdtd_grid::reserve_cs_table(size_t floats)
{
    if (floats <= cs_cap) return FDTD_OK;
    CK(cudaEventSynchronize(table_done));
    if (h_cs) { cudaFreeHost(h_cs); h_cs = nullptr; }
    CK(cudaMallocHost((void **)&h_cs, floats * sizeof(float)));
    int rc = alloc((void **)&d_cs, floats * sizeof(float));
    if (rc) return rc;
    cs_cap = floats;
    return FDTD_OK;
}

namespace {

// (cos, sin) of omega_f*(n+1) for n < n_steps, fp64 on the host, stored fp32 (reading R13)
int upload_cs_table(fdtd_grid *g, const fdtd_detector *det, int n_det, int total_freq, int n_steps, cudaStream_t st)
{
    if (total_freq == 0 || n_steps == 0) return FDTD_OK;
    // the same frequencies and step count as the table on the device (the calls of a range sequence): nothing to do
    std::vector<float> ck;
    ck.push_back((float)n_steps);
    for (int s = 0; s < n_det; ++s) for (int q = 0; q < det[s].n_freq; ++q) ck.push_back(det[s].omega[q]);
    if (ck == g->cs_key) return FDTD_OK;
    g->cs_key.clear();
    const size_t need = (size_t)n_steps * total_freq * 2;
    if (need > g->cs_cap) {       // more than CS_PREALLOC_FREQ frequencies: grow
        int rc = g->reserve_cs_table((size_t)std::max(n_steps, g->desc.max_steps) * total_freq * 2);
        if (rc) return rc;
    }
    CK(cudaEventSynchronize(g->table_done));      // the previous call's upload has left the pinned staging table
    int f0 = 0;
    for (int s = 0; s < n_det; ++s) {
        for (int q = 0; q < det[s].n_freq; ++q) {
            const double om = (double)det[s].omega[q];
            for (int n = 0; n < n_steps; ++n) {
                const double phi = om * (double)(n + 1);
                g->h_cs[((size_t)n * total_freq + f0 + q) * 2] = (float)std::cos(phi);
                g->h_cs[((size_t)n * total_freq + f0 + q) * 2 + 1] = (float)std::sin(phi);
            }
        }
        f0 += det[s].n_freq;
    }
    CK(cudaMemcpyAsync(g->d_cs, g->h_cs, need * sizeof(float), cudaMemcpyHostToDevice, st));
    CK(cudaEventRecord(g->table_done, st));
    g->cs_key = ck;
    return FDTD_OK;
}

// Replays a captured per-step sequence: `unroll` steps per graph launch plus single-step launches for
// the remainder.  `enqueue(stream)` must enqueue exactly one step (reading n from *d_step).
template <class F>
int run_steps(fdtd_grid *g, fdtd_grid::GraphCache &gc, const std::string &key, int n_steps, int launches_per_step,
              cudaStream_t st, F enqueue)
{
    if (n_steps == 0) return FDTD_OK;
    if (g->profiling) {
        g->step_par = 0;
        const long long s0 = g->enq_step, i0 = g->enq_inv;
        for (int n = 0; n < n_steps; ++n) { enqueue(st); g->step_par ^= 1; }
        g->kernel_launches += (long long)n_steps * launches_per_step;
        g->fused_step_launches += g->enq_step - s0; g->fused_inverse_launches += g->enq_inv - i0;
        return FDTD_OK;
    }
    static const int env_unroll = getenv("FDTD_GRAPH_UNROLL") ? std::max(2, atoi(getenv("FDTD_GRAPH_UNROLL")) / 2 * 2) : 0;
    const int unroll = env_unroll ? env_unroll : g->graph_unroll;   // even: a replay of the main graph ends in the slot it began in
    if (gc.key != key || !gc.exec_tail[1]) {
        if (gc.key.size()) CK(cudaEventSynchronize(gc.done));
        if (gc.exec_main) { cudaGraphExecDestroy(gc.exec_main); gc.exec_main = nullptr; }
        for (int q = 0; q < 2; ++q) if (gc.exec_tail[q]) { cudaGraphExecDestroy(gc.exec_tail[q]); gc.exec_tail[q] = nullptr; }
        gc.key.clear();
        for (int which = 0; which < 3; ++which) {            // 0: main graph (slot 0 first), 1 / 2: one step from slot 0 / 1
            const int reps = which ? 1 : unroll;
            cudaGraph_t graph = nullptr;
            CK(cudaStreamBeginCapture(g->cap_stream, cudaStreamCaptureModeThreadLocal));
            g->prof_capturing = true;
            g->step_par = which == 2 ? 1 : 0;
            const long long s0 = g->enq_step, i0 = g->enq_inv;
            for (int r = 0; r < reps; ++r) { enqueue(g->cap_stream); g->step_par ^= 1; }
            if (which == 1) { gc.step_per = g->enq_step - s0; gc.inv_per = g->enq_inv - i0; }   // fused kernels per time step
            g->prof_capturing = false;
            cudaError_t e = cudaStreamEndCapture(g->cap_stream, &graph);
            if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture");
            cudaGraphExec_t exec = nullptr;
            e = cudaGraphInstantiate(&exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) return cuda_fail(e, "cudaGraphInstantiate");
            (which ? gc.exec_tail[which - 1] : gc.exec_main) = exec;
        }
        gc.key = key;
    }
    int left = n_steps, par = 0;
    while (left >= unroll) { CK(cudaGraphLaunch(gc.exec_main, st)); left -= unroll; }
    while (left > 0) { CK(cudaGraphLaunch(gc.exec_tail[par], st)); par ^= 1; --left; }
    CK(cudaEventRecord(gc.done, st));
    g->kernel_launches += (long long)n_steps * launches_per_step;
    g->fused_step_launches += n_steps * gc.step_per; g->fused_inverse_launches += n_steps * gc.inv_per;
    return FDTD_OK;
}

}  // namespace
int fdtd_run_steps_fwd(fdtd_grid *g, const std::string &key, int n_steps, int launches_per_step, cudaStream_t st,
                       void (*enqueue)(void *, cudaStream_t), void *ctx)
{
    return run_steps(g, g->fwd_graph, key, n_steps, launches_per_step, st, [&](cudaStream_t cs) { enqueue(ctx, cs); });
}
int fdtd_run_steps_bwd(fdtd_grid *g, const std::string &key, int n_steps, int launches_per_step, cudaStream_t st,
                       void (*enqueue)(void *, cudaStream_t), void *ctx)
{
    return run_steps(g, g->bwd_graph, key, n_steps, launches_per_step, st, [&](cudaStream_t cs) { enqueue(ctx, cs); });
}
namespace {

std::string make_key(const char *tag, const void *a, const void *b, const void *c, const void *d, const void *e,
                     const std::vector<SourceDev> &S, const std::vector<DetectorDev> &D, int extra)
{
    std::string k(tag);
    auto add = [&](const void *p, size_t n) { k.append((const char *)p, n); };
    add(&a, sizeof a); add(&b, sizeof b); add(&c, sizeof c); add(&d, sizeof d); add(&e, sizeof e);
    add(&extra, sizeof extra);
    if (!S.empty()) add(S.data(), S.size() * sizeof(SourceDev));
    if (!D.empty()) add(D.data(), D.size() * sizeof(DetectorDev));
    return k;
}

}  // namespace

// ================================================================================================
// forward
// ================================================================================================
extern "C" int fdtd_forward(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                            const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                            int32_t n_steps, void *cuda_stream)
{
    return fdtd_forward_td(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, nullptr, 0, n_steps, cuda_stream);
}

static int forward_impl(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                        const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                        const fdtd_time_detector *td, int32_t n_td, int n_begin, int n_end, int n_total, void *cuda_stream);
static int forward_core(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                        const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                        const fdtd_time_detector *td, int32_t n_td, int n_begin, int n_end, int n_total, void *cuda_stream);

// record = 3: the whole state n (fields + the psi set state n lives in) to / from checkpoint slot idx
static int copy_checkpoint(fdtd_grid *g, float *fields, bool fused, int n, int idx, bool restore, cudaStream_t st)
{
    const Dims &G = g->G;
    float *ck = g->ckpt + (size_t)idx * g->ck_stride;
    float *vol = fused ? fused_volume(g, fields, 0, n) : fields;
    const int set = fused ? (n & 1) : 0;
    auto cp = [&](float *dev, float *slot, size_t floats) -> cudaError_t {
        return floats ? cudaMemcpyAsync(restore ? dev : slot, restore ? slot : dev, floats * sizeof(float), cudaMemcpyDeviceToDevice, st) : cudaSuccess;
    };
    CK(cp(vol, ck, 6 * (size_t)G.nc));
    size_t off = 6 * (size_t)G.nc;
    for (int fam = 0; fam < 2; ++fam)
        for (int c = 0; c < 3; ++c)
            for (int q = 0; q < 2; ++q) {
                const size_t fl = (size_t)psi_elems(G, psi_axis(c, q));
                CK(cp((fam ? g->psiH[set] : g->psiE[set]).p[c][q], ck + off, fl));
                off += fl;
            }
    return FDTD_OK;
}

// fdtd_forward on a record = 3 grid: segment by segment, a checkpoint of the state in front of each
static int forward_impl(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                        const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                        const fdtd_time_detector *td, int32_t n_td, int n_begin, int n_end, int n_total, void *cuda_stream)
{
    if (!g || g->desc.record != 3)
        return forward_core(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, td, n_td, n_begin, n_end, n_total, cuda_stream);
    if (n_td) return fail(FDTD_EINVAL, "time-domain detectors are not available on a record = 3 grid");
    if (n_begin != 0 || n_end != n_total) return fail(FDTD_EINVAL, "range calls are not available on a record = 3 grid");
    if (!fields) return fail(FDTD_EINVAL, "fdtd_forward: fields and inv_eps are required");
    const bool fused = g->path == FDTD_PATH_FUSED && n_src <= FDTD_FUSED_MAX_SRC && n_det <= FDTD_FUSED_MAX_DET;
    const int K = g->ck_every;
    int rc = FDTD_OK;
    if (n_total == 0) return forward_core(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, nullptr, 0, 0, 0, 0, cuda_stream);
    if (n_total > g->desc.max_steps) return fail(FDTD_EINVAL, "fdtd_forward: need 0 <= n_steps <= max_steps");
    for (int a = 0; a < n_total && !rc; a += K) {
        const int b = std::min(n_total, a + K);
        if (a > 0) rc = copy_checkpoint(g, fields, fused, a, a / K, false, (cudaStream_t)cuda_stream);   // (state 0 is restored by zeroing psi: slot 0 holds the fields only)
        else CK(cudaMemcpyAsync(g->ckpt, fields, 6 * (size_t)g->G.nc * sizeof(float), cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
        if (!rc) rc = forward_core(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, nullptr, 0, a, b, n_total, cuda_stream);
    }
    if (!rc) g->recorded_steps = n_total;
    return rc;
}

extern "C" int fdtd_forward_td(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                               const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                               const fdtd_time_detector *td, int32_t n_td, int32_t n_steps, void *cuda_stream)
{
    return forward_impl(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, td, n_td, 0, n_steps, n_steps, cuda_stream);
}

extern "C" int fdtd_forward_range(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                                  const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                                  int32_t n_begin, int32_t n_end, int32_t n_total, void *cuda_stream)
{
    if (n_begin < 0 || n_end < n_begin || n_total < n_end) return fail(FDTD_EINVAL, "fdtd_forward_range: need 0 <= n_begin <= n_end <= n_total");
    if (g && n_begin != 0 && g->fwd_pos != n_begin) return fail(FDTD_ESTATE, "fdtd_forward_range: n_begin does not continue the previous range");
    return forward_impl(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, nullptr, 0, n_begin, n_end, n_total, cuda_stream);
}

// steps n_begin .. n_end-1 of a run of n_total steps (fdtd_forward: 0 .. n_steps-1)
static int forward_core(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                        const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                        const fdtd_time_detector *td, int32_t n_td, int n_begin, int n_end, int n_total, void *cuda_stream)
{
    const int n_steps = n_total;
    int rc = check_common(g, fields, inv_eps, src, n_src, det, n_det, n_steps, "fdtd_forward");
    if (rc) return rc;
    for (int s = 0; s < n_det; ++s)
        if (!det[s].phasor) return fail(FDTD_EINVAL, "fdtd_forward: detector phasor is NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Dims &G = g->G;
    std::vector<SourceDev> S;
    std::vector<DetectorDev> D;
    std::vector<TimeDetDev> TD;
    if ((rc = translate_td(g, td, n_td, n_steps, TD, "fdtd_forward_td"))) return rc;
    for (const TimeDetDev &q : TD) if (!q.out) return fail(FDTD_EINVAL, "fdtd_forward_td: time detector out is NULL");
    translate(src, n_src, S);
    const int total_freq = translate(det, n_det, D);
    const bool recording = (g->desc.record == 1 || g->desc.record == 2) && G.d > 0;
    g->recorded_steps = -1;
    g->fwd_pos = -1;
    if ((rc = upload_cs_table(g, det, n_det, total_freq, n_steps, st))) return rc;
    launch_set_step(g->d_step, n_begin, st);             // the first step of the call reads slot 0

    // more descriptors than the fused kernels' parameter block holds: this call runs on the generic kernels (same
    // psi slabs, same recorder layout, so a fused or generic fdtd_backward can follow)
    const bool fused_call = g->path == FDTD_PATH_FUSED && n_src <= FDTD_FUSED_MAX_SRC && n_det <= FDTD_FUSED_MAX_DET;
    if (g->path == FDTD_PATH_FUSED && !fused_call && g->desc.path == FDTD_PATH_FUSED)
        return fail(FDTD_EINVAL, "FDTD_PATH_FUSED takes at most 4 sources and 4 detectors per call (FDTD_PATH_AUTO falls back to the generic kernels)");
    if (g->sigma && recording) return fail(FDTD_ESTATE, "a lossy medium cannot be time-reversed (PAPER.md L84): use record = 0 or the checkpointed sweep, record = 3");
    if (!fused_call && (g->peer[0][0].vol[0] || g->peer[0][1].vol[0]))
        return fail(FDTD_ESTATE, "fdtd_forward: neighbours are attached (fdtd_halo_attach) but this call runs on the generic kernels");
    if (fused_call) {
        rc = fused_forward(g, fields, inv_eps, inv_mu, S, D, TD, total_freq, n_begin, n_end, n_total, recording, st);
        if (rc) return rc;
    } else {
        if (n_begin == 0 && ((rc = g->zero_psi(g->psiE[0], st)) || (rc = g->zero_psi(g->psiH[0], st)))) return rc;
        const int launches = 3 + n_src + n_det + n_td + (recording ? 1 : 0);
        std::string key = make_key("gf", fields, inv_eps, inv_mu, g->rec, g->d_cs, S, D, recording);
        if (!TD.empty()) key.append((const char *)TD.data(), TD.size() * sizeof(TimeDetDev));
        key.append((const char *)&g->sigma, sizeof(g->sigma));
        rc = run_steps(g, g->fwd_graph, key, n_end - n_begin, launches, st, [&](cudaStream_t cs) {
            { ProfScope p(g, fdtd_grid::PC_UPDATE_E, cs); launch_update_E(G, g->T, fields, inv_eps, g->psiE[0], cs, g->sigma); }
            { ProfScope p(g, fdtd_grid::PC_SRC_DET, cs);
              for (const SourceDev &s : S) if (s.comp < 3) launch_add_source(G, fields, s, g->step_in(), 1.f, cs); }
            if (recording) { ProfScope p(g, fdtd_grid::PC_RECORD, cs); launch_record(G, g->R, fields, fields, g->rec, g->step_in(), cs); }
            { ProfScope p(g, fdtd_grid::PC_UPDATE_H, cs); launch_update_H(G, g->T, fields, inv_mu, g->psiH[0], cs); }
            { ProfScope p(g, fdtd_grid::PC_SRC_DET, cs);
              for (const SourceDev &s : S) if (s.comp >= 3) launch_add_source(G, fields, s, g->step_in(), 1.f, cs);
              for (const DetectorDev &dt : D) launch_detector(G, fields, dt, g->d_cs, total_freq, g->step_in(), cs);
              for (const TimeDetDev &q : TD) launch_time_detect(G, fields, nullptr, 0, inv_eps, inv_mu, q, g->red, g->step_in(), cs); }
            { ProfScope p(g, fdtd_grid::PC_OTHER, cs); launch_next_step(g->step_in(), g->step_out(), 1, cs); }
        });
        if (rc) return rc;
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "fdtd_forward launch");
    g->fwd_pos = n_end;
    g->fwd_fused = fused_call;
    if (recording && n_end == n_total) g->recorded_steps = n_steps;
    return FDTD_OK;
}

// ================================================================================================
// backward
// ================================================================================================
int fdtd_grid::ensure_backward_buffers()
{
    if (lam) return FDTD_OK;
    int rc;
    if ((rc = alloc((void **)&lam, (size_t)G.nc * 6 * sizeof(float)))) return rc;
    for (int q = 0; q < 2; ++q)
        if ((rc = alloc_psi(lpsiE[q])) || (rc = alloc_psi(lpsiH[q]))) return rc;
    return fused ? fused_alloc_backward(this) : FDTD_OK;
}

extern "C" int fdtd_backward(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                             const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                             const float *const *dL_dphasor, const float *dL_dfields,
                             int32_t n_steps, float *dL_dinv_eps, float *dL_dfields0, void *cuda_stream)
{
    return fdtd_backward_td(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, nullptr, 0, nullptr, dL_dfields,
                            n_steps, dL_dinv_eps, dL_dfields0, cuda_stream);
}

static int backward_impl(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                         const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                         const float *const *dL_dphasor,
                         const fdtd_time_detector *td, int32_t n_td, const float *const *dL_dtd,
                         const float *dL_dfields, int n_hi, int n_lo, int n_total, float *dL_dinv_eps, float *dL_dfields0,
                         void *cuda_stream, float *dL_dinv_mu = nullptr);

extern "C" int fdtd_backward_mu(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                                const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                                const float *const *dL_dphasor, const float *dL_dfields,
                                int32_t n_steps, float *dL_dinv_eps, float *dL_dinv_mu, float *dL_dfields0, void *cuda_stream)
{
    if (dL_dinv_mu && !dL_dinv_eps) return fail(FDTD_EINVAL, "fdtd_backward_mu: dL_dinv_mu needs the reconstructed fields (request dL_dinv_eps too)");
    return backward_impl(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, nullptr, 0, nullptr, dL_dfields,
                         n_steps, 0, n_steps, dL_dinv_eps, dL_dfields0, cuda_stream, dL_dinv_mu);
}

extern "C" int fdtd_backward_td(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                                const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                                const float *const *dL_dphasor,
                                const fdtd_time_detector *td, int32_t n_td, const float *const *dL_dtd,
                                const float *dL_dfields, int32_t n_steps, float *dL_dinv_eps, float *dL_dfields0,
                                void *cuda_stream)
{
    return backward_impl(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, td, n_td, dL_dtd, dL_dfields,
                         n_steps, 0, n_steps, dL_dinv_eps, dL_dfields0, cuda_stream);
}

extern "C" int fdtd_backward_range(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                                   const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                                   const float *const *dL_dphasor, const float *dL_dfields,
                                   int32_t n_hi, int32_t n_lo, int32_t n_total, float *dL_dinv_eps, float *dL_dfields0,
                                   void *cuda_stream)
{
    if (n_lo < 0 || n_hi < n_lo || n_total < n_hi) return fail(FDTD_EINVAL, "fdtd_backward_range: need 0 <= n_lo <= n_hi <= n_total");
    if (g && n_hi != n_total && g->bwd_pos != n_hi) return fail(FDTD_ESTATE, "fdtd_backward_range: n_hi does not continue the previous range");
    return backward_impl(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, nullptr, 0, nullptr, dL_dfields,
                         n_hi, n_lo, n_total, dL_dinv_eps, dL_dfields0, cuda_stream);
}

static int backward_core(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                         const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                         const float *const *dL_dphasor,
                         const fdtd_time_detector *td, int32_t n_td, const float *const *dL_dtd,
                         const float *dL_dfields, int n_hi, int n_lo, int n_total, float *dL_dinv_eps, float *dL_dfields0,
                         void *cuda_stream, float *dL_dinv_mu, bool sweep_only);

// record = 3: the reverse sweep from checkpoints, segment by segment from the last one --
// restore the checkpoint, run the segment's forward steps again keeping dE = E' - E (sources subtracted) on the gradient box,
// then the segment's adjoint steps, each followed by g += sum_c lamE'_c dE_c / inv_eps.  No inverse step.
static int checkpointed_backward(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                                 const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                                 const float *const *dL_dphasor, const float *dL_dfields, int n_total,
                                 float *dL_dinv_eps, float *dL_dfields0, void *cuda_stream)
{
    const Dims &G = g->G;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (g->recorded_steps != n_total) return fail(FDTD_ESTATE, "fdtd_backward: no matching checkpointed forward (need record=3 and the same n_steps)");
    std::vector<SourceDev> S;
    translate(src, n_src, S);
    const bool fused_f = g->path == FDTD_PATH_FUSED && n_src <= FDTD_FUSED_MAX_SRC;      // the replay runs without detectors
    const size_t vol = (size_t)G.nc * sizeof(float);
    CK(cudaMemsetAsync(dL_dinv_eps, 0, (G.aniso ? 3 : 1) * vol, st));
    const int K = g->ck_every;
    int rc = FDTD_OK;
    const bool fused_b = g->path == FDTD_PATH_FUSED && g->fused_backward_ready && (!g->sigma || g->e2buf);
    for (int a = (n_total - 1) / K * K; a >= 0 && n_total > 0; a -= K) {
        const int b = std::min(n_total, a + K);
        // ---- the segment's forward steps again, from its checkpoint
        if (a > 0) { if ((rc = copy_checkpoint(g, fields, fused_f, a, a / K, true, st))) return rc; }
        else CK(cudaMemcpyAsync(fields, g->ckpt, 6 * vol, cudaMemcpyDeviceToDevice, st));
        if (fused_f) {
            // one call for the segment: the D store runs after every step inside the replayed graph (enqueue_fwd)
            g->replaying = true; g->ck_store = true;
            rc = forward_core(g, fields, inv_eps, inv_mu, src, n_src, nullptr, 0, nullptr, 0, a, b, n_total, st);
            g->replaying = false; g->ck_store = false;
            if (rc) return rc;
        } else {
            for (int n = a; n < b; ++n) {
                // in-place step: E before it (the counter slot the step will read), D after it
                launch_set_step(g->d_step, n, st);
                launch_dE_store(G, fields, nullptr, g->dE, K, 1, inv_eps, g->sigma, g->d_step, st);
                g->replaying = true;
                rc = forward_core(g, fields, inv_eps, inv_mu, src, n_src, nullptr, 0, nullptr, 0, n, n + 1, n_total, st);
                g->replaying = false;
                if (rc) return rc;
                // the step's first launch read n from counter slot 0, which still holds it
                launch_dE_store(G, fields, nullptr, g->dE, K, 2, inv_eps, g->sigma, g->d_step, st);
                for (const SourceDev &q : S) if (q.comp < 3) launch_dE_source(G, g->dE, K, q, inv_eps, g->sigma, g->d_step, st);
                g->kernel_launches += 4;
            }
        }
        // ---- the segment's adjoint steps, gradient from the stored D
        if (fused_b) {
            // one call for the segment: g += lamE' . D runs after every adjoint step inside the replayed graph (enqueue_bwd)
            g->ck_gradhook = dL_dinv_eps;
            g->ck_e2 = g->sigma ? g->e2buf : nullptr;
            rc = backward_core(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, nullptr, 0, nullptr, dL_dfields,
                               b, a, n_total, nullptr, dL_dfields0, st, nullptr, true);
            g->ck_gradhook = nullptr; g->ck_e2 = nullptr;
            if (rc) return rc;
        } else {
            for (int n = b - 1; n >= a; --n) {       // generic path: the gradient kernel sits between its two adjoint kernels
                g->ck_grad = dL_dinv_eps;
                rc = backward_core(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, nullptr, 0, nullptr, dL_dfields,
                                   n + 1, n, n_total, nullptr, dL_dfields0, st, nullptr, true);
                g->ck_grad = nullptr;
                if (rc) return rc;
            }
        }
    }
    // (`fields` was the replay's scratch: it ends at the state the first segment's replay left)
    g->recorded_steps = n_total;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "fdtd_backward launch");
    return FDTD_OK;
}

static int backward_impl(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                         const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                         const float *const *dL_dphasor,
                         const fdtd_time_detector *td, int32_t n_td, const float *const *dL_dtd,
                         const float *dL_dfields, int n_hi, int n_lo, int n_total, float *dL_dinv_eps, float *dL_dfields0,
                         void *cuda_stream, float *dL_dinv_mu)
{
    if (g && g->desc.record == 3 && dL_dinv_eps) {
        int rc = check_common(g, fields, inv_eps, src, n_src, det, n_det, n_total, "fdtd_backward");
        if (rc) return rc;
        if (n_td || dL_dinv_mu) return fail(FDTD_EINVAL, "time-domain detectors and dL_dinv_mu are not available on a record = 3 grid");
        if (n_hi != n_total || n_lo != 0) return fail(FDTD_EINVAL, "range calls are not available on a record = 3 grid");
        return checkpointed_backward(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, dL_dfields, n_total,
                                     dL_dinv_eps, dL_dfields0, cuda_stream);
    }
    return backward_core(g, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, td, n_td, dL_dtd, dL_dfields, n_hi, n_lo,
                         n_total, dL_dinv_eps, dL_dfields0, cuda_stream, dL_dinv_mu, false);
}

// reverse steps n_hi-1 .. n_lo of a run of n_total steps (fdtd_backward: n_steps-1 .. 0); the cotangent seed (B0) is
// placed by the call with n_hi == n_total, dL_dfields0 is written by the call with n_lo == 0
static int backward_core(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                         const fdtd_source *src, int32_t n_src, const fdtd_detector *det, int32_t n_det,
                         const float *const *dL_dphasor,
                         const fdtd_time_detector *td, int32_t n_td, const float *const *dL_dtd,
                         const float *dL_dfields, int n_hi, int n_lo, int n_total, float *dL_dinv_eps, float *dL_dfields0,
                         void *cuda_stream, float *dL_dinv_mu, bool sweep_only)
{
    const int n_steps = n_total;
    const bool first = n_hi == n_total, last = n_lo == 0;
    int rc = check_common(g, fields, inv_eps, src, n_src, det, n_det, n_steps, "fdtd_backward");
    if (rc) return rc;
    if (!dL_dinv_eps && !dL_dfields0 && !sweep_only) return fail(FDTD_EINVAL, "fdtd_backward: dL_dinv_eps or dL_dfields0 is required");
    const Dims &G = g->G;
    if (dL_dinv_eps && G.d > 0 && (!g->desc.record || g->recorded_steps != n_steps))
        return fail(FDTD_ESTATE, "fdtd_backward: no matching recorded forward (need record=1 and the same n_steps)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    std::vector<SourceDev> S;
    std::vector<DetectorDev> D;
    // time-domain detectors: only those with a cotangent take part; `out` carries the cotangent from here on
    std::vector<TimeDetDev> TDall, TD;
    if ((rc = translate_td(g, td, n_td, n_steps, TDall, "fdtd_backward_td"))) return rc;
    for (int s = 0; s < n_td; ++s) {
        if (!dL_dtd || !dL_dtd[s]) continue;
        TimeDetDev q = TDall[s];
        q.out = const_cast<float *>(dL_dtd[s]);
        if (q.kind == FDTD_TD_ENERGY) {
            if (!dL_dinv_eps) return fail(FDTD_EINVAL, "fdtd_backward_td: the energy detector's transpose needs the reconstructed fields (request dL_dinv_eps)");
            for (int a = 0; a < 3; ++a)
                if (q.lo[a] < G.lo[a] || q.hi[a] > G.hi[a]) return fail(FDTD_EINVAL, "fdtd_backward_td: energy detector box outside the reconstruction box");
        }
        TD.push_back(q);
    }
    translate(src, n_src, S);
    const int total_freq = translate(det, n_det, D);
    for (int s = 0; s < n_det; ++s)
        D[s].phasor = const_cast<float *>(dL_dphasor ? dL_dphasor[s] : nullptr);
    if ((rc = g->ensure_backward_buffers())) return rc;
    if ((rc = upload_cs_table(g, det, n_det, total_freq, n_steps, st))) return rc;

    // B0: seed cotangents
    const size_t vol = (size_t)G.nc * sizeof(float);
    g->bwd_pos = -1;
    const bool fused_call = g->path == FDTD_PATH_FUSED && g->fused_backward_ready && (!g->sigma || !sweep_only || g->ck_e2);
    if (first) {
        // the fused sweep ping-pongs: the cotangent of state n lives in volume n&1, so the seed goes where state n_steps lives
        if (fused_call && (rc = fused_alloc_backward(g))) return rc;
        float *seed = fused_call ? fused_volume(g, fields, 1, n_steps) : g->lam;
        if (dL_dfields) CK(cudaMemcpyAsync(seed, dL_dfields, 6 * vol, cudaMemcpyDeviceToDevice, st));
        else            CK(cudaMemsetAsync(seed, 0, 6 * vol, st));
        for (int q = 0; q < 2; ++q)
            if ((rc = g->zero_psi(g->lpsiE[q], st)) || (rc = g->zero_psi(g->lpsiH[q], st))) return rc;
        if (dL_dinv_eps) CK(cudaMemsetAsync(dL_dinv_eps, 0, (G.aniso ? 3 : 1) * vol, st));
        if (dL_dinv_mu) CK(cudaMemsetAsync(dL_dinv_mu, 0, vol, st));
    }
    launch_set_step(g->d_step, std::max(n_hi - 1, 0), st);      // the first reverse step of the call reads slot 0
    const bool want_grad = dL_dinv_eps != nullptr;              // false: adjoint sweep only (B1, B2, B5)
    if (g->sigma && want_grad) return fail(FDTD_ESTATE, "a lossy medium cannot be time-reversed (PAPER.md L84): its gradient comes from the checkpointed sweep (record = 3)");

    if (!fused_call && (g->peer[1][0].vol[0] || g->peer[1][1].vol[0]))
        return fail(FDTD_ESTATE, "fdtd_backward: neighbours are attached (fdtd_halo_attach) but this call runs on the generic kernels");
    if (fused_call) {
        // seeded_H: the H part of the seed can be non-zero (it is scaled by inv_mu for the sweep)
        rc = fused_backward(g, fields, inv_eps, inv_mu, S, D, TD, total_freq, n_hi, n_lo, n_total, dL_dinv_eps, dL_dfields != nullptr, st, dL_dinv_mu);
        if (rc) return rc;
        // the fused sweep carried im lamH in the H part (kernels_step.cu); the cotangent of state 0 is lamH
        if (last && inv_mu && dL_dfields0) launch_scale_H(G, g->lam, inv_mu, true, st);
    } else {
        int n_adj = 0;
        for (const DetectorDev &dt : D) if (dt.phasor) ++n_adj;
        const int launches = (want_grad ? 5 + n_adj + n_src + (G.d > 0 ? 1 : 0) : 3 + n_adj) + (int)TD.size() + (g->ck_grad ? 1 : 0) + (g->sigma ? 1 : 0);
        std::string key = make_key("gb", fields, inv_eps, inv_mu, g->rec, dL_dinv_eps, S, D, 0);
        key.append((const char *)&g->d_cs, sizeof(g->d_cs));
        key.append((const char *)&dL_dinv_mu, sizeof(dL_dinv_mu));
        key.append((const char *)&g->sigma, sizeof(g->sigma));
        key.append((const char *)&g->ck_grad, sizeof(g->ck_grad));
        if (!TD.empty()) key.append((const char *)TD.data(), TD.size() * sizeof(TimeDetDev));
        rc = run_steps(g, g->bwd_graph, key, n_hi - n_lo, launches, st, [&](cudaStream_t cs) {
            { ProfScope p(g, fdtd_grid::PC_SRC_DET, cs);
              // N2 transposes first: they act on the state after step n, before anything of reverse step n
              for (const TimeDetDev &q : TD)
                  launch_time_detect_adjoint(G, g->lam, nullptr, fields, nullptr, 0, inv_eps, inv_mu, false, q, dL_dinv_eps, g->step_in(), cs);
              for (const DetectorDev &dt : D) if (dt.phasor) launch_detector_adjoint(G, g->lam, dt, g->d_cs, total_freq, g->step_in(), cs); }
            { ProfScope p(g, fdtd_grid::PC_ADJ_H, cs); launch_adj_H(G, g->T, g->lam, inv_mu, g->lpsiH[0], g->lpsiH[1], g->step_in(), cs); }
            if (want_grad) {
            { ProfScope p(g, fdtd_grid::PC_SRC_DET, cs);
              for (const SourceDev &s : S) if (s.comp >= 3) launch_add_source(G, fields, s, g->step_in(), -1.f, cs); }
            if (G.d > 0) { ProfScope p(g, fdtd_grid::PC_INJECT, cs); launch_inject(G, g->R, fields, g->rec, g->step_in(), cs); }
            { ProfScope p(g, fdtd_grid::PC_INV_H, cs); launch_inv_H(G, fields, inv_mu, cs, g->lam, nullptr, nullptr, false, dL_dinv_mu); }
            { ProfScope p(g, fdtd_grid::PC_SRC_DET, cs);
              for (const SourceDev &s : S) if (s.comp < 3) launch_add_source(G, fields, s, g->step_in(), -1.f, cs); }
            { ProfScope p(g, fdtd_grid::PC_INV_E_GRAD, cs); launch_inv_E_grad(G, fields, inv_eps, g->lam, dL_dinv_eps, cs); }
            }
            // checkpointed sweep (record = 3): the gradient from the replay's D = dE'/d inv_eps, with lamE' as it stands here
            if (g->ck_grad) { ProfScope p(g, fdtd_grid::PC_INV_E_GRAD, cs);
              launch_grad_from_dE(G, g->lam, nullptr, g->dE, g->ck_every, g->ck_grad, g->step_in(), cs); }
            { ProfScope p(g, fdtd_grid::PC_ADJ_E, cs); launch_adj_E(G, g->T, g->lam, inv_eps, g->lpsiE[0], g->lpsiE[1], g->step_in(), cs, g->sigma); }
            { ProfScope p(g, fdtd_grid::PC_OTHER, cs); launch_next_step(g->step_in(), g->step_out(), -1, cs); }
        });
        if (rc) return rc;
    }
    if (last && dL_dfields0) CK(cudaMemcpyAsync(dL_dfields0, g->lam, 6 * vol, cudaMemcpyDeviceToDevice, st));
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "fdtd_backward launch");
    g->bwd_pos = n_lo;
    g->bwd_fused = fused_call;
    return FDTD_OK;
}

extern "C" int fdtd_set_conductivity(fdtd_grid *g, const float *sigma)
{
    if (!g) return fail(FDTD_EINVAL, "fdtd_set_conductivity: NULL grid");
    if (sigma && (g->desc.record == 1 || g->desc.record == 2))
        return fail(FDTD_ESTATE, "a lossy medium cannot be time-reversed (PAPER.md L84): create the grid with record = 0 or record = 3");
    // fused record = 3 grid: the lossy adjoint step leaves lamE' (before its scaling by Ca) in three scratch volumes for the
    // checkpointed sweep's gradient; allocated by the first call that sets a conductivity
    if (sigma && g->desc.record == 3 && g->path == FDTD_PATH_FUSED && !g->e2buf) {
        int rc = g->alloc((void **)&g->e2buf, 3 * (size_t)g->G.nc * sizeof(float));
        if (rc) return rc;
    }
    g->sigma = sigma;
    return FDTD_OK;
}

extern "C" int fdtd_grad_rho(fdtd_grid *g, const float *dL_dinv_eps, const float *inv_eps, float delta_eps,
                             const int32_t lo[3], const int32_t hi[3], float *dL_drho, void *cuda_stream)
{
    if (!g || !dL_dinv_eps || !inv_eps || !lo || !hi || !dL_drho) return fail(FDTD_EINVAL, "fdtd_grad_rho: NULL argument");
    if (!box_ok(g->G, lo, hi)) return fail(FDTD_EINVAL, "fdtd_grad_rho: box outside the grid or empty");
    if (g->G.aniso) return fail(FDTD_EINVAL, "fdtd_grad_rho is stated for one inv_eps per voxel (no FDTD_FLAG_ANISO_EPS)");
    launch_grad_rho(g->G, dL_dinv_eps, inv_eps, delta_eps, lo, hi, dL_drho, (cudaStream_t)cuda_stream);
    g->kernel_launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "fdtd_grad_rho launch");
    return FDTD_OK;
}

// ================================================================================================
// N3: halo planes of a z-slab sub-grid (include/fdtd.h "Domain decomposition")
// ================================================================================================
namespace {
// volume that holds state n: primal (which = 0) or cotangents (which = 1)
int halo_volume(fdtd_grid *g, float *fields, int which, int n, float **vol, const char *who)
{
    if (!g) return fail(FDTD_EINVAL, std::string(who) + ": NULL grid");
    if (which != 0 && which != 1) return fail(FDTD_EINVAL, std::string(who) + ": which must be 0 (fields) or 1 (cotangents)");
    if (which == 0 && !fields) return fail(FDTD_EINVAL, std::string(who) + ": fields is NULL");
    if (which == 1 && !g->lam) return fail(FDTD_ESTATE, std::string(who) + ": no cotangent volumes yet (call fdtd_backward_range first)");
    const bool fused = which == 0 ? g->fwd_fused : g->bwd_fused;
    *vol = fused ? fused_volume(g, fields, which, n) : (which == 0 ? fields : g->lam);
    return FDTD_OK;
}
}  // namespace

extern "C" int fdtd_halo_export(fdtd_grid *g, float *fields, int32_t which, int32_t n, int32_t side, float *out, void *cuda_stream)
{
    float *vol = nullptr;
    int rc = halo_volume(g, fields, which, n, &vol, "fdtd_halo_export");
    if (rc) return rc;
    if (!out || (side != 0 && side != 1)) return fail(FDTD_EINVAL, "fdtd_halo_export: bad argument");
    const Dims &G = g->G;
    const int k = side ? G.nz - 1 - g->desc.z_ghost_hi : g->desc.z_ghost_lo;        // highest / lowest owned plane
    const size_t plane = (size_t)G.nx * G.ny;
    for (int c = 0; c < 3; ++c)
        CK(cudaMemcpyAsync(out + c * plane, vol + (3 + c) * G.nc + (size_t)k * plane, plane * sizeof(float), cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
    return FDTD_OK;
}

extern "C" int fdtd_halo_import(fdtd_grid *g, float *fields, int32_t which, int32_t n, int32_t side, const float *in, void *cuda_stream)
{
    float *vol = nullptr;
    int rc = halo_volume(g, fields, which, n, &vol, "fdtd_halo_import");
    if (rc) return rc;
    if (!in || (side != 0 && side != 1)) return fail(FDTD_EINVAL, "fdtd_halo_import: bad argument");
    if (side ? !g->desc.z_ghost_hi : !g->desc.z_ghost_lo) return fail(FDTD_EINVAL, "fdtd_halo_import: the grid has no ghost plane on that side");
    const Dims &G = g->G;
    const int k = side ? G.nz - 1 : 0;
    const size_t plane = (size_t)G.nx * G.ny;
    for (int c = 0; c < 3; ++c)
        CK(cudaMemcpyAsync(vol + (3 + c) * G.nc + (size_t)k * plane, in + c * plane, plane * sizeof(float), cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
    return FDTD_OK;
}

// N3 peer stores: the step kernels write the halo planes into the neighbour's volumes themselves
extern "C" int fdtd_halo_volumes(fdtd_grid *g, float *fields, int32_t which, float **vol0, float **vol1)
{
    if (!g || !vol0 || !vol1) return fail(FDTD_EINVAL, "fdtd_halo_volumes: NULL argument");
    if (which != 0 && which != 1) return fail(FDTD_EINVAL, "fdtd_halo_volumes: which must be 0 (fields) or 1 (cotangents)");
    if (g->path != FDTD_PATH_FUSED) return fail(FDTD_ESTATE, "fdtd_halo_volumes: peer stores run on the fused kernels only (this grid: " + g->fused_why_not + ")");
    if (which == 0 && !fields) return fail(FDTD_EINVAL, "fdtd_halo_volumes: fields is NULL");
    if (which == 1) {
        if (!g->fused_backward_ready) return fail(FDTD_ESTATE, "fdtd_halo_volumes: this grid's reverse sweep runs on the generic kernels");
        int rc = g->ensure_backward_buffers();
        if (rc) return rc;
    }
    *vol0 = fused_volume(g, fields, which, 0);
    *vol1 = fused_volume(g, fields, which, 1);
    return FDTD_OK;
}

extern "C" int fdtd_halo_attach(fdtd_grid *g, int32_t which, int32_t side, float *peer_vol0, float *peer_vol1, int32_t peer_nz)
{
    if (!g) return fail(FDTD_EINVAL, "fdtd_halo_attach: NULL grid");
    if ((which != 0 && which != 1) || (side != 0 && side != 1)) return fail(FDTD_EINVAL, "fdtd_halo_attach: which and side must be 0 or 1");
    fdtd_grid::PeerLink &L = g->peer[which][side];
    if (!peer_vol0 && !peer_vol1) { L = fdtd_grid::PeerLink{}; return FDTD_OK; }      // detach (the flag too)
    if (!peer_vol0 || !peer_vol1) return fail(FDTD_EINVAL, "fdtd_halo_attach: both volumes of the neighbour are needed");
    if (g->path != FDTD_PATH_FUSED || (which == 1 && !g->fused_backward_ready))
        return fail(FDTD_ESTATE, "fdtd_halo_attach: peer stores run on the fused kernels only");
    if (side ? !g->desc.z_ghost_hi : !g->desc.z_ghost_lo) return fail(FDTD_EINVAL, "fdtd_halo_attach: the grid has no cut on that side");
    if (peer_nz < 3) return fail(FDTD_EINVAL, "fdtd_halo_attach: peer_nz is the neighbour's local plane count (>= 3: a ghost plane, an owned plane, ...)");
    // my lowest owned plane is the neighbour-below's ghost plane above (its last local plane); my highest owned plane is
    // the neighbour-above's ghost plane below (its local plane 0)
    const size_t plane = (size_t)g->G.nx * g->G.ny;
    const long long pnc = (long long)peer_nz * (long long)plane;
    const size_t k = side ? 0 : (size_t)peer_nz - 1;
    L.vol[0] = peer_vol0 + 3 * pnc + k * plane;
    L.vol[1] = peer_vol1 + 3 * pnc + k * plane;
    L.nc = pnc;
    return FDTD_OK;
}

// device-side ordering of the slabs (halo_sync.cu)
extern "C" int fdtd_halo_flags(fdtd_grid *g, int32_t which, int32_t **flags)
{
    if (!g || !flags) return fail(FDTD_EINVAL, "fdtd_halo_flags: NULL argument");
    if (which != 0 && which != 1) return fail(FDTD_EINVAL, "fdtd_halo_flags: which must be 0 (fields) or 1 (cotangents)");
    if (g->path != FDTD_PATH_FUSED) return fail(FDTD_ESTATE, "fdtd_halo_flags: peer stores run on the fused kernels only");
    if (!g->d_hflags) {
        int rc = g->alloc((void **)&g->d_hflags, 5 * sizeof(int));       // [which][side] + the error flag
        if (rc) return rc;
        CK(cudaMemset(g->d_hflags, 0xff, 4 * sizeof(int)));               // -1: no state reached yet
        CK(cudaMemset(g->d_hflags + 4, 0, sizeof(int)));
        g->d_herr = g->d_hflags + 4;
    }
    *flags = g->d_hflags + which * 2;
    return FDTD_OK;
}

extern "C" int fdtd_halo_attach_flags(fdtd_grid *g, int32_t which, int32_t side, int32_t *peer_flags)
{
    if (!g) return fail(FDTD_EINVAL, "fdtd_halo_attach_flags: NULL grid");
    if ((which != 0 && which != 1) || (side != 0 && side != 1)) return fail(FDTD_EINVAL, "fdtd_halo_attach_flags: which and side must be 0 or 1");
    fdtd_grid::PeerLink &L = g->peer[which][side];
    if (!peer_flags) { L.flag = nullptr; return FDTD_OK; }
    if (!L.vol[0]) return fail(FDTD_ESTATE, "fdtd_halo_attach_flags: attach the neighbour's volumes first (fdtd_halo_attach)");
    if (!g->d_hflags) return fail(FDTD_ESTATE, "fdtd_halo_attach_flags: call fdtd_halo_flags first (the neighbour needs this grid's flags too)");
    // the neighbour below keeps the flag I write in its slot "above" (1); the neighbour above in its slot "below" (0)
    L.flag = peer_flags + (side == 0 ? 1 : 0);
    return FDTD_OK;
}

extern "C" int fdtd_halo_sync_error(fdtd_grid *g, int32_t *timed_out)
{
    if (!g || !timed_out) return fail(FDTD_EINVAL, "fdtd_halo_sync_error: NULL argument");
    *timed_out = 0;
    if (!g->d_herr) return FDTD_OK;
    int v = 0;
    CK(cudaMemcpy(&v, g->d_herr, sizeof(int), cudaMemcpyDeviceToHost));
    if (v) CK(cudaMemset(g->d_herr, 0, sizeof(int)));
    *timed_out = v;
    return FDTD_OK;
}

// cudaIpc* behind the ABI, so that a binding needs no CUDA API of its own to hand a volume to another process
extern "C" int fdtd_ipc_export(const void *dev_ptr, uint8_t handle[64], int64_t *offset)
{
    if (!dev_ptr || !handle || !offset) return fail(FDTD_EINVAL, "fdtd_ipc_export: NULL argument");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "cudaIpcMemHandle_t is 64 bytes");
    cudaIpcMemHandle_t h;
    CK(cudaIpcGetMemHandle(&h, const_cast<void *>(dev_ptr)));
    // the handle names the whole allocation; the pointer may sit inside it (a caching allocator's block)
    typedef int (*range_fn)(unsigned long long *, size_t *, unsigned long long);      // CUresult cuMemGetAddressRange(CUdeviceptr *, size_t *, CUdeviceptr)
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn)
        return fail(FDTD_ECUDA, "fdtd_ipc_export: cuMemGetAddressRange is not available");
    unsigned long long base = 0;
    size_t size = 0;
    if (((range_fn)fn)(&base, &size, (unsigned long long)(uintptr_t)dev_ptr) != 0) return fail(FDTD_ECUDA, "fdtd_ipc_export: cuMemGetAddressRange failed");
    memcpy(handle, &h, 64);
    *offset = (int64_t)((unsigned long long)(uintptr_t)dev_ptr - base);
    return FDTD_OK;
}

extern "C" int fdtd_ipc_open(const uint8_t handle[64], int64_t offset, void **dev_ptr)
{
    if (!handle || !dev_ptr || offset < 0) return fail(FDTD_EINVAL, "fdtd_ipc_open: bad argument");
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, 64);
    void *base = nullptr;
    CK(cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess));
    *dev_ptr = (char *)base + offset;
    return FDTD_OK;
}

extern "C" int fdtd_ipc_close(void *dev_ptr, int64_t offset)
{
    if (!dev_ptr) return FDTD_OK;
    CK(cudaIpcCloseMemHandle((char *)dev_ptr - offset));
    return FDTD_OK;
}

// ================================================================================================
// N2: flux from phasors, TFSF plane source (kernels_n2.cu)
// ================================================================================================
namespace {
int flux_common(fdtd_grid *g, const fdtd_detector *det, const float *phasor, int axis, int interpolate, DetectorDev &dt, const char *who)
{
    if (!g || !det || !phasor) return fail(FDTD_EINVAL, std::string(who) + ": NULL argument");
    if (axis < 0 || axis > 2) return fail(FDTD_EINVAL, std::string(who) + ": axis must be 0..2");
    if (det->component_mask <= 0 || det->component_mask > 63 || !box_ok(g->G, det->lo, det->hi) || det->n_freq < 1 || !det->omega)
        return fail(FDTD_EINVAL, std::string(who) + ": bad detector descriptor");
    std::vector<DetectorDev> D;
    translate(det, 1, D);
    dt = D[0];
    const int b = (axis + 1) % 3, c = (axis + 2) % 3;
    const int need = (1 << b) | (1 << c) | (1 << (3 + b)) | (1 << (3 + c));
    if ((dt.mask & need) != need) return fail(FDTD_EINVAL, std::string(who) + ": the detector lacks a tangential component of the plane");
    if (dt.hi[axis] - dt.lo[axis] != (interpolate ? 2 : 1))
        return fail(FDTD_EINVAL, std::string(who) + ": the box must be 1 plane thick along the axis (2 with interpolation)");
    return FDTD_OK;
}
}  // namespace

extern "C" int fdtd_flux(fdtd_grid *g, const fdtd_detector *det, const float *phasor, int32_t axis, int32_t interpolate,
                         float *flux, void *cuda_stream)
{
    DetectorDev dt;
    int rc = flux_common(g, det, phasor, axis, interpolate, dt, "fdtd_flux");
    if (rc) return rc;
    if (!flux) return fail(FDTD_EINVAL, "fdtd_flux: flux is NULL");
    for (int f = 0; f < dt.n_freq; ++f)
        launch_flux(dt, phasor, axis, interpolate ? 1 : 0, f, (float)std::cos(0.5 * (double)det->omega[f]),
                    (float)std::sin(0.5 * (double)det->omega[f]), flux, g->red, (cudaStream_t)cuda_stream);
    g->kernel_launches += dt.n_freq;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "fdtd_flux launch");
    return FDTD_OK;
}

extern "C" int fdtd_flux_vjp(fdtd_grid *g, const fdtd_detector *det, const float *phasor, int32_t axis, int32_t interpolate,
                             const float *dL_dflux, float *dL_dphasor, void *cuda_stream)
{
    DetectorDev dt;
    int rc = flux_common(g, det, phasor, axis, interpolate, dt, "fdtd_flux_vjp");
    if (rc) return rc;
    if (!dL_dflux || !dL_dphasor) return fail(FDTD_EINVAL, "fdtd_flux_vjp: NULL argument");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t bytes = (size_t)dt.n_freq * dt.ncomp * (size_t)(dt.hi[0] - dt.lo[0]) * (dt.hi[1] - dt.lo[1]) * (dt.hi[2] - dt.lo[2]) * 2 * sizeof(float);
    CK(cudaMemsetAsync(dL_dphasor, 0, bytes, st));
    for (int f = 0; f < dt.n_freq; ++f)
        launch_flux_vjp(dt, phasor, axis, interpolate ? 1 : 0, f, (float)std::cos(0.5 * (double)det->omega[f]),
                        (float)std::sin(0.5 * (double)det->omega[f]), dL_dflux, dL_dphasor, st);
    g->kernel_launches += dt.n_freq;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "fdtd_flux_vjp launch");
    return FDTD_OK;
}

extern "C" int fdtd_tfsf_plane(float courant, float eps_r, float mu_r, int32_t axis, int32_t pol, int32_t dir, int32_t n_steps,
                               const float *base, float *wE, float *wH, int32_t *h_component, int32_t *h_plane_offset,
                               void *cuda_stream)
{
    if (axis < 0 || axis > 2 || pol < 0 || pol > 2 || pol == axis || (dir != 1 && dir != -1))
        return fail(FDTD_EINVAL, "fdtd_tfsf_plane: need axis, pol in 0..2, pol != axis, dir = +1 or -1");
    if (!(courant > 0.f) || !(eps_r > 0.f) || !(mu_r > 0.f)) return fail(FDTD_EINVAL, "fdtd_tfsf_plane: courant, eps_r, mu_r must be > 0");
    if (n_steps < 0 || n_steps > 50000) return fail(FDTD_EINVAL, "fdtd_tfsf_plane: need 0 <= n_steps <= 50000");
    if (n_steps && (!base || !wE || !wH)) return fail(FDTD_EINVAL, "fdtd_tfsf_plane: NULL argument");
    const int c = 3 - axis - pol;
    const float sgn = (axis == (pol + 1) % 3) ? 1.f : -1.f;
    if (h_component) *h_component = 3 + c;
    if (h_plane_offset) *h_plane_offset = dir > 0 ? -1 : 0;
    if (n_steps == 0) return FDTD_OK;
    cudaError_t e = launch_tfsf_aux(courant, 1.f / eps_r, 1.f / mu_r, sgn, dir > 0 ? 1.f : -1.f, n_steps, base, wE, wH,
                                    (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "fdtd_tfsf_plane launch");
    return FDTD_OK;
}

// ================================================================================================
// host-buffer entry points (end-to-end measurement): stage through grid-owned device buffers
// ================================================================================================
namespace {

struct HostStage {
    std::vector<fdtd_source> src;
    std::vector<fdtd_detector> det;
    std::vector<size_t> phasor_bytes;
};

size_t box_cells(const int32_t lo[3], const int32_t hi[3])
{
    return (size_t)(hi[0] - lo[0]) * (hi[1] - lo[1]) * (hi[2] - lo[2]);
}

}  // namespace

int fdtd_grid::ensure_host_buffers(bool need_mu, bool need_grad)
{
    int rc;
    const size_t vol = (size_t)G.nc * sizeof(float);
    if (!hb_fields && (rc = alloc((void **)&hb_fields, 6 * vol))) return rc;
    if (!hb_ie && (rc = alloc((void **)&hb_ie, vol))) return rc;
    if (need_mu && !hb_im && (rc = alloc((void **)&hb_im, vol))) return rc;
    if (need_grad && !hb_grad && (rc = alloc((void **)&hb_grad, vol))) return rc;
    return FDTD_OK;
}

// copies the descriptor payloads (profiles, waveforms, phasors) to device scratch; grows on demand
static int stage_descriptors(fdtd_grid *g, const fdtd_source *h_src, int n_src, const fdtd_detector *h_det, int n_det,
                             int n_steps, bool copy_phasors_in, const float *const *h_cot, HostStage &hs, cudaStream_t st)
{
    size_t need = 0;
    auto pad = [](size_t b) { return (b + 255) / 256 * 256; };
    for (int s = 0; s < n_src; ++s) {
        if (h_src[s].profile) need += pad(box_cells(h_src[s].lo, h_src[s].hi) * sizeof(float));
        need += pad((size_t)n_steps * sizeof(float));
    }
    hs.phasor_bytes.resize(n_det);
    for (int s = 0; s < n_det; ++s) {
        hs.phasor_bytes[s] = (size_t)h_det[s].n_freq * popcount6(h_det[s].component_mask) * box_cells(h_det[s].lo, h_det[s].hi) * 2 * sizeof(float);
        need += 2 * pad(hs.phasor_bytes[s]);
    }
    if (need > g->hb_desc_cap) {
        int rc = g->alloc((void **)&g->hb_desc, need);
        if (rc) return rc;
        g->hb_desc_cap = need;
    }
    char *cur = (char *)g->hb_desc;
    hs.src.assign(h_src, h_src + n_src);
    hs.det.assign(h_det, h_det + n_det);
    for (int s = 0; s < n_src; ++s) {
        if (h_src[s].profile) {
            const size_t b = box_cells(h_src[s].lo, h_src[s].hi) * sizeof(float);
            CK(cudaMemcpyAsync(cur, h_src[s].profile, b, cudaMemcpyHostToDevice, st));
            hs.src[s].profile = (const float *)cur; cur += pad(b);
        }
        const size_t b = (size_t)n_steps * sizeof(float);
        if (b) CK(cudaMemcpyAsync(cur, h_src[s].waveform, b, cudaMemcpyHostToDevice, st));
        hs.src[s].waveform = (const float *)cur; cur += pad(b);
    }
    g->hb_cot.assign(n_det, nullptr);
    for (int s = 0; s < n_det; ++s) {
        const size_t b = hs.phasor_bytes[s];
        hs.det[s].phasor = (float *)cur;
        if (copy_phasors_in && h_det[s].phasor) CK(cudaMemcpyAsync(cur, h_det[s].phasor, b, cudaMemcpyHostToDevice, st));
        cur += pad(b);
        if (h_cot && h_cot[s]) {
            CK(cudaMemcpyAsync(cur, h_cot[s], b, cudaMemcpyHostToDevice, st));
            g->hb_cot[s] = (const float *)cur;
        }
        cur += pad(b);
    }
    return FDTD_OK;
}

extern "C" int fdtd_forward_host(fdtd_grid *g, float *h_fields, const float *h_inv_eps, const float *h_inv_mu,
                                 const fdtd_source *h_src, int32_t n_src, const fdtd_detector *h_det, int32_t n_det,
                                 int32_t n_steps, void *cuda_stream)
{
    if (!g) return fail(FDTD_EINVAL, "fdtd_forward_host: NULL grid");
    if (!h_inv_eps) return fail(FDTD_EINVAL, "fdtd_forward_host: inv_eps is required");
    if (n_steps < 0 || n_steps > g->desc.max_steps) return fail(FDTD_EINVAL, "fdtd_forward_host: need 0 <= n_steps <= max_steps");
    if (n_src < 0 || n_det < 0 || (n_src && !h_src) || (n_det && !h_det)) return fail(FDTD_EINVAL, "fdtd_forward_host: bad descriptor arrays");
    for (int s = 0; s < n_src; ++s) if (!box_ok(g->G, h_src[s].lo, h_src[s].hi) || !h_src[s].waveform) return fail(FDTD_EINVAL, "fdtd_forward_host: bad source");
    for (int s = 0; s < n_det; ++s) if (!box_ok(g->G, h_det[s].lo, h_det[s].hi) || !h_det[s].phasor || h_det[s].n_freq < 1) return fail(FDTD_EINVAL, "fdtd_forward_host: bad detector");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = g->ensure_host_buffers(h_inv_mu != nullptr, false);
    if (rc) return rc;
    const size_t vol = (size_t)g->G.nc * sizeof(float);
    if (h_fields) CK(cudaMemcpyAsync(g->hb_fields, h_fields, 6 * vol, cudaMemcpyHostToDevice, st));
    else          CK(cudaMemsetAsync(g->hb_fields, 0, 6 * vol, st));
    CK(cudaMemcpyAsync(g->hb_ie, h_inv_eps, vol, cudaMemcpyHostToDevice, st));
    if (h_inv_mu) CK(cudaMemcpyAsync(g->hb_im, h_inv_mu, vol, cudaMemcpyHostToDevice, st));
    HostStage hs;
    if ((rc = stage_descriptors(g, h_src, n_src, h_det, n_det, n_steps, true, nullptr, hs, st))) return rc;
    rc = fdtd_forward(g, g->hb_fields, g->hb_ie, h_inv_mu ? g->hb_im : nullptr, hs.src.data(), n_src, hs.det.data(), n_det, n_steps, st);
    if (rc) return rc;
    for (int s = 0; s < n_det; ++s)
        CK(cudaMemcpyAsync(h_det[s].phasor, hs.det[s].phasor, hs.phasor_bytes[s], cudaMemcpyDeviceToHost, st));
    if (h_fields) CK(cudaMemcpyAsync(h_fields, g->hb_fields, 6 * vol, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return FDTD_OK;
}

extern "C" int fdtd_backward_host(fdtd_grid *g, float *h_fields, const float *h_inv_eps, const float *h_inv_mu,
                                  const fdtd_source *h_src, int32_t n_src, const fdtd_detector *h_det, int32_t n_det,
                                  const float *const *h_dL_dphasor, const float *h_dL_dfields,
                                  int32_t n_steps, float *h_dL_dinv_eps, float *h_dL_dfields0, void *cuda_stream)
{
    if (!g) return fail(FDTD_EINVAL, "fdtd_backward_host: NULL grid");
    if (!h_inv_eps || !h_dL_dinv_eps) return fail(FDTD_EINVAL, "fdtd_backward_host: inv_eps and dL_dinv_eps are required");
    if (n_steps < 0 || n_steps > g->desc.max_steps) return fail(FDTD_EINVAL, "fdtd_backward_host: need 0 <= n_steps <= max_steps");
    if (n_src < 0 || n_det < 0 || (n_src && !h_src) || (n_det && !h_det)) return fail(FDTD_EINVAL, "fdtd_backward_host: bad descriptor arrays");
    for (int s = 0; s < n_src; ++s) if (!box_ok(g->G, h_src[s].lo, h_src[s].hi) || !h_src[s].waveform) return fail(FDTD_EINVAL, "fdtd_backward_host: bad source");
    for (int s = 0; s < n_det; ++s) if (!box_ok(g->G, h_det[s].lo, h_det[s].hi) || h_det[s].n_freq < 1) return fail(FDTD_EINVAL, "fdtd_backward_host: bad detector");
    if (!h_fields && !g->hb_fields) return fail(FDTD_ESTATE, "fdtd_backward_host: no state left by fdtd_forward_host");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = g->ensure_host_buffers(h_inv_mu != nullptr, true);
    if (rc) return rc;
    const size_t vol = (size_t)g->G.nc * sizeof(float);
    if ((h_dL_dfields || h_dL_dfields0) && !g->hb_cotf && (rc = g->alloc((void **)&g->hb_cotf, 6 * vol))) return rc;
    if (h_fields) CK(cudaMemcpyAsync(g->hb_fields, h_fields, 6 * vol, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(g->hb_ie, h_inv_eps, vol, cudaMemcpyHostToDevice, st));
    if (h_inv_mu) CK(cudaMemcpyAsync(g->hb_im, h_inv_mu, vol, cudaMemcpyHostToDevice, st));
    if (h_dL_dfields) CK(cudaMemcpyAsync(g->hb_cotf, h_dL_dfields, 6 * vol, cudaMemcpyHostToDevice, st));
    HostStage hs;
    if ((rc = stage_descriptors(g, h_src, n_src, h_det, n_det, n_steps, false, h_dL_dphasor, hs, st))) return rc;
    rc = fdtd_backward(g, g->hb_fields, g->hb_ie, h_inv_mu ? g->hb_im : nullptr, hs.src.data(), n_src, hs.det.data(), n_det,
                       h_dL_dphasor ? g->hb_cot.data() : nullptr, h_dL_dfields ? g->hb_cotf : nullptr, n_steps,
                       g->hb_grad, h_dL_dfields0 ? g->hb_cotf : nullptr, st);
    if (rc) return rc;
    CK(cudaMemcpyAsync(h_dL_dinv_eps, g->hb_grad, vol, cudaMemcpyDeviceToHost, st));
    if (h_dL_dfields0) CK(cudaMemcpyAsync(h_dL_dfields0, g->hb_cotf, 6 * vol, cudaMemcpyDeviceToHost, st));
    if (h_fields) CK(cudaMemcpyAsync(h_fields, g->hb_fields, 6 * vol, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return FDTD_OK;
}
