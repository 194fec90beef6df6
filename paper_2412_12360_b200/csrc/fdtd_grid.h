// fdtd_grid.h -- the grid object behind the opaque fdtd_grid handle (host side, private).
#pragma once
#include <string>
#include <vector>
#include "fdtd_internal.h"

struct FusedState;   // kernels_step.cu

// descriptor slots of the fused step kernels' parameter block; a call with more sources or detectors runs on the
// generic kernels (FDTD_PATH_AUTO) -- see include/fdtd.h "Kernel paths"
constexpr int FDTD_FUSED_MAX_SRC = 4, FDTD_FUSED_MAX_DET = 4;

struct fdtd_grid {
    fdtd_grid_desc desc{};
    fdtd::Dims G{};
    fdtd::Tables T{};
    fdtd::RecLayout R{};
    std::vector<float> h_tables;          // host copy of the CPML tables (layout as uploaded)

    int path = FDTD_PATH_GENERIC;
    int tile_x = 0, tile_y = 0, tile_z = 0;
    std::string fused_why_not;
    bool fused_backward_ready = false;    // false: fdtd_backward uses the generic reverse kernels
    int graph_unroll = 8;
    int pipelined_inverse_ctas = 0;       // fused path: CTAs of the inverse step in the pipelined reverse sweep (0: sequential)

    // device memory owned by the grid
    std::vector<void *> owned;
    long long recorder_bytes = 0, scratch_bytes = 0;
    int *d_step = nullptr;                 // two slots; the step being enqueued reads slot step_par, the next one the other
    int step_par = 0;
    int *step_in() const { return d_step + step_par; }
    int *step_out() const { return d_step + (step_par ^ 1); }
    fdtd::PsiSet psiE[2]{}, psiH[2]{};     // primal psi ([1] only used by the fused path's ping-pong)
    fdtd::PsiSet lpsiE[2]{}, lpsiH[2]{};   // psi cotangents, ping-ponged by step parity
    float *lam = nullptr;                  // cotangent fields [6][nz][ny][nx]
    float *rec = nullptr;                  // interface recorder
    float *ckpt = nullptr, *dE = nullptr;  // record = 3: checkpoints [ck_count][ck_stride], dE [ck_every][3][box cells]
    int ck_every = 0, ck_count = 0;
    float *e2buf = nullptr;                // lossy medium on a fused record = 3 grid: lamE' before its scaling by Ca, [3][nc] (fdtd_set_conductivity)
    float *ck_e2 = nullptr;                // = e2buf while the checkpointed sweep runs a fused adjoint step of a lossy medium
    bool ck_store = false;                 // set while the checkpointed sweep replays a segment on the fused kernels: D = dE'/d inv_eps after every step
    float *ck_gradhook = nullptr;          // set while it runs the segment's fused adjoint steps: g += lamE' . D after every step
    float *ck_grad = nullptr;              // set while the checkpointed sweep runs an adjoint step on the generic kernels: g += lamE' . D there
    const float *sigma = nullptr;          // N4: conductivity volume of the caller (fdtd_set_conductivity), or NULL
    bool replaying = false;                // the checkpointed reverse sweep is re-running forward steps: the state stays in its ping-pong volume
    size_t ck_stride = 0;
    int recorded_steps = -1;               // n_steps of the last recorded forward, or -1
    int fwd_pos = -1, bwd_pos = -1;        // fdtd_forward_range / fdtd_backward_range: the state index the last call left
    bool fwd_fused = false, bwd_fused = false;   // which kernels the last (range) call ran on: where its state lives
    float *d_cs = nullptr;                 // per-step (cos, sin) table
    float *h_cs = nullptr;                 // pinned staging of the same
    size_t cs_cap = 0;
    std::vector<float> cs_key;             // n_steps and the frequencies of the table on the device
    cudaEvent_t table_done = nullptr;
    fdtd::ReduceScratch red{};             // block partials + ticket of the N2 reductions (energy, flux)

    // host-buffer entry points
    float *hb_fields = nullptr, *hb_ie = nullptr, *hb_im = nullptr, *hb_grad = nullptr, *hb_cotf = nullptr;
    void *hb_desc = nullptr;
    size_t hb_desc_cap = 0;
    std::vector<const float *> hb_cot;

    // graphs
    struct GraphCache {
        std::string key;
        cudaGraphExec_t exec_main = nullptr, exec_tail[2] = { nullptr, nullptr };   // tail: one step, per counter slot
        cudaEvent_t done = nullptr;
        long long step_per = 0, inv_per = 0;   // fused step / inverse kernels per time step in this graph
    } fwd_graph, bwd_graph;
    cudaStream_t cap_stream = nullptr;
    // fork / join of the launches that run beside a step kernel (recorder, inverse step, face injection): the side
    // streams wait for fork_ev recorded on the main stream, the main stream waits for their join events
    cudaStream_t side_stream[2] = { nullptr, nullptr };
    cudaEvent_t fork_ev = nullptr, join_ev[2] = { nullptr, nullptr };
    long long kernel_launches = 0;
    long long fused_step_launches = 0, fused_inverse_launches = 0;   // counted as they are enqueued (graph nodes x replays)
    int partition = FDTD_PARTITION_NONE;
    long long enq_step = 0, enq_inv = 0;   // bumped by every enqueue of a fused step / inverse kernel (run_steps turns them into launch counts)

    FusedState *fused = nullptr;

    // N3 peer stores (fdtd_halo_attach): [which: 0 primal, 1 cotangents][side: 0 below, 1 above].  vol[q] = component 3 of
    // the plane of the neighbour's volume q that this grid's step kernel writes; nc = the neighbour's component stride
    struct PeerLink { float *vol[2] = { nullptr, nullptr }; long long nc = 0; int *flag = nullptr; };
    PeerLink peer[2][2];
    // device-side ordering of the slabs (halo_sync.cu): my flags [which][side] (written by that neighbour), PeerLink.flag =
    // the flag of mine in the neighbour's set; herr: raised by a wait that gave up
    int *d_hflags = nullptr, *d_herr = nullptr;

    // per-kernel profiling (fdtd_set_profiling)
    enum ProfClass { PC_UPDATE_E, PC_UPDATE_H, PC_ADJ_H, PC_INV_H, PC_INV_E_GRAD, PC_ADJ_E,
                     PC_FUSED_FWD, PC_FUSED_BWD, PC_FUSED_INV, PC_RECORD, PC_INJECT, PC_SRC_DET, PC_OTHER, PC_COUNT };
    bool profiling = false;
    struct ProfSpan { int cls; cudaEvent_t a, b; };
    std::vector<ProfSpan> prof_spans;
    std::vector<cudaEvent_t> prof_pool;
    long long prof_launches[PC_COUNT] = {};
    double prof_ms[PC_COUNT] = {};
    bool prof_capturing = false;           // true while a graph is being captured (no events then)
    cudaEvent_t prof_begin(cudaStream_t st);
    void prof_end(int cls, cudaEvent_t a, cudaStream_t st);

    int alloc(void **p, size_t bytes, bool recorder = false);
    int alloc_psi(fdtd::PsiSet &s);
    int zero_psi(const fdtd::PsiSet &s, cudaStream_t st);
    int ensure_backward_buffers();
    int ensure_host_buffers(bool need_mu, bool need_grad);
    int reserve_cs_table(size_t floats);
    void drop_graphs();
};

// fused TMA path (kernels_step.cu).  fused_setup decides whether the grid qualifies and, if so,
// sets g->path = FDTD_PATH_FUSED; otherwise it records the reason in g->fused_why_not.
int fused_setup(fdtd_grid *g);
void fused_teardown(fdtd_grid *g);
int fused_alloc_backward(fdtd_grid *g);    // second cotangent volume of the ping-pong
int fused_forward(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                  const std::vector<fdtd::SourceDev> &S, const std::vector<fdtd::DetectorDev> &D,
                  const std::vector<fdtd::TimeDetDev> &TD, int total_freq, int n_begin, int n_end, int n_total, bool recording,
                  cudaStream_t st);
int fused_backward(fdtd_grid *g, float *fields, const float *inv_eps, const float *inv_mu,
                   const std::vector<fdtd::SourceDev> &S, const std::vector<fdtd::DetectorDev> &D,
                   const std::vector<fdtd::TimeDetDev> &TD, int total_freq, int n_hi, int n_lo, int n_total, float *dL_dinv_eps,
                   bool seeded_H, cudaStream_t st, float *dL_dinv_mu = nullptr);
// the volume that holds state n of the fused path's ping-pong: which = 0 primal (fields / second buffer), 1 cotangents
float *fused_volume(fdtd_grid *g, float *fields, int which, int n);

namespace fdtd {
void launch_halo_signal(int *f_lo, int *f_hi, const int *slot, int add, cudaStream_t st);
void launch_halo_wait(const int *f_lo, const int *f_hi, const int *slot, int add, int skip, int dir, int *err, cudaStream_t st);
}

// RAII span: brackets the launches made in its lifetime with two events when profiling is on
struct ProfScope {
    fdtd_grid *g; int cls; cudaStream_t st; cudaEvent_t a;
    ProfScope(fdtd_grid *g_, int cls_, cudaStream_t st_) : g(g_), cls(cls_), st(st_), a(g_->prof_begin(st_)) {}
    ~ProfScope() { if (a) g->prof_end(cls, a, st); }
};

// shared by the API and the fused path
int fdtd_fail(int code, const std::string &msg);
