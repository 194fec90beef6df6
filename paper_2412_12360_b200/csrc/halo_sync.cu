// halo_sync.cu -- N3 (include/fdtd.h "Peer stores"): the ordering between the
// z slabs of one grid kept on the device.  With peer stores the step kernel of a slab writes its boundary planes into
// the neighbours' volumes; what is left of the halo exchange is "all slabs finish step n before any starts step n+1".
// Each slab owns two flags per direction of time (one per neighbour); after a step it publishes the index of the state
// it has reached in the flags its neighbours own (k_halo_signal, a release store at system scope behind the step
// kernel's completion), and before a step it waits until its own flags show the state it is about to read
// (k_halo_wait, acquire loads).  Both are graph nodes beside the step kernel, so a range of steps replays without the
// host.  A wait gives up after a bounded time and raises the grid's error flag instead of hanging the device.
#include <cuda_runtime.h>
#include <cstdlib>

#include "fdtd_grid.h"

namespace fdtd {
namespace {

__device__ __forceinline__ void st_release_sys(int *p, int v) { asm volatile("st.release.sys.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory"); }
__device__ __forceinline__ int ld_acquire_sys(const int *p)
{
    int v;
    asm volatile("ld.acquire.sys.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// state index reached = *slot + add (forward step n: n + 1; reverse step n: n)
__global__ void k_halo_signal(int *f_lo, int *f_hi, const int *slot, int add)
{
    const int v = *slot + add;
    __threadfence_system();
    if (f_lo) st_release_sys(f_lo, v);
    if (f_hi) st_release_sys(f_hi, v);
}

// state index about to be read = *slot + add (forward step n: n; reverse step n: n + 1); the state a run starts from
// (`skip`) is the caller's, nobody signals it.  A neighbour may already be one state further (it only needed my
// previous one), never two: the flag must show `want` or `want + dir` (dir = +1 forward, -1 reverse) -- an equality
// window, not an inequality, so that the value a previous run left behind does not pass (runs of >= 3 steps).
__global__ void k_halo_wait(const int *f_lo, const int *f_hi, const int *slot, int add, int skip, int dir, long long limit_ns, int *err)
{
    const int want = *slot + add;
    if (want == skip) return;
    long long t0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    for (int q = 0; q < 2; ++q) {
        const int *f = q ? f_hi : f_lo;
        if (!f) continue;
        for (;;) {
            const int v = ld_acquire_sys(f);
            if (v == want || v == want + dir) break;
            __nanosleep(200);
            long long t;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
            if (t - t0 > limit_ns) { atomicExch(err, want + 1); return; }
        }
    }
}

}  // namespace

void launch_halo_signal(int *f_lo, int *f_hi, const int *slot, int add, cudaStream_t st)
{
    k_halo_signal<<<1, 1, 0, st>>>(f_lo, f_hi, slot, add);
}

void launch_halo_wait(const int *f_lo, const int *f_hi, const int *slot, int add, int skip, int dir, int *err, cudaStream_t st)
{
    const char *e = getenv("FDTD_HALO_TIMEOUT_MS");        // read when the launch is enqueued (captured into the graph with it)
    const long long limit_ns = (e ? atoll(e) : 10000LL) * 1000000LL;
    k_halo_wait<<<1, 1, 0, st>>>(f_lo, f_hi, slot, add, skip, dir, limit_ns, err);
}

}  // namespace fdtd
