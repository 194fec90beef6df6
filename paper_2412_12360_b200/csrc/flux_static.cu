// flux_static.cu -- fdtd_flux_static: the Poynting flux of fdtd_flux (reading R24) for callers that
// cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// fdtd_flux takes its reduction scratch (block partials + ticket) from a grid object, which fdtd_create_grid allocated with
// cudaMalloc.  This variant needs no grid and allocates nothing: its scratch is the file-scope array below, part of the
// library image on every GPU that loads it (16.25 KB per device until the process exits).  The array bounds the launch:
// one partial per block, a block sums FS_CHUNK plane cells, so a plane of more than FDTD_FLUX_STATIC_MAX_CELLS cells is
// rejected.  All calls share the array and it keeps the last call's contents: the ticket is cleared on the caller's stream
// at the start of every call, the partials are written before they are read.  Calls that overlap on the GPU (two streams,
// two threads) race on it.
//
// In host code the array's name is a host-side stand-in, not a device address: the entry point resolves the address once
// per device with cudaGetSymbolAddress (that device current) and passes the pointer to the kernel.
#include <cmath>
#include <mutex>
#include <string>
#include "fdtd_grid.h"

namespace {

constexpr int FS_THREADS = 256;
constexpr int FS_ITEMS = 8;                                    // plane cells per thread
constexpr int FS_CHUNK = FS_THREADS * FS_ITEMS;                // plane cells per block
constexpr int FS_MAX_BLOCKS = FDTD_FLUX_STATIC_MAX_CELLS / FS_CHUNK;
constexpr int FS_TICKET_OFF = FS_MAX_BLOCKS * (int)sizeof(double);
constexpr int FS_SCRATCH_BYTES = FS_TICKET_OFF + 256;          // [FS_MAX_BLOCKS] double partials, then the ticket
constexpr int FS_MAX_DEVICES = 64;
static_assert(FDTD_FLUX_STATIC_MAX_CELLS % FS_CHUNK == 0, "the cell limit is a whole number of blocks");

static __device__ __align__(256) unsigned char g_flux_static_scratch[FS_SCRATCH_BYTES];

// geometry of the detector slab (normal axis a; box cells ordered [k][j][i]) and the slots of the four tangential
// components among the detector's components
struct FsGeom {
    int ext[3];
    int a, u, v;               // normal axis; the two in-plane axes, u the lower-numbered (fastest) one
    int t1;                    // plane of E (and of the upper H) inside the box
    int sEb, sEc, sHb, sHc;
    long long bc, plane_cells;
    int interpolate;
    float cw, sw;              // cos, sin(omega_f / 2): H is stamped half a step late (co-location in time)
};

// flux_f = 1/2 sum_cells Re(E_b conj(H~_c) - E_c conj(H~_b)), H~ = H (interpolate == 0) or
// exp(-i omega_f / 2) (H[p-1] + H[p]) / 2.  Block b sums cells [b FS_CHUNK, (b+1) FS_CHUNK) into partial[b]; the block
// that draws the last ticket adds the partials in slot order (the result does not depend on the block schedule),
// writes *out and leaves the ticket at zero for the next launch.
__global__ void __launch_bounds__(FS_THREADS) k_flux_static(FsGeom q, const float2 *__restrict__ P, float *__restrict__ out,
                                                            unsigned char *__restrict__ scratch)
{
    double *partial = reinterpret_cast<double *>(scratch);
    unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch + FS_TICKET_OFF);
    __shared__ double sh[FS_THREADS / 32];
    __shared__ bool last;
    double acc = 0.0;
    const long long base = (long long)blockIdx.x * FS_CHUNK + threadIdx.x;
#pragma unroll
    for (int it = 0; it < FS_ITEMS; ++it) {
        const long long t = base + (long long)it * FS_THREADS;
        if (t >= q.plane_cells) break;
        int pos[3];
        pos[q.u] = (int)(t % q.ext[q.u]); pos[q.v] = (int)(t / q.ext[q.u]); pos[q.a] = q.t1;
        const long long cell = ((long long)pos[2] * q.ext[1] + pos[1]) * q.ext[0] + pos[0];
        pos[q.a] -= 1;
        const long long cellm = q.interpolate ? ((long long)pos[2] * q.ext[1] + pos[1]) * q.ext[0] + pos[0] : cell;
#pragma unroll
        for (int pr = 0; pr < 2; ++pr) {          // pair 0: E_b with H_c (+), pair 1: E_c with H_b (-)
            const int sE = pr ? q.sEc : q.sEb, sH = pr ? q.sHb : q.sHc;
            const float2 E = __ldg(P + (long long)sE * q.bc + cell);
            const float2 H1 = __ldg(P + (long long)sH * q.bc + cell), H0 = __ldg(P + (long long)sH * q.bc + cellm);
            const float hr = q.interpolate ? 0.5f * (H0.x + H1.x) : H1.x, hi = q.interpolate ? 0.5f * (H0.y + H1.y) : H1.y;
            const float tr = hr * q.cw + hi * q.sw, ti = hi * q.cw - hr * q.sw;
            const float s = 0.5f * (E.x * tr + E.y * ti);
            acc += pr ? -(double)s : (double)s;
        }
    }
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) sh[warp] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
        for (int w = 0; w < FS_THREADS / 32; ++w) v += sh[w];
        partial[blockIdx.x] = v;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double s = 0.0;
    for (unsigned b = threadIdx.x; b < gridDim.x; b += FS_THREADS) s += *((volatile double *)partial + b);
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    __syncthreads();
    if (lane == 0) sh[warp] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < FS_THREADS / 32; ++w) t += sh[w];
        *out = (float)t;
        *ticket = 0u;
    }
}

// device address of the scratch array, resolved once per device (with that device current)
std::mutex s_mu;
unsigned char *s_scratch[FS_MAX_DEVICES] = {};

int scratch_of_current_device(unsigned char **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, std::string("fdtd_flux_static: cudaGetDevice: ") + cudaGetErrorString(e)); }
    if (dev < 0 || dev >= FS_MAX_DEVICES) return fdtd_fail(FDTD_EINVAL, "fdtd_flux_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(s_mu);
    if (!s_scratch[dev]) {
        unsigned char *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_flux_static_scratch);
        if (e != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return fdtd_fail(FDTD_ECUDA, std::string("fdtd_flux_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        }
        s_scratch[dev] = p;
    }
    *out = s_scratch[dev];
    return FDTD_OK;
}

}  // namespace

extern "C" int fdtd_flux_static(const fdtd_detector *det, const float *phasor, int32_t axis, int32_t interpolate, float *flux,
                                void *cuda_stream)
{
    if (!det || !phasor || !flux) return fdtd_fail(FDTD_EINVAL, "fdtd_flux_static: NULL argument");
    if (axis < 0 || axis > 2) return fdtd_fail(FDTD_EINVAL, "fdtd_flux_static: axis must be 0..2");
    if (det->component_mask <= 0 || det->component_mask > 63 || det->n_freq < 1 || !det->omega)
        return fdtd_fail(FDTD_EINVAL, "fdtd_flux_static: bad detector descriptor");
    FsGeom q;
    for (int x = 0; x < 3; ++x) {
        if (det->lo[x] < 0 || det->hi[x] <= det->lo[x]) return fdtd_fail(FDTD_EINVAL, "fdtd_flux_static: bad detector descriptor (empty box)");
        q.ext[x] = det->hi[x] - det->lo[x];
    }
    const int a = axis, b = (a + 1) % 3, c = (a + 2) % 3;
    const int need = (1 << b) | (1 << c) | (1 << (3 + b)) | (1 << (3 + c));
    if ((det->component_mask & need) != need)
        return fdtd_fail(FDTD_EINVAL, "fdtd_flux_static: the detector lacks a tangential component of the plane");
    if (q.ext[a] != (interpolate ? 2 : 1))
        return fdtd_fail(FDTD_EINVAL, "fdtd_flux_static: the box must be 1 plane thick along the axis (2 with interpolation)");
    q.plane_cells = (long long)q.ext[b] * q.ext[c];
    if (q.plane_cells > FDTD_FLUX_STATIC_MAX_CELLS)
        return fdtd_fail(FDTD_EINVAL, "fdtd_flux_static: a plane of " + std::to_string(q.plane_cells) + " cells is beyond the static scratch's maximum of " +
                                      std::to_string((long long)FDTD_FLUX_STATIC_MAX_CELLS) + " cells (use fdtd_flux)");
    auto slot = [&](int comp) { int ci = 0; for (int x = 0; x < comp; ++x) ci += (det->component_mask >> x) & 1; return ci; };
    int ncomp = 0;
    for (int x = 0; x < 6; ++x) ncomp += (det->component_mask >> x) & 1;
    q.a = a; q.u = b < c ? b : c; q.v = b < c ? c : b;
    q.t1 = q.ext[a] - 1;
    q.sEb = slot(b); q.sEc = slot(c); q.sHb = slot(3 + b); q.sHc = slot(3 + c);
    q.bc = (long long)q.ext[0] * q.ext[1] * q.ext[2];
    q.interpolate = interpolate ? 1 : 0;

    unsigned char *scratch = nullptr;
    int rc = scratch_of_current_device(&scratch);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the array keeps whatever the last call (or an aborted one) left: the ticket must start at zero
    cudaError_t e = cudaMemsetAsync(scratch + FS_TICKET_OFF, 0, 256, st);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, std::string("fdtd_flux_static: cudaMemsetAsync: ") + cudaGetErrorString(e)); }
    const unsigned blocks = (unsigned)((q.plane_cells + FS_CHUNK - 1) / FS_CHUNK);
    for (int f = 0; f < det->n_freq; ++f) {
        q.cw = q.interpolate ? (float)std::cos(0.5 * (double)det->omega[f]) : 1.f;
        q.sw = q.interpolate ? (float)std::sin(0.5 * (double)det->omega[f]) : 0.f;
        const float2 *P = reinterpret_cast<const float2 *>(phasor) + (long long)f * ncomp * q.bc;
        k_flux_static<<<blocks, FS_THREADS, 0, st>>>(q, P, flux + f, scratch);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return fdtd_fail(FDTD_ECUDA, std::string("fdtd_flux_static launch: ") + cudaGetErrorString(e));
    return FDTD_OK;
}
