// probe.cu -- bandwidth probes for the roofline discussion (bench.py --probe).  Not on the hot path: they
// move the step kernel's bytes (7 volumes read, 6 written, float4 per thread) WITHOUT its arithmetic, halo or CPML, so that the
// step kernels can be held against what the memory system gives for their access pattern, not only against a plain copy.
//   pattern 0: grid-stride streaming over the volumes (every SM next to its neighbours' addresses), `runs` passes per launch
//              (a volume that fits in L2 then measures the L2 <-> SM rate without the launch overhead);
//   pattern 1: the step kernel's traversal -- a block marches a tile column (whole x rows, tile_y rows) plane by plane over
//              its run of planes (nz / runs), `unroll` planes per iteration in flight;
//   pattern 2: pattern 1 on ping-pong volumes, the way one time step hands its results to the next (launch r reads the six
//              volumes launch r-1 wrote, plus the seventh, constant one);
//   pattern 3: pattern 2 with the marching direction alternating from launch to launch (a launch starts on the planes the
//              previous one wrote last, which are still in L2).
#include <algorithm>
#include <string>
#include "fdtd_grid.h"

namespace {

__device__ __forceinline__ float4 mix(float4 a, float4 b, float4 e, float s)
{
    return make_float4(a.x + s * e.x * b.x, a.y + s * e.y * b.y, a.z + s * e.z * b.z, a.w + s * e.w * b.w);
}

__global__ void k_probe_stream(const float4 *__restrict__ in, float4 *__restrict__ out, size_t n4, float s, int inner)
{
    for (int it = 0; it < inner; ++it)
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n4; p += (size_t)gridDim.x * blockDim.x) {
        float4 v[7];
#pragma unroll
        for (int c = 0; c < 7; ++c) v[c] = __ldg(in + c * n4 + p);
#pragma unroll
        for (int c = 0; c < 6; ++c) out[c * n4 + p] = mix(v[c], v[(c + 1) % 6], v[6], s);
    }
}

template <int U>
__global__ void k_probe_tile(const float4 *__restrict__ in, const float4 *__restrict__ in7, float4 *__restrict__ out, int nx4, int ny,
                             int nz, int TY, int ncol, int nrun, float s, int down)
{
    const int col = blockIdx.x % ncol, run = blockIdx.x / ncol;
    if (run >= nrun) return;
    const int k0 = (int)((long long)nz * run / nrun), k1 = (int)((long long)nz * (run + 1) / nrun);
    const int j0 = col * TY, rows = min(TY, ny - j0), per_plane = rows * nx4;
    const size_t n4 = (size_t)nx4 * ny * nz;
    for (int kq = k0; kq < k1; kq += U)
        for (int t = threadIdx.x; t < per_plane; t += blockDim.x) {
            float4 v[U][7];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if (kq + u >= k1) break;
                const int k = down ? k1 - 1 - (kq - k0) - u : kq + u;
                const size_t p = ((size_t)k * ny + j0) * nx4 + t;
#pragma unroll
                for (int c = 0; c < 6; ++c) v[u][c] = __ldg(in + c * n4 + p);
                v[u][6] = __ldg(in7 + p);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if (kq + u >= k1) break;
                const int k = down ? k1 - 1 - (kq - k0) - u : kq + u;
                const size_t p = ((size_t)k * ny + j0) * nx4 + t;
#pragma unroll
                for (int c = 0; c < 6; ++c) out[c * n4 + p] = mix(v[u][c], v[u][(c + 1) % 6], v[u][6], s);
            }
        }
}

}  // namespace

// in: DEVICE, 7 volumes of nx*ny*nz floats; out: DEVICE, 6 volumes.  Synchronous (it times `reps` launches with CUDA events on
// cuda_stream after 3 warm-up launches).  *gbs = 13 volumes * 4 bytes * reps / time.
extern "C" int fdtd_probe_bandwidth(int32_t pattern, int32_t nx, int32_t ny, int32_t nz, int32_t tile_y, int32_t runs, int32_t unroll,
                                    int32_t blocks, int32_t threads, int32_t reps, const float *in, float *out, double *gbs,
                                    void *cuda_stream)
{
    if (nx < 4 || nx % 4 || ny < 1 || nz < 1 || !in || !out || !gbs || reps < 1 || threads < 32 || threads > 1024 || threads % 32)
        return fdtd_fail(FDTD_EINVAL, "fdtd_probe_bandwidth: bad argument (nx % 4 == 0, threads a multiple of 32 up to 1024)");
    if (pattern >= 1 && (tile_y < 1 || runs < 1 || runs > nz || (unroll != 1 && unroll != 2 && unroll != 4) || threads > 512))
        return fdtd_fail(FDTD_EINVAL, "fdtd_probe_bandwidth: patterns 1-3 need tile_y >= 1, 1 <= runs <= nz, unroll in {1, 2, 4}, threads <= 512");
    if (pattern < 0 || pattern > 3) return fdtd_fail(FDTD_EINVAL, "fdtd_probe_bandwidth: pattern must be 0 .. 3");
    if (pattern == 0 && blocks < 1) return fdtd_fail(FDTD_EINVAL, "fdtd_probe_bandwidth: blocks must be >= 1");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int inner = pattern == 0 ? std::max(1, runs) : 1;      // pattern 0: `runs` passes over the volumes inside one launch
    const size_t n4 = (size_t)nx / 4 * ny * nz;
    const int ncol = pattern ? (ny + tile_y - 1) / tile_y : 0;
    int launch_no = 0;
    auto launch = [&]() {
        const float4 *i4 = reinterpret_cast<const float4 *>(in);
        float4 *o4 = reinterpret_cast<float4 *>(out);
        const float4 *i7 = i4 + 6 * n4;
        int down = 0;
        if (pattern >= 2) {      // ping-pong: the first six volumes of `in` and the six of `out` swap roles with every launch
            if (launch_no & 1) { const float4 *t = i4; i4 = o4; o4 = const_cast<float4 *>(t); }
            down = pattern == 3 ? (launch_no & 1) : 0;
            ++launch_no;
        }
        // (s = 0: the ping-pong copies keep their values, launch after launch)
        const float sc = pattern >= 2 ? 0.f : 0.5f;
        if (pattern == 0) k_probe_stream<<<blocks, threads, 0, st>>>(i4, o4, n4, 0.5f, inner);
        else if (unroll == 1) k_probe_tile<1><<<ncol * runs, threads, 0, st>>>(i4, i7, o4, nx / 4, ny, nz, tile_y, ncol, runs, sc, down);
        else if (unroll == 2) k_probe_tile<2><<<ncol * runs, threads, 0, st>>>(i4, i7, o4, nx / 4, ny, nz, tile_y, ncol, runs, sc, down);
        else k_probe_tile<4><<<ncol * runs, threads, 0, st>>>(i4, i7, o4, nx / 4, ny, nz, tile_y, ncol, runs, sc, down);
    };
    cudaEvent_t a = nullptr, b = nullptr;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, "cudaEventCreate"); }
    for (int w = 0; w < 3; ++w) launch();
    cudaEventRecord(a, st);
    for (int r = 0; r < reps; ++r) launch();
    cudaEventRecord(b, st);
    cudaError_t e = cudaEventSynchronize(b);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventDestroy(a); cudaEventDestroy(b);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fdtd_fail(FDTD_ECUDA, std::string("fdtd_probe_bandwidth: ") + cudaGetErrorString(e)); }
    *gbs = 13.0 * (double)n4 * 16.0 * reps * inner / ((double)ms * 1e-3) / 1e9;
    return FDTD_OK;
}
