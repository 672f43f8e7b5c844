// tb_noalloc.cu -- tb_series_mean_noalloc: the series mean (the resampler's default fill value,
// DESIGN.md reading G8) for callers that must not allocate device memory.
//
// Who this is for.  Two kinds of caller cannot use tb_plan_create / tb_plan_set_series just to get
// the fill value of a fresh time series, because both of those call cudaMalloc:
//   * a telescope back end's real-time loop.  cudaMalloc and cudaFree take a driver-wide lock and
//     cudaFree waits for the whole device to drain, so an allocation made while ingest copies and
//     searches are in flight on other streams stalls all of them; such loops allocate at start-up
//     and never again.
//   * a process that gave all of the GPU's memory to a pool of its own (or to a framework's
//     caching allocator) when it started.  There is nothing left for cudaMalloc to hand out, so a
//     library that allocates behind the caller's back fails with out-of-memory at a moment the
//     caller does not control.
// For them the partial sums of the reduction -- the only scratch memory k_sum_f64's plan-owned
// variant needs (tb_api.cu load_series) -- live in the file-scope array below, which the CUDA
// runtime places on a device when it loads this library's kernels there and which stays until the
// process ends: TB_NOALLOC_SCRATCH_BYTES (33 024 bytes) per GPU that uses the library.  The caller
// passes the series and the output word; nothing in this file calls cudaMalloc, cudaFree or any
// library routine that allocates.
//
// What it computes: mean = (1/n) sum_j x_j in fp64, deterministically.  Tile b (65 536 consecutive
// samples) is summed by CTA b: thread t adds x[b*65536 + t + 256 i], i = 0..255, in that order, the
// 256 thread sums are added in a fixed tree, and the CTA that finishes last adds the tile sums the
// same way.  The result does not depend on the grid, the SM count or the timing of the CTAs.  It
// differs from load_series' value (296 strided subsets, summed on the host in long double) only by
// fp64 rounding order, i.e. by a few 1e-16 relative, far below one float32 ulp of the fill value.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/tb.h"

namespace {

constexpr uint32_t NA_TILE_LOG2 = 16;                       // samples per partial sum
constexpr uint32_t NA_TILE = 1u << NA_TILE_LOG2;
constexpr uint32_t NA_THREADS = 256;
constexpr uint32_t NA_MAX_TILES = (uint32_t)(TB_NOALLOC_MAX_SAMPLES >> NA_TILE_LOG2);   // 4096
constexpr uint32_t NA_HEADER = 32;                          // 256 bytes: [0] is the arrival ticket
static_assert(((uint64_t)NA_MAX_TILES << NA_TILE_LOG2) == TB_NOALLOC_MAX_SAMPLES, "tile count");
static_assert((NA_HEADER + NA_MAX_TILES) * sizeof(double) == TB_NOALLOC_SCRATCH_BYTES, "tb.h states the size");

// The scratch.  One copy per device, shared by every call in the process; it keeps whatever the
// last call left in it.  In HOST code this name is only a handle for the runtime (passing it to a
// kernel would hand the kernel a host address); the device address is looked up per device in
// scratch_for() and that pointer is what the kernel receives.
static __device__ __align__(256) double g_na_scratch[NA_HEADER + NA_MAX_TILES];

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mutex;
double* g_na_ptr[NA_MAX_DEVICES] = {};                      // device address of g_na_scratch, per ordinal

__device__ __forceinline__ double block_sum_256(double s, double* s_w)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = s;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < (int)(NA_THREADS / 32); ++w) t += s_w[w];
    __syncthreads();                                        // s_w may be reused
    return t;                                               // valid in thread 0
}

// grid = n_tiles CTAs of 256 threads.  scratch[0] (as a 32-bit word) must be zero at launch.
__global__ void __launch_bounds__(NA_THREADS)
k_mean_tiles(const float* __restrict__ x, size_t n, double* __restrict__ scratch, uint32_t n_tiles,
             double* __restrict__ mean_out)
{
    __shared__ double s_w[NA_THREADS / 32];
    __shared__ bool s_last;
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
    double* part = scratch + NA_HEADER;

    const size_t base = (size_t)blockIdx.x << NA_TILE_LOG2;
    const size_t end = (n - base < (size_t)NA_TILE) ? n : base + NA_TILE;
    double s = 0.0;
#pragma unroll 8
    for (size_t i = base + threadIdx.x; i < end; i += NA_THREADS) s += (double)__ldg(x + i);
    const double tile_sum = block_sum_256(s, s_w);
    if (threadIdx.x == 0) {
        part[blockIdx.x] = tile_sum;
        __threadfence();                                    // the tile sum is visible before the ticket moves
        s_last = atomicAdd(ticket, 1u) == n_tiles - 1;
    }
    __syncthreads();
    if (!s_last) return;

    __threadfence();                                        // every other CTA's tile sum is visible now
    double a = 0.0;
    for (uint32_t i = threadIdx.x; i < n_tiles; i += NA_THREADS) a += __ldcg(part + i);   // L2, never a stale L1 line
    const double total = block_sum_256(a, s_w);
    if (threadIdx.x == 0) {
        *mean_out = total / (double)n;
        *ticket = 0u;                                       // leave the array ready (the host clears it again anyway)
    }
}

int na_fail(char* errbuf, uint64_t errbuf_len, int code, const char* fmt, ...)
{
    if (errbuf && errbuf_len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, (size_t)errbuf_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// Device address of the scratch array on the CURRENT device; looked up once per device.
cudaError_t scratch_for(int device, double** out)
{
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[device]) {
        double* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_na_scratch);
        if (e != cudaSuccess) return e;
        g_na_ptr[device] = ptr;
    }
    *out = g_na_ptr[device];
    return cudaSuccess;
}

bool on_device(const void* p, int device)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) && at.device == device;
}

}  // namespace

extern "C" int tb_series_mean_noalloc(const float* d_series, uint64_t n_samples, double* d_mean_out, void* stream,
                                      char* errbuf, uint64_t errbuf_len)
{
    if (errbuf && errbuf_len) errbuf[0] = '\0';
    if (n_samples > TB_NOALLOC_MAX_SAMPLES)
        return na_fail(errbuf, errbuf_len, TB_ERR_CAPACITY,
                       "tb_series_mean_noalloc: n_samples = %llu is beyond TB_NOALLOC_MAX_SAMPLES = %llu (the static scratch "
                       "array holds %u partial sums of %u samples); use a plan (tb_plan_create), which allocates",
                       (unsigned long long)n_samples, (unsigned long long)TB_NOALLOC_MAX_SAMPLES, NA_MAX_TILES, NA_TILE);
    if (n_samples == 0) return na_fail(errbuf, errbuf_len, TB_ERR_INVALID_ARG, "tb_series_mean_noalloc: n_samples is 0 (no mean)");
    if (!d_series || !d_mean_out) return na_fail(errbuf, errbuf_len, TB_ERR_INVALID_ARG, "tb_series_mean_noalloc: null pointer");

    int device = -1;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) { cudaGetLastError(); return na_fail(errbuf, errbuf_len, TB_ERR_CUDA, "tb_series_mean_noalloc: cudaGetDevice: %s", cudaGetErrorString(e)); }
    if (device < 0 || device >= NA_MAX_DEVICES)
        return na_fail(errbuf, errbuf_len, TB_ERR_INVALID_ARG, "tb_series_mean_noalloc: device ordinal %d is not below %d", device, NA_MAX_DEVICES);
    if (!on_device(d_series, device) || !on_device(d_mean_out, device))
        return na_fail(errbuf, errbuf_len, TB_ERR_INVALID_ARG,
                       "tb_series_mean_noalloc: d_series and d_mean_out must be device memory of the current device (%d)", device);

    double* scratch = nullptr;
    e = scratch_for(device, &scratch);
    if (e != cudaSuccess) { cudaGetLastError(); return na_fail(errbuf, errbuf_len, TB_ERR_CUDA, "tb_series_mean_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e)); }

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const uint32_t n_tiles = (uint32_t)((n_samples + NA_TILE - 1) >> NA_TILE_LOG2);
    // the ticket must start at zero whatever an earlier (possibly overlapping, hence broken) call left
    e = cudaMemsetAsync(scratch, 0, NA_HEADER * sizeof(double), st);
    if (e != cudaSuccess) { cudaGetLastError(); return na_fail(errbuf, errbuf_len, TB_ERR_CUDA, "tb_series_mean_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e)); }
    k_mean_tiles<<<n_tiles, NA_THREADS, 0, st>>>(d_series, (size_t)n_samples, scratch, n_tiles, d_mean_out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(errbuf, errbuf_len, TB_ERR_CUDA, "tb_series_mean_noalloc: kernel launch: %s", cudaGetErrorString(e));
    return TB_OK;
}
