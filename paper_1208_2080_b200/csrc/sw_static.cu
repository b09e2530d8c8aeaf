// sw_static.cu -- sw_cluster_stats_static: cluster statistics of a labeled lattice for callers that
// must not allocate device memory (include/sw.h, "no device allocation").
//
// The context calls sw_measure(largest_cluster) / sw_measure_clusters count the sites of every cluster
// in a per-site counter array of 4 N bytes that the library cudaMalloc's on first use (k_cluster_sizes
// in sw_observe.cuh).  That is no use to a caller whose device memory is all spoken for: a process that
// handed every byte to its own pool at start-up (a cudaMalloc from a library then fails or eats into
// the pool's headroom), a simulation loop that cannot take the device-wide synchronisation a cudaMalloc
// implies in the middle of its sweeps, a host that runs under a fixed memory budget checked at load
// time.  This file gives them the same counting pass with the counters in a file-scope __device__ array
// of fixed size instead: the memory is part of the library's image on every GPU that loads it, nothing
// is allocated or freed by the call, and lattices beyond the fixed size are refused.
//
// A translation unit of its own: it shares no code with sw_api.cu and changes none of its paths.
#include "../../include/sw.h"

#include <cstdint>
#include <mutex>

#include <cuda_runtime.h>

namespace {

constexpr uint64_t kMaxSites = SW_STATIC_MAX_SITES;     // 2^20 sites = 4 MiB of counters per GPU
constexpr int kMaxDevices = 64;
constexpr int kThreads = 256;

// The counters.  In HOST code the name `g_sizes` is only a handle for the runtime's symbol table -- it is not a device
// address and must never be handed to a kernel; device_scratch() below asks the runtime where the array lives on the
// current device.
static __device__ __align__(256) uint32_t g_sizes[kMaxSites];

std::mutex g_lock;
uint32_t *g_sizes_on[kMaxDevices];        // device address of g_sizes per device ordinal, nullptr = not asked yet
thread_local const char *t_err = "";

int fail(int code, const char *what) { t_err = what; return code; }

// Set-up, once per device, with that device current: the address of g_sizes in that device's copy of the module.
int device_scratch(int dev, uint32_t **out)
{
    std::lock_guard<std::mutex> hold(g_lock);
    if (!g_sizes_on[dev]) {
        uint32_t *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_sizes);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return fail(SW_ERR_CUDA, "sw_cluster_stats_static: cudaGetSymbolAddress of the static scratch failed");
        }
        g_sizes_on[dev] = p;
    }
    *out = g_sizes_on[dev];
    return SW_OK;
}

// is p device (or managed) memory of device `dev`?  (cudaPointerGetAttributes allocates nothing)
bool on_device(const void *p, int dev)
{
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    if (a.type == cudaMemoryTypeManaged) return true;
    return a.type == cudaMemoryTypeDevice && a.device == dev;
}

// every call starts from zero counters and a zero result, whatever the call before left behind
__global__ void __launch_bounds__(kThreads)
k_static_clear(uint32_t *__restrict__ sizes, uint32_t n, unsigned long long *__restrict__ out)
{
    const uint32_t stride = gridDim.x * blockDim.x;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) sizes[i] = 0u;
    if (blockIdx.x == 0 && threadIdx.x < 4) out[threadIdx.x] = 0ull;
}

// sizes[labels[i]] += 1 for every site: the counting pass of k_cluster_sizes (sw_observe.cuh) on canonical labels,
// 16 consecutive sites per thread with runs of equal labels added at once (clusters are spatially coherent).
// A label that cannot be a canonical root of this lattice (>= n, or not its own label) is counted in out[3] and skipped,
// so a bad input can neither write outside the array nor pass unnoticed.
__global__ void __launch_bounds__(kThreads)
k_static_count(const uint32_t *__restrict__ labels, uint32_t n, uint32_t *__restrict__ sizes, unsigned long long *__restrict__ out)
{
    const uint32_t n_groups = (n + 15u) >> 4;
    const uint32_t stride = gridDim.x * blockDim.x;
    uint32_t bad = 0;
    for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < n_groups; g += stride) {
        uint32_t cur = 0, run = 0;
        for (uint32_t j = 0; j < 16u; ++j) {
            const uint32_t i = (g << 4) + j;
            if (i >= n) break;
            const uint32_t l = labels[i];
            if (run && l == cur) { ++run; continue; }
            if (run) atomicAdd(sizes + cur, run);
            run = 0;
            if (l >= n || labels[l] != l) { ++bad; continue; }
            cur = l; run = 1;
        }
        if (run) atomicAdd(sizes + cur, run);
    }
    if (bad) atomicAdd(out + 3, (unsigned long long)bad);
}

// out[0] = #{non-zero counters} = clusters, out[1] = the largest, out[2] = sum of squares (<= 2^40 for n <= 2^20)
__global__ void __launch_bounds__(kThreads)
k_static_reduce(const uint32_t *__restrict__ sizes, uint32_t n, unsigned long long *__restrict__ out)
{
    const uint32_t stride = gridDim.x * blockDim.x;
    unsigned long long count = 0, sq = 0;
    uint32_t big = 0;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const uint32_t s = sizes[i];
        if (!s) continue;
        count += 1;
        big = max(big, s);
        sq += (unsigned long long)s * s;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        count += __shfl_xor_sync(0xFFFFFFFFu, count, o);
        sq += __shfl_xor_sync(0xFFFFFFFFu, sq, o);
        big = max(big, __shfl_xor_sync(0xFFFFFFFFu, big, o));
    }
    if ((threadIdx.x & 31) == 0 && count) {
        atomicAdd(out + 0, count);
        atomicMax(out + 1, (unsigned long long)big);
        atomicAdd(out + 2, sq);
    }
}

}  // namespace

extern "C" {

uint64_t sw_static_max_sites(void) { return kMaxSites; }

const char *sw_static_last_error(void) { return t_err; }

int sw_cluster_stats_static(const uint32_t *dev_labels, uint64_t n_sites, uint64_t *dev_out, void *cuda_stream)
{
    // arguments first: these answers need no device
    if (!dev_labels || !dev_out) return fail(SW_ERR_INVALID_ARG, "sw_cluster_stats_static: dev_labels and dev_out must not be NULL");
    if (n_sites > kMaxSites)
        return fail(SW_ERR_INVALID_ARG, "sw_cluster_stats_static: n_sites is larger than SW_STATIC_MAX_SITES (1048576 sites, L = 1024): "
                                        "the static scratch cannot hold it; use sw_measure_clusters on a context instead");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return fail(SW_ERR_CUDA, "sw_cluster_stats_static: no CUDA device"); }
    if (dev < 0 || dev >= kMaxDevices) return fail(SW_ERR_CUDA, "sw_cluster_stats_static: device ordinal out of range (64 devices at most)");
    if (!on_device(dev_labels, dev) || !on_device(dev_out, dev))
        return fail(SW_ERR_INVALID_ARG, "sw_cluster_stats_static: dev_labels and dev_out must be device memory of the current device");
    uint32_t *sizes = nullptr;
    const int rc = device_scratch(dev, &sizes);
    if (rc != SW_OK) return rc;

    cudaStream_t stream = (cudaStream_t)cuda_stream;
    unsigned long long *out = reinterpret_cast<unsigned long long *>(dev_out);
    const uint32_t n = (uint32_t)n_sites;
    const int blocks_sites = (int)((n + kThreads - 1) / kThreads), blocks_groups = (int)(((n + 15u) / 16u + kThreads - 1) / kThreads);
    k_static_clear<<<blocks_sites > 0 ? blocks_sites : 1, kThreads, 0, stream>>>(sizes, n, out);
    if (n) {
        k_static_count<<<blocks_groups, kThreads, 0, stream>>>(dev_labels, n, sizes, out);
        k_static_reduce<<<blocks_sites, kThreads, 0, stream>>>(sizes, n, out);
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SW_ERR_CUDA, cudaGetErrorString(e));
    t_err = "";
    return SW_OK;
}

}  // extern "C"
