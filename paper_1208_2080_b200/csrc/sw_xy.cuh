// sw_xy.cuh -- embedded-cluster Swendsen-Wang sweeps of the 2D classical XY model ("This computation is
// easily extended to continuous spin models, such as the classical XY model, using the Wolff's idea of embedded
// cluster").  The same three steps on the Ising variables embedded by a
// random direction r: a_i = s_i . r,
//   (1) bond <ij> active iff a_i a_j > 0 and draw < floor(p_ij 2^32), p_ij = 1 - exp(-2 K a_i a_j)   (k_xy_bonds)
//   (2) clusters of active bonds, canonical label = smallest site: the any-L union-find kernels of
//       sw_generic.cuh, unchanged -- the labeling core does not care what made the bonds
//   (3) every cluster is reflected, s -> s - 2 (s . r) r, iff the FLIP draw of its root maps to 1       (k_xy_flip)
// Draws: Philox4x32-10 with the Potts layout (BOND per site pair, FLIP per root) plus purpose 3 REFLECT for r, whose
// cos / sin are taken once per sweep on the host.  Arithmetic: IEEE double with every rounding spelled out
// (__dmul_rn / __fma_rn / __dadd_rn, which the compiler never contracts), so that spins agree bit for bit with a CPU
// implementation using the same correctly rounded operations (readings X1-X6).
// Compiled as part of sw_api.cu (one translation unit).
#pragma once

#include "../../include/sw.h"

#include <cmath>
#include <new>
#include <string>
#include <vector>

#include "sw_host.h"
#include "sw_common.cuh"
#include "sw_generic.cuh"
#include "sw_observe.cuh"

namespace sw {

constexpr uint32_t kPurposeReflect = 3u;

__device__ __forceinline__ double xy_projection(double2 s, double rx, double ry)
{
    return __fma_rn(s.x, rx, __dmul_rn(s.y, ry));
}

// floor((1 - exp(-2 K a_i a_j)) 2^32) as a 33-bit integer; 0 unless a_i a_j > 0
__device__ __forceinline__ unsigned long long xy_bond_threshold(double two_K, double ai, double aj)
{
    const double x = __dmul_rn(__dmul_rn(two_K, ai), aj);
    if (!(x > 0.0)) return 0ull;
    if (isinf(x)) return 1ull << 32;
    const double scaled = floor(ldexp(-expm1(-x), 32));
    if (scaled <= 0.0) return 0ull;
    if (scaled >= 4294967296.0) return 1ull << 32;
    return (unsigned long long)scaled;
}

__global__ void k_xy_init_random(double2 *__restrict__ spins, Params P)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) {
        const uint4 w = philox4x32_10((uint32_t)i, (uint32_t)(i >> 32), 0u, kPurposeInit, P);
        const double c = 1.0 / 2147483648.0;
        double x = __dadd_rn(__dmul_rn(__dadd_rn((double)w.x, 0.5), c), -1.0);
        double y = __dadd_rn(__dmul_rn(__dadd_rn((double)w.y, 0.5), c), -1.0);
        double n2 = __fma_rn(x, x, __dmul_rn(y, y));
        if (n2 > 1.0) {
            x = __dadd_rn(__dmul_rn(__dadd_rn((double)w.z, 0.5), c), -1.0);
            y = __dadd_rn(__dmul_rn(__dadd_rn((double)w.w, 0.5), c), -1.0);
            n2 = __fma_rn(x, x, __dmul_rn(y, y));
        }
        const double n = __dsqrt_rn(n2);
        spins[i] = make_double2(__ddiv_rn(x, n), __ddiv_rn(y, n));
    }
}

__global__ void k_xy_ordered(double2 *__restrict__ spins, Params P)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) spins[i] = make_double2(1.0, 0.0);
}

// step (1): one thread per 16-site bond word (the storage of sw_generic.cuh)
__global__ void k_xy_bonds(const double2 *__restrict__ spins, uint32_t *__restrict__ bonds, Params P, double two_K, double rx, double ry)
{
    const uint64_t n_words = (P.N + 15) >> 4;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t L = P.L;
    for (uint64_t w = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_words; w += stride) {
        uint32_t word = 0;
        for (uint32_t j = 0; j < 16; ++j) {
            const uint64_t i = (w << 4) + j;
            if (i >= P.N) break;
            const uint64_t y = i / L, x = i - y * L;
            const uint64_t ir = y * L + (x + 1 == L ? 0 : x + 1);
            const uint64_t id = (y + 1 == L ? 0 : y + 1) * L + x;
            const double a = xy_projection(spins[i], rx, ry);
            const unsigned long long tr = xy_bond_threshold(two_K, a, xy_projection(spins[ir], rx, ry));
            const unsigned long long td = xy_bond_threshold(two_K, a, xy_projection(spins[id], rx, ry));
            if (tr | td) {
                const uint64_t pair = i >> 1;
                const uint4 d = philox4x32_10((uint32_t)pair, (uint32_t)(pair >> 32), P.t, kPurposeBond, P);
                const uint32_t dr = (i & 1) ? d.z : d.x;
                const uint32_t dd = (i & 1) ? d.w : d.y;
                if ((unsigned long long)dr < tr) word |= 1u << j;
                if ((unsigned long long)dd < td) word |= 1u << (16 + j);
            }
        }
        bonds[w] = word;
    }
}

// step (3): labels are canonical roots (k_flatten_generic ran); the reflection is two fused multiply-adds
__global__ void k_xy_flip(const uint32_t *__restrict__ labels, double2 *__restrict__ spins, Params P, double rx, double ry)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) {
        const uint32_t root = labels[i];
        const uint4 w = philox4x32_10(root, 0u, P.t, kPurposeFlip, P);
        if (state_from_draw(w.x, 2u) == 1u) {
            const double2 s = spins[i];
            const double m = __dmul_rn(-2.0, xy_projection(s, rx, ry));
            spins[i] = make_double2(__fma_rn(m, rx, s.x), __fma_rn(m, ry, s.y));
        }
    }
}

// observables: out[0] = sum over bonds of s_i . s_j, out[1..2] = sum of the spins; roots counted into row[1]
__global__ void __launch_bounds__(kObsThreads)
k_xy_observe(const double2 *__restrict__ spins, const uint32_t *__restrict__ labels, Params P, uint32_t want_clusters,
             double *out, unsigned long long *row)
{
    __shared__ double s_red[3][kObsThreads / 32];
    __shared__ unsigned long long s_scratch[kObsThreads / 32];
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t L = P.L;
    double e = 0.0, mx = 0.0, my = 0.0;
    unsigned long long roots = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) {
        const uint64_t y = i / L, x = i - y * L;
        const double2 s = spins[i], sr = spins[y * L + (x + 1 == L ? 0 : x + 1)], sd = spins[(y + 1 == L ? 0 : y + 1) * L + x];
        e += s.x * sr.x + s.y * sr.y + s.x * sd.x + s.y * sd.y;
        mx += s.x; my += s.y;
        if (want_clusters) roots += (labels[i] == (uint32_t)i);
    }
    double v[3] = {e, mx, my};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xFFFFFFFFu, v[k], o);
        if ((threadIdx.x & 31) == 0) s_red[k][threadIdx.x >> 5] = v[k];
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        double t = 0.0;
        for (int w = 0; w < kObsThreads / 32; ++w) t += s_red[threadIdx.x][w];
        atomicAdd(out + threadIdx.x, t);
    }
    if (want_clusters) block_add_u64(roots, row + 1, s_scratch);
}

}  // namespace sw

struct sw_xy {
    uint32_t L = 0;
    uint64_t N = 0, seed = 0, t = 0;
    double K = 0, last_r[2] = {0, 0};
    int device = 0;
    bool have_spins = false, have_labels = false;
    cudaStream_t stream = nullptr;
    uint8_t *ws = nullptr;
    double2 *spins = nullptr;
    uint32_t *bonds = nullptr, *labels = nullptr, *sizes = nullptr;
    uint8_t *stage = nullptr;
    size_t stage_bytes = 0, ws_bytes = 0;
    double *obs = nullptr;
    unsigned long long *row = nullptr;
    uint64_t launches = 0;
    std::string err;
};

namespace {

int xfail(sw_xy *c, int code, const char *what) { if (c) c->err = what; return code; }
int xcuda(sw_xy *c, cudaError_t e, const char *what) { if (c) c->err = std::string(what) + ": " + cudaGetErrorString(e); return SW_ERR_CUDA; }
#define SX_CUDA(c, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return xcuda((c), e_, #call); } while (0)

struct XyGuard {
    int prev = -1;
    explicit XyGuard(const sw_xy *c) { if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) cudaSetDevice(c->device); else prev = -1; }
    ~XyGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

sw::Params xy_params(const sw_xy *c, uint64_t t) { return swh::make_params(c->L, 2, c->N, c->seed, 1, t); }
int xy_grid(uint64_t items, int threads) { return (int)std::max<uint64_t>(1, std::min<uint64_t>((items + threads - 1) / threads, 148 * 16)); }

// the direction of sweep t: angle 2 pi (w0 + 1/2) / 2^32 of Philox(counter (0, 0, t, REFLECT), key seed); host, once per sweep
void xy_reflection(const sw_xy *c, uint32_t t, double r[2])
{
    const uint64_t M0 = 0xD2511F53ull, M1 = 0xCD9E8D57ull;
    uint32_t c0 = 0, c1 = 0, c2 = t, c3 = sw::kPurposeReflect, k0 = (uint32_t)c->seed, k1 = (uint32_t)(c->seed >> 32);
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = M0 * c0, p1 = M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    const double two_pi = 6.283185307179586476925286766559;
    const double phi = two_pi * (((double)c0 + 0.5) * (1.0 / 4294967296.0));
    r[0] = std::cos(phi);
    r[1] = std::sin(phi);
}

}  // namespace

extern "C" {

int sw_xy_create(sw_xy **out, uint32_t L, double K, uint64_t seed)
{
    if (!out) return SW_ERR_INVALID_ARG;
    *out = nullptr;
    if (L < 2 || L > 65536 || std::isnan(K) || K < 0.0) return SW_ERR_INVALID_ARG;
    sw_xy *c = new (std::nothrow) sw_xy();
    if (!c) return SW_ERR_OOM;
    c->L = L; c->N = (uint64_t)L * L; c->K = K; c->seed = seed;
    if (cudaGetDevice(&c->device) != cudaSuccess) { delete c; return SW_ERR_CUDA; }
    size_t off = 0;
    auto carve = [&](size_t bytes) { const size_t at = off; off = swh::align_up(off + bytes); return at; };
    const size_t o_spins = carve(c->N * 16), o_bonds = carve(((c->N + 15) / 16) * 4), o_labels = carve(c->N * 4), o_sizes = carve(c->N * 4);
    c->stage_bytes = (size_t)std::min<uint64_t>(c->N, 32ull << 20);
    const size_t o_stage = carve(c->stage_bytes), o_obs = carve(3 * 8), o_row = carve(5 * 8);
    c->ws_bytes = off;
    if (cudaMalloc(&c->ws, off) != cudaSuccess) { cudaGetLastError(); delete c; return SW_ERR_OOM; }
    if (cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) != cudaSuccess) { cudaFree(c->ws); delete c; return SW_ERR_CUDA; }
    c->spins = (double2 *)(c->ws + o_spins); c->bonds = (uint32_t *)(c->ws + o_bonds); c->labels = (uint32_t *)(c->ws + o_labels);
    c->sizes = (uint32_t *)(c->ws + o_sizes); c->stage = c->ws + o_stage; c->obs = (double *)(c->ws + o_obs); c->row = (unsigned long long *)(c->ws + o_row);
    *out = c;
    return SW_OK;
}

void sw_xy_destroy(sw_xy *c)
{
    if (!c) return;
    XyGuard g(c);
    cudaStreamSynchronize(c->stream);
    cudaFree(c->ws);
    cudaStreamDestroy(c->stream);
    delete c;
}

int sw_xy_init(sw_xy *c, int mode)
{
    if (!c) return SW_ERR_INVALID_ARG;
    XyGuard g(c);
    const sw::Params P = xy_params(c, 0);
    if (mode == SW_INIT_ORDERED) sw::k_xy_ordered<<<xy_grid(c->N, 256), 256, 0, c->stream>>>(c->spins, P);
    else if (mode == SW_INIT_RANDOM) sw::k_xy_init_random<<<xy_grid(c->N, 256), 256, 0, c->stream>>>(c->spins, P);
    else return xfail(c, SW_ERR_INVALID_ARG, "sw_xy_init: unknown mode");
    SX_CUDA(c, cudaGetLastError());
    c->launches += 1;
    c->t = 0; c->have_spins = true; c->have_labels = false;
    return SW_OK;
}

int sw_xy_set_state(sw_xy *c, const double *src, uint64_t t)
{
    if (!c || !src || t > 0xFFFFFFFFull) return xfail(c, SW_ERR_INVALID_ARG, "sw_xy_set_state: bad argument");
    for (uint64_t i = 0; i < 2 * c->N; ++i) if (!std::isfinite(src[i])) return xfail(c, SW_ERR_INVALID_ARG, "sw_xy_set_state: spin component not finite");
    XyGuard g(c);
    SX_CUDA(c, cudaMemcpyAsync(c->spins, src, c->N * 16, cudaMemcpyHostToDevice, c->stream));
    SX_CUDA(c, cudaStreamSynchronize(c->stream));
    c->t = t; c->have_spins = true; c->have_labels = false;
    return SW_OK;
}

int sw_xy_sweep(sw_xy *c, uint64_t n)
{
    if (!c) return SW_ERR_INVALID_ARG;
    if (!c->have_spins) return xfail(c, SW_ERR_STATE, "sw_xy_sweep: no spins (call sw_xy_init or sw_xy_set_state)");
    if (c->t + n > 0x100000000ull) return xfail(c, SW_ERR_STATE, "sw_xy_sweep: sweep counter would pass 2^32");
    XyGuard g(c);
    const int th = 256;
    for (uint64_t k = 0; k < n; ++k) {
        const sw::Params P = xy_params(c, c->t);
        double r[2];
        xy_reflection(c, (uint32_t)c->t, r);
        sw::k_xy_bonds<<<xy_grid((c->N + 15) / 16, th), th, 0, c->stream>>>(c->spins, c->bonds, P, 2.0 * c->K, r[0], r[1]);
        sw::k_label_identity<<<xy_grid(c->N, th), th, 0, c->stream>>>(c->labels, P);
        sw::k_union_generic<<<xy_grid(c->N, th), th, 0, c->stream>>>(c->bonds, c->labels, P);
        sw::k_flatten_generic<<<xy_grid(c->N, th), th, 0, c->stream>>>(c->labels, P);
        sw::k_xy_flip<<<xy_grid(c->N, th), th, 0, c->stream>>>(c->labels, c->spins, P, r[0], r[1]);
        c->launches += 5;
        c->last_r[0] = r[0]; c->last_r[1] = r[1];
        c->t += 1;
        c->have_labels = true;
    }
    SX_CUDA(c, cudaGetLastError());
    return SW_OK;
}

int sw_xy_measure(sw_xy *c, double *energy_sum, double mag[2], uint64_t *n_clusters, uint64_t *largest_cluster)
{
    if (!c) return SW_ERR_INVALID_ARG;
    if (!c->have_spins) return xfail(c, SW_ERR_STATE, "sw_xy_measure: no spins");
    XyGuard g(c);
    const sw::Params P = xy_params(c, c->t);
    const bool cl = c->have_labels && (n_clusters || largest_cluster), big = c->have_labels && largest_cluster;
    SX_CUDA(c, cudaMemsetAsync(c->obs, 0, 3 * 8, c->stream));
    SX_CUDA(c, cudaMemsetAsync(c->row, 0, 5 * 8, c->stream));
    sw::k_xy_observe<<<xy_grid(c->N, sw::kObsThreads), sw::kObsThreads, 0, c->stream>>>(c->spins, c->labels, P, cl ? 1u : 0u, c->obs, c->row);
    c->launches += 1;
    if (big) {
        SX_CUDA(c, cudaMemsetAsync(c->sizes, 0, c->N * 4, c->stream));
        sw::k_cluster_sizes<<<xy_grid((c->N + 15) / 16, 256), 256, 0, c->stream>>>(c->labels, c->sizes, P);
        sw::k_max_size<<<xy_grid(c->N, 256), 256, 0, c->stream>>>(c->sizes, P, c->row);
        c->launches += 2;
    }
    SX_CUDA(c, cudaGetLastError());
    double obs[3];
    uint64_t row[5];
    SX_CUDA(c, cudaMemcpyAsync(obs, c->obs, sizeof(obs), cudaMemcpyDeviceToHost, c->stream));
    SX_CUDA(c, cudaMemcpyAsync(row, c->row, sizeof(row), cudaMemcpyDeviceToHost, c->stream));
    SX_CUDA(c, cudaStreamSynchronize(c->stream));
    if (row[1] == 1) row[2] = c->N;
    if (energy_sum) *energy_sum = obs[0];
    if (mag) { mag[0] = obs[1]; mag[1] = obs[2]; }
    if (n_clusters) *n_clusters = c->have_labels ? row[1] : 0;
    if (largest_cluster) *largest_cluster = c->have_labels ? row[2] : 0;
    return SW_OK;
}

int sw_xy_get_spins(sw_xy *c, double *dst)
{
    if (!c || !dst) return SW_ERR_INVALID_ARG;
    if (!c->have_spins) return xfail(c, SW_ERR_STATE, "no spins");
    XyGuard g(c);
    SX_CUDA(c, cudaMemcpyAsync(dst, c->spins, c->N * 16, cudaMemcpyDeviceToHost, c->stream));
    SX_CUDA(c, cudaStreamSynchronize(c->stream));
    return SW_OK;
}

int sw_xy_get_labels(sw_xy *c, uint32_t *dst)
{
    if (!c || !dst) return SW_ERR_INVALID_ARG;
    if (!c->have_labels) return xfail(c, SW_ERR_STATE, "no labels: no sweep since sw_xy_init");
    XyGuard g(c);
    SX_CUDA(c, cudaMemcpyAsync(dst, c->labels, c->N * 4, cudaMemcpyDeviceToHost, c->stream));
    SX_CUDA(c, cudaStreamSynchronize(c->stream));
    return SW_OK;
}

int sw_xy_get_bonds(sw_xy *c, uint8_t *dst)
{
    if (!c || !dst) return SW_ERR_INVALID_ARG;
    if (!c->have_labels) return xfail(c, SW_ERR_STATE, "no bonds: no sweep since sw_xy_init");
    XyGuard g(c);
    for (uint64_t done = 0; done < c->N;) {
        const uint64_t m = std::min<uint64_t>(c->N - done, c->stage_bytes);
        sw::k_expand_bonds<<<xy_grid(m, 256), 256, 0, c->stream>>>(c->bonds, c->stage, done, m);
        c->launches += 1;
        SX_CUDA(c, cudaMemcpyAsync(dst + done, c->stage, m, cudaMemcpyDeviceToHost, c->stream));
        SX_CUDA(c, cudaStreamSynchronize(c->stream));
        done += m;
    }
    return SW_OK;
}

int sw_xy_get_reflection(sw_xy *c, double r[2])
{
    if (!c || !r) return SW_ERR_INVALID_ARG;
    if (!c->have_labels) return xfail(c, SW_ERR_STATE, "no sweep since sw_xy_init");
    r[0] = c->last_r[0]; r[1] = c->last_r[1];
    return SW_OK;
}

int sw_xy_get_time(sw_xy *c, uint64_t *t)
{
    if (!c || !t) return SW_ERR_INVALID_ARG;
    *t = c->t;
    return SW_OK;
}

const char *sw_xy_last_error(const sw_xy *c) { return c ? c->err.c_str() : "null context"; }

}  // extern "C"
