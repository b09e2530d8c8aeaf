// sw_observe.cuh -- observables of the current state ("measurement of energy and
// magnetization"; cluster statistics per BASELINE.json config 4).  Runs only on sw_measure /
// sw_sweep_measure.  All accumulators are 64-bit: energy_bonds can reach 2^33 at L = 65536.
//
// Result row layout (device uint64): [0] energy_bonds, [1] n_clusters, [2] largest_cluster,
// [3 .. 3+q) mag_counts.
#pragma once

#include "sw_common.cuh"

namespace sw {

constexpr int kObsThreads = 256;

__device__ __forceinline__ void block_add_u64(unsigned long long v, unsigned long long *dst, unsigned long long *s_scratch)
{
    // warp shuffle reduce, then one atomic per block
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) s_scratch[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = (lane < (blockDim.x >> 5)) ? s_scratch[lane] : 0ull;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
        if (lane == 0 && v) atomicAdd(dst, v);
    }
}

// n_clusters on the tiled path: the flip kernel has counted the canonical roots of every tile
__global__ void __launch_bounds__(kObsThreads)
k_sum_tile_clusters(const uint32_t *__restrict__ tile_clusters, uint32_t n_tiles, unsigned long long *row)
{
    __shared__ unsigned long long s_scratch[kObsThreads / 32];
    unsigned long long v = 0;
    for (uint32_t k = blockIdx.x * blockDim.x + threadIdx.x; k < n_tiles; k += gridDim.x * blockDim.x) v += tile_clusters[k];
    block_add_u64(v, row + 1, s_scratch);
}

// Scalar version: any L.  want: bit0 energy, bit1 magnetisation, bit2 n_clusters.
__global__ void __launch_bounds__(kObsThreads)
k_observe_scalar(const uint8_t *__restrict__ spins, const uint32_t *__restrict__ labels, Params P,
                 uint32_t want, unsigned long long *row)
{
    __shared__ unsigned int s_hist[256];
    __shared__ unsigned long long s_scratch[kObsThreads / 32];
    for (int k = threadIdx.x; k < 256; k += blockDim.x) s_hist[k] = 0;
    __syncthreads();
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t L = P.L;
    unsigned long long e = 0, roots = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) {
        const uint8_t s = spins[i];
        if (want & 1u) {
            const uint64_t y = i / L, x = i - y * L;
            e += (s == spins[y * L + (x + 1 == L ? 0 : x + 1)]);
            e += (s == spins[(y + 1 == L ? 0 : y + 1) * L + x]);
        }
        if (want & 2u) atomicAdd(&s_hist[s], 1u);
        if (want & 4u) roots += (labels[i] == (uint32_t)i);
    }
    __syncthreads();
    if (want & 2u)
        for (int k = threadIdx.x; k < (int)P.q; k += blockDim.x)
            if (s_hist[k]) atomicAdd(row + 3 + k, (unsigned long long)s_hist[k]);
    if (want & 1u) block_add_u64(e, row + 0, s_scratch);
    if (want & 4u) block_add_u64(roots, row + 1, s_scratch);
}

// Vector version: L % 16 == 0; one thread per block of 4 rows x 16 consecutive sites.
__global__ void __launch_bounds__(kObsThreads)
k_observe_vec16(const uint8_t *__restrict__ spins, const uint32_t *__restrict__ labels, Params P,
                uint32_t want, unsigned long long *row)
{
    __shared__ unsigned int s_hist[256];
    __shared__ unsigned long long s_scratch[kObsThreads / 32];
    for (int k = threadIdx.x; k < 256; k += blockDim.x) s_hist[k] = 0;
    __syncthreads();
    // unit of work: 4 rows x 16 columns (L % 16 == 0), so the row below is re-read once per 4 rows, not once per row
    const uint32_t n_units = (uint32_t)(P.N >> 6);         // <= 2^26: 32-bit index arithmetic throughout
    const uint32_t stride = gridDim.x * blockDim.x;
    const uint32_t L = P.L, gpr = L >> 4;                  // 16-site groups per row
    unsigned long long e = 0, roots = 0;
    unsigned int cnt[4] = {0, 0, 0, 0};                    // q <= 4 fast path
    for (uint32_t u = blockIdx.x * blockDim.x + threadIdx.x; u < n_units; u += stride) {
        const uint32_t y4 = u / gpr, gx = u - y4 * gpr, y0 = y4 << 2;
        const uint32_t x0 = gx << 4, xn = (gx + 1 == gpr) ? 0u : ((gx + 1) << 4);
        uint4 rows[5];
        uint32_t nxt[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            rows[r] = *reinterpret_cast<const uint4 *>(spins + (uint64_t)(y0 + r) * L + x0);
            if (want & 1u) nxt[r] = spins[(uint64_t)(y0 + r) * L + xn];
        }
        if (want & 1u) rows[4] = *reinterpret_cast<const uint4 *>(spins + (uint64_t)((y0 + 4 == L) ? 0u : y0 + 4) * L + x0);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const uint32_t w[4] = {rows[r].x, rows[r].y, rows[r].z, rows[r].w};
            if (want & 1u) {
                const uint32_t dw[4] = {rows[r + 1].x, rows[r + 1].y, rows[r + 1].z, rows[r + 1].w};
                uint32_t acc = 0;                              // per byte lane: equal pairs seen (<= 8)
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t hi = (k < 3) ? w[k + 1] : nxt[r];
                    const uint32_t rn = __funnelshift_r(w[k], hi, 8);        // the right neighbours of the 4 bytes
                    acc += (__vcmpeq4(w[k], rn) & 0x01010101u) + (__vcmpeq4(w[k], dw[k]) & 0x01010101u);
                }
                e += (acc * 0x01010101u) >> 24;
            }
            if (want & 2u) {
                if (P.q <= 4) {
                    // states are two bits per byte: per byte lane, count bit 0, bit 1 and both (each <= 4 over the 4 words)
                    uint32_t s0 = 0, s1 = 0, s3 = 0;
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const uint32_t b0 = w[k] & 0x01010101u, b1 = (w[k] >> 1) & 0x01010101u;
                        s0 += b0; s1 += b1; s3 += b0 & b1;
                    }
                    const uint32_t n3 = (s3 * 0x01010101u) >> 24;
                    const uint32_t n1 = ((s0 * 0x01010101u) >> 24) - n3, n2 = ((s1 * 0x01010101u) >> 24) - n3;
                    cnt[0] += 16u - n1 - n2 - n3; cnt[1] += n1; cnt[2] += n2; cnt[3] += n3;
                } else {
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        atomicAdd(&s_hist[w[k] & 0xFF], 1u);
                        atomicAdd(&s_hist[(w[k] >> 8) & 0xFF], 1u);
                        atomicAdd(&s_hist[(w[k] >> 16) & 0xFF], 1u);
                        atomicAdd(&s_hist[w[k] >> 24], 1u);
                    }
                }
            }
            if (want & 4u) {
                const uint64_t base = (uint64_t)(y0 + r) * L + x0;
                const uint4 *lp = reinterpret_cast<const uint4 *>(labels + base);
                const uint32_t i0 = (uint32_t)base;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint4 l = lp[k];
                    roots += (l.x == i0 + 4 * k) + (l.y == i0 + 4 * k + 1) + (l.z == i0 + 4 * k + 2) + (l.w == i0 + 4 * k + 3);
                }
            }
        }
    }
    if ((want & 2u) && P.q <= 4) {
#pragma unroll
        for (uint32_t a = 0; a < 4; ++a) if (cnt[a]) atomicAdd(&s_hist[a], cnt[a]);
    }
    __syncthreads();
    if (want & 2u)
        for (int k = threadIdx.x; k < (int)P.q; k += blockDim.x)
            if (s_hist[k]) atomicAdd(row + 3 + k, (unsigned long long)s_hist[k]);
    if (want & 1u) block_add_u64(e, row + 0, s_scratch);
    if (want & 4u) block_add_u64(roots, row + 1, s_scratch);
}

// sizes[root(i)] += 1.  Clusters are spatially coherent, so a thread's 16 consecutive sites usually belong to one or two
// clusters: it counts them in two private slots (a third label evicts the slot with the smaller count), and at the end of
// the group the lanes of a warp that hold the same root add their counts up (match_any + reduce) so that ONE lane does the
// atomic.  At criticality one cluster holds a large fraction of all sites: without the two slots every hole in it cost an
// atomic on the same address, and without the warp step 2^32 / 16 threads queued up on that one address (420 ms per call at
// L = 65536; SURVEY.md sec. 8 config 4's largest_cluster through sw_measure).  Works on a forest too.
__device__ __forceinline__ void warp_add_size(uint32_t *sizes, uint32_t root, uint32_t n)
{
    const unsigned here = __activemask();
    const unsigned has = __ballot_sync(here, n != 0u);
    if (n) {
        const unsigned peers = __match_any_sync(has, root);
        const uint32_t total = __reduce_add_sync(peers, n);
        if ((threadIdx.x & 31u) == (uint32_t)__ffs(peers) - 1u) atomicAdd(sizes + root, total);
    }
}

__global__ void k_cluster_sizes(const uint32_t *__restrict__ labels, uint32_t *sizes, Params P)
{
    const uint64_t n_groups = (P.N + 15) >> 4;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t g = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; g < n_groups; g += stride) {
        uint32_t ra = 0, na = 0, rb = 0, nb = 0;
        for (uint32_t j = 0; j < 16; ++j) {
            const uint64_t i = (g << 4) + j;
            if (i >= P.N) break;
            uint32_t l = labels[i];
            if (l != (uint32_t)i) l = find_root(labels, l);
            if (na && l == ra) ++na;
            else if (nb && l == rb) ++nb;
            else if (!na) { ra = l; na = 1; }
            else if (!nb) { rb = l; nb = 1; }
            else if (na < nb) { atomicAdd(sizes + ra, na); ra = l; na = 1; }
            else { atomicAdd(sizes + rb, nb); rb = l; nb = 1; }
        }
        warp_add_size(sizes, ra, na);
        warp_add_size(sizes, rb, nb);
    }
}

// row[2] = max over roots of sizes[]; only roots (labels[i] == i) hold a count
__global__ void k_max_size(const uint32_t *__restrict__ sizes, Params P, unsigned long long *row)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint32_t m = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride)
        m = max(m, sizes[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xFFFFFFFFu, m, o));
    if ((threadIdx.x & 31) == 0 && m) atomicMax(row + 2, (unsigned long long)m);
}

// the same, and every counter that was read non-zero is set back to zero: sizes[] stays all zero between measurements
// (the counting sweeps rely on that), without a memset of 4N bytes per measurement.  A site without any bond is a
// cluster of one whose counter may have been left at zero (k_tile_blocks_sizes): the maximum is at least 1.
__global__ void k_max_size_zero(uint32_t *__restrict__ sizes, Params P, unsigned long long *row)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x * 4;
    uint32_t m = (blockIdx.x == 0 && threadIdx.x == 0) ? 1u : 0u;
    for (uint64_t i = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4; i < P.N; i += stride) {    // N % 4 == 0 on the tiled path
        const uint4 v = *reinterpret_cast<const uint4 *>(sizes + i);
        if (v.x | v.y | v.z | v.w) {
            m = max(m, max(max(v.x, v.y), max(v.z, v.w)));
            *reinterpret_cast<uint4 *>(sizes + i) = make_uint4(0, 0, 0, 0);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xFFFFFFFFu, m, o));
    if ((threadIdx.x & 31) == 0 && m) atomicMax(row + 2, (unsigned long long)m);
}

// Moments of the cluster-size distribution from sizes[] (only roots hold a count): row[2] = max, and the 128-bit sum of
// squares c2[0] + 2^64 c2[1] = sum over clusters of |c|^2 -- the improved estimator of the susceptibility (the cluster
// representation of <m^2>).  |c|^2 can reach 2^64 (one cluster of 2^32 sites), hence two words.
__global__ void k_size_moments(const uint32_t *__restrict__ sizes, Params P, unsigned long long *row, unsigned long long *c2)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint32_t m = 0;
    unsigned long long lo = 0, hi = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) {
        const uint32_t sz = sizes[i];
        if (!sz) continue;
        m = max(m, sz);
        const unsigned long long sq = (unsigned long long)sz * sz, before = lo;
        lo += sq;
        hi += lo < before;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        m = max(m, __shfl_xor_sync(0xFFFFFFFFu, m, o));
        const unsigned long long olo = __shfl_xor_sync(0xFFFFFFFFu, lo, o), ohi = __shfl_xor_sync(0xFFFFFFFFu, hi, o), before = lo;
        lo += olo;
        hi += ohi + (lo < before);
    }
    if ((threadIdx.x & 31) == 0) {
        if (m) atomicMax(row + 2, (unsigned long long)m);
        if (lo | hi) {
            const unsigned long long old = atomicAdd(c2, lo);
            if (old + lo < old) hi += 1;
            if (hi) atomicAdd(c2 + 1, hi);
        }
    }
}

}  // namespace sw
