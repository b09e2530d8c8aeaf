// sw_cluster.cuh -- the small-lattice path: ONE launch per sw_sweep(n) / sw_sweep_measure(n).
//
// Lattices of at most 16 tiles (L = 64 ... 256; BASELINE.json config 1 is L = 256, 200 sweeps, observables every
// sweep) are bound by launch latency on the three-kernel path: three launches of <= 16 CTAs per sweep.  Here the
// tiles are the CTAs of ONE thread-block cluster (<= 16 CTAs, one per SM, co-scheduled by the hardware), the three
// steps of the sweep are phases of one persistent kernel separated by the cluster's hardware barrier
// (barrier.cluster: release / acquire at cluster scope) instead of kernel boundaries, and the kernel loops over the n
// sweeps; the observables of sw_sweep_measure go to a device ring, one row per sweep, with no host round trip.
// The phases are the very bodies of k_tile_blocks / k_tile_merge / k_tile_flip (sw_tile_blocks.cuh, sw_tiled.cuh),
// so the results are bit-identical by construction; data another CTA wrote in an earlier phase is read from L2.
#pragma once

#include <cooperative_groups.h>

#include "sw_common.cuh"
#include "sw_observe.cuh"
#include "sw_tile_blocks.cuh"
#include "sw_tiled.cuh"

namespace sw {

constexpr int kClusterThreads = kBlkThreads;          // 128: the tile body's thread count; the flip body runs with 8 accesses per thread
constexpr uint32_t kClusterMaxTiles = 16;             // largest (non-portable) cluster size

struct ObserveShared {
    unsigned int hist[256];
    unsigned long long scratch[kClusterThreads / 32];
};

union ClusterShared {
    BlkShared blk;
    MergeShared merge;
    FlipShared<kClusterThreads> flip;
    ObserveShared obs;
};

// observables of tile (tx, ty) after the flip, thread (bx, by) looks at the 8 x 4 block the tile kernel gave it:
// equal pairs (right and down, periodic), state histogram, cluster sizes (sizes[root] += members, run-length
// aggregated along the rows); `what`: SW_OBS_* bits 1 energy, 2 magnetisation, 8 largest cluster
__device__ __forceinline__ void
cluster_observe_tile(ObserveShared &S, uint32_t tx, uint32_t ty, const uint8_t *spins, const uint32_t *labels, uint32_t *sizes,
                     const Params &P, uint32_t what, unsigned long long *row)
{
    const uint32_t tid = threadIdx.x, bx = tid & 7u, by = tid >> 3, L = P.L;
    const uint32_t x0 = (tx << 6) + (bx << 3), y0 = (ty << 6) + (by << 2);
    for (uint32_t k = tid; k < 256; k += kClusterThreads) S.hist[k] = 0;
    __syncthreads();
    unsigned long long e = 0;
    if (what & 3u) {
        const uint32_t xr = (x0 + 8u == L) ? 0u : x0 + 8u;
        uint2 s[5];
#pragma unroll
        for (int r = 0; r < 5; ++r) {
            const uint32_t y = (y0 + r == L) ? 0u : y0 + r;
            s[r] = __ldcg(reinterpret_cast<const uint2 *>(spins + (uint64_t)y * L + x0));
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const uint32_t nb = __ldcg(spins + (uint64_t)(y0 + r) * L + xr);
            const uint32_t a0 = s[r].x, a1 = s[r].y;
            const uint32_t n0 = __funnelshift_r(a0, a1, 8), n1 = __funnelshift_r(a1, nb, 8);
            if (what & 1u) {
                const uint32_t acc = (__vcmpeq4(a0, n0) & 0x01010101u) + (__vcmpeq4(a1, n1) & 0x01010101u) +
                                     (__vcmpeq4(a0, s[r + 1].x) & 0x01010101u) + (__vcmpeq4(a1, s[r + 1].y) & 0x01010101u);
                e += (acc * 0x01010101u) >> 24;
            }
            if (what & 2u) {
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    atomicAdd(&S.hist[(a0 >> (8 * c)) & 0xFFu], 1u);
                    atomicAdd(&S.hist[(a1 >> (8 * c)) & 0xFFu], 1u);
                }
            }
        }
    }
    if (what & 8u) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const uint4 *lp = reinterpret_cast<const uint4 *>(labels + (uint64_t)(y0 + r) * L + x0);
            const uint4 l0 = __ldcg(lp), l1 = __ldcg(lp + 1);
            const uint32_t lab[8] = {l0.x, l0.y, l0.z, l0.w, l1.x, l1.y, l1.z, l1.w};
            uint32_t cur = lab[0], run = 1;
#pragma unroll
            for (int c = 1; c < 8; ++c) {
                if (lab[c] == cur) { ++run; continue; }
                atomicAdd(sizes + cur, run);
                cur = lab[c]; run = 1;
            }
            atomicAdd(sizes + cur, run);
        }
    }
    __syncthreads();
    if (what & 2u)
        for (uint32_t k = tid; k < P.q; k += kClusterThreads)
            if (S.hist[k]) atomicAdd(row + 3 + k, (unsigned long long)S.hist[k]);
    if (what & 1u) block_add_u64(e, row + 0, S.scratch);
}

// kMeasure: after every sweep, the observables `what` (SW_OBS_* bits) go to rows[sweep][3 + q] (zeroed by the host)
template <bool kMeasure>
__global__ void __launch_bounds__(kClusterThreads, 1)
k_cluster_sweeps(uint8_t *spins, uint32_t *bonds, uint32_t *labels, uint16_t *rootbits, TileBorder *border, TileEdges *edges,
                 uint2 *draws, uint32_t *tile_clusters, Params P, uint32_t n_sweeps, uint32_t what, unsigned long long *rows,
                 uint32_t *sizes)
{
    __shared__ ClusterShared S;
    cooperative_groups::cluster_group cluster = cooperative_groups::this_cluster();
    const uint32_t tx = blockIdx.x, ty = blockIdx.y, tile = ty * (P.L >> 6) + tx;
    const uint32_t tid = threadIdx.x;
    const Dom none{};

    for (uint32_t s = 0; s < n_sweeps; ++s) {
        uint32_t pk_t[3], pk_n[3];
        sweep_keys(P, P.t + s, pk_t);
        sweep_keys(P, P.t + s + 1u, pk_n);

        // -- phase 1: bonds + tile-local labels (a1 + a2)
        if (kMeasure && (what & 8u)) {                        // cluster-size counters of my tile: zero
            const uint32_t x0 = (tx << 6) + ((tid & 7u) << 3), y0 = (ty << 6) + ((tid >> 3) << 2);
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                uint4 *zp = reinterpret_cast<uint4 *>(sizes + (uint64_t)(y0 + r) * P.L + x0);
                zp[0] = make_uint4(0, 0, 0, 0); zp[1] = make_uint4(0, 0, 0, 0);
            }
        }
        tile_blocks_body<false, true, CtaBar>(S.blk, tx, ty, spins, bonds, labels, rootbits, border, edges, draws, P, none);
        cluster.sync();
        // -- phase 2: links across the borders of my tile (a3)
        tile_merge_body<false, false, true, MergeBar>(S.merge, labels, border, edges, P, none, tile, tile + 1u, nullptr);
        cluster.sync();
        // -- phase 3: canonical labels + new spins (a4 + a5), the bond draws of the next sweep, cluster count of my tile
        tile_flip_body<true, true, true, false, false, kClusterThreads, MergeBar>(
            S.flip, tx, ty, labels, rootbits, spins, P, pk_t, pk_n, none, tile_clusters, draws, nullptr);
        cluster.sync();
        // -- observables (a6)
        if (kMeasure) {
            unsigned long long *row = rows + (size_t)s * (3u + P.q);
            cluster_observe_tile(S.obs, tx, ty, spins, labels, sizes, P, what, row);
            if ((what & 12u) && tid == 0) {
                unsigned long long nc = 0;
                for (uint32_t w = 0; w < kClusterThreads / 32; ++w) nc += tile_clusters[tile * (kClusterThreads / 32) + w];
                atomicAdd(row + 1, nc);
            }
            if (what & 8u) {
                cluster.sync();                               // all sizes[] are complete
                const uint32_t x0 = (tx << 6) + ((tid & 7u) << 3), y0 = (ty << 6) + ((tid >> 3) << 2);
                uint32_t m = 0;
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const uint4 *zp = reinterpret_cast<const uint4 *>(sizes + (uint64_t)(y0 + r) * P.L + x0);
                    const uint4 a = __ldcg(zp), b = __ldcg(zp + 1);
                    m = max(m, max(max(max(a.x, a.y), max(a.z, a.w)), max(max(b.x, b.y), max(b.z, b.w))));
                }
                m = __reduce_max_sync(0xFFFFFFFFu, m);
                if ((tid & 31u) == 0 && m) atomicMax(row + 2, (unsigned long long)m);
            }
            __syncthreads();                                  // S.obs is reused as S.blk by the next sweep
        }
    }
}

}  // namespace sw
