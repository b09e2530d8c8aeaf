// sw_tiled.cuh -- the hot path of libsw.so for L % 64 == 0: three kernels per sweep.
//
//   k_tile_blocks   step (1) + tile-local part of step (2)   (sw_tile_blocks.cuh)
//   k_tile_merge    union-find over the bonds that cross a tile border (PAPER.md:66-68 uses the
//                   same boundary-only idea one level up, between GPUs)
//   k_tile_flip     pointer-jumping flatten to the canonical root ("tracks back
//                   the label variable until [it] remains unchanged") fused with step (3)
//
// A tile is 64 x 64 sites.  Between the tile kernel and the flip kernel, labels[] holds
//   * at a tile-local root (a set bit of `rootbits`): its link into the global forest -- itself, or
//     the smaller root the merge hooked it under (a global site index);
//   * at any other site: the TILE-LOCAL id (y * 64 + x, 12 bits) of its tile-local root, so the flip
//     kernel needs no index arithmetic to find it.
// After the flip kernel (eager mode) every entry is the canonical root (global site index).
#pragma once

#include "sw_common.cuh"

namespace sw {

constexpr uint32_t kTile = 64;                       // tile edge
constexpr uint32_t kTileSites = kTile * kTile;       // 4096
constexpr int kMergeThreads = 128;

// per-tile record of the bonds that leave the tile (written by the tile kernel, read by k_tile_merge)
struct __align__(16) TileBorder {
    unsigned long long right_col;   // bit y: bond (X0+63, Y0+y) -> (X0+64, Y0+y)
    unsigned long long bottom_row;  // bit x: bond (X0+x, Y0+63) -> (X0+x, Y0+64)
};

// per-tile copy of the tile-local roots (global site indices) of the four edges of the tile (written by the
// tile kernel, read by k_tile_merge): the merge never has to decode labels[], and a column costs 256
// contiguous bytes instead of one 32-byte sector per site
struct __align__(16) TileEdges {
    uint32_t left[kTile];           // root of site (X0,      Y0 + y)
    uint32_t right[kTile];          // root of site (X0 + 63, Y0 + y)
    uint32_t top[kTile];            // root of site (X0 + x,  Y0)
    uint32_t bottom[kTile];         // root of site (X0 + x,  Y0 + 63)
};

// the four 0x00/0xFF bytes of a __vcmpeq4 result -> 4 bits
__device__ __forceinline__ uint32_t pack4(uint32_t eq) { return ((eq & 0x01010101u) * 0x01020408u) >> 24; }

// ---- bond draws, made ahead of time ------------------------------------------------------------
// Whether a bond's draw is below the threshold depends on (seed, sweep, site) only, not on the spins (counter-based
// Philox, R11), so the tests of sweep t + 1 can be made while sweep t is still running.  The tile kernel is
// bound by its integer ALU pipe and a quarter of its instructions were these draws; the flip kernel waits for HBM and
// has the issue slots to spare.  One uint2 per 8 x 4 block of the tile kernel (index tile * 128 + block): bit 8r + c
// of .x / .y = the right / down draw of site (r, c) of the block is below the threshold.

// mask * 2 + (draw >= T): add.cc sets the carry iff draw + (2^32 - T) overflows, addc shifts it into the mask
__device__ __forceinline__ uint32_t shift_in_not_below(uint32_t mask, uint32_t draw, uint32_t above)
{
    uint32_t out;
    asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\taddc.u32 %0, %3, %3;\n\t}" : "=r"(out) : "r"(draw), "r"(above), "r"(mask));
    return out;
}

// 256 threads per tile: thread u makes the draws of rows 2h, 2h + 1 (h = u % 2) of block u / 2: one Philox call per
// site pair (words: right, down, right, down), last pair first so that the bits are shifted in in order.
// `origin` = global index of the tile's first site, `Lg` = global row stride (the draws are keyed by the global site)
__device__ __forceinline__ void tile_draw_masks(uint2 *draws, uint32_t tile, uint32_t origin, uint32_t u,
                                                const uint32_t (&pk)[3], const Params &P, const uint32_t Lg)
{
    const uint32_t b = u >> 1, h = u & 1u, bx = b & 7u, by = b >> 3;
    const uint32_t above = ~P.thr_m1;                          // 2^32 - T (T >= 1; T = 0 is masked by thr_any)
    uint32_t off_r = 0, off_d = 0;                             // the draws that are NOT below the threshold
#pragma unroll
    for (int rr = 1; rr >= 0; --rr) {
        const uint32_t pair0 = (origin + ((by << 2) + 2u * h + rr) * Lg + (bx << 3)) >> 1;
#pragma unroll
        for (int p = 3; p >= 0; --p) {
            const uint4 d = philox_sweep(pair0 + p, kPurposeBond, pk, P);
            off_r = shift_in_not_below(off_r, d.z, above);
            off_d = shift_in_not_below(off_d, d.w, above);
            off_r = shift_in_not_below(off_r, d.x, above);
            off_d = shift_in_not_below(off_d, d.y, above);
        }
    }
    const uint32_t m_r = ~off_r & 0xFFFFu & P.thr_any, m_d = ~off_d & 0xFFFFu & P.thr_any;
    const uint32_t o_r = __shfl_xor_sync(0xFFFFFFFFu, m_r, 1), o_d = __shfl_xor_sync(0xFFFFFFFFu, m_d, 1);
    if (h == 0) draws[tile * 128u + b] = make_uint2(m_r | (o_r << 16), m_d | (o_d << 16));
}

// the draws of sweep P.t for every tile (first sweep after sw_init / sw_set_state; later ones come from k_tile_flip)
__global__ void __launch_bounds__(256)
k_draws(uint2 *__restrict__ draws, Params P)
{
    const uint32_t tiles_x = P.L >> 6;
    const uint32_t ty = blockIdx.y, tx = blockIdx.x, tile = ty * tiles_x + tx;   // grid = (tiles_x, tiles_x): no division
    tile_draw_masks(draws, tile, (ty << 6) * P.L + (tx << 6), threadIdx.x, P.pk_t, P, P.L);
}

__global__ void __launch_bounds__(256)
k_draws_super(uint2 *__restrict__ draws, Params P, Dom dom)
{
    const uint32_t tile = blockIdx.y * (dom.W >> 6) + blockIdx.x;
    tile_draw_masks(draws, tile, (dom.oy + (blockIdx.y << 6)) * dom.Lg + dom.ox + (blockIdx.x << 6), threadIdx.x, P.pk_t, P, dom.Lg);
}

// ---- kernel 2: merge across tile borders -------------------------------------------------------
// One thread per border site (64 on the right column, 64 on the bottom row of a tile).  Only about a
// third of them carry a link worth uniting (active bond, not a repeat of its neighbour's link), and a
// unite is a chain of dependent L2 / HBM round trips, so the kernel is latency-bound: a CTA therefore
// gathers the links of kTiles tiles into a dense list first (coalesced loads, all independent)
// and then unites them with every lane busy.  kTiles = 4 for the largest lattices; up to L = 16384 (65536 tiles) two
// tiles per CTA are faster -- more, shorter CTAs: 18.6 instead of 25.3 us at L = 4096 (config 2, where the merge is a
// fifth of the sweep), 35.9 instead of 38.3 us at L = 8192; at L = 65536 four win by 2 % (merge_tiles_per_cta).

constexpr int kMergeTiles = 4;                       // the most a CTA takes (MergeShared is sized for it)
__host__ __device__ constexpr int merge_tiles_per_cta(unsigned n_tiles) { return n_tiles <= 65536u ? 2 : 4; }

struct MergeShared {
    uint2 link[kMergeTiles * kMergeThreads];
    uint32_t n;
};

// The links of tiles [tile_begin, tile_end) (at most kTiles of them), by kMergeThreads threads.
//   kSuper: borders that leave the piece are NOT united here (the inter-domain merge of sw_super.cu does that,
//   PAPER.md:66-68); label values are global, addresses local (DomAddr).
template <bool kStats, bool kSuper, bool kCoherent, class Bar, int kTiles = kMergeTiles>
__device__ __forceinline__ void
tile_merge_body(MergeShared &S, uint32_t *labels, const TileBorder *border, const TileEdges *edges, const Params &P, const Dom &dom,
                const uint32_t tile_begin, const uint32_t tile_end, PassCounters *counters)
{
    const uint32_t b = threadIdx.x, lane = b & 31u;
    const uint32_t tiles_x = (kSuper ? dom.W : P.L) >> 6, tiles_y = (kSuper ? dom.H : P.L) >> 6;
    if (b == 0) S.n = 0;
    Bar::sync();

    static_assert(kTiles <= kMergeTiles, "MergeShared holds the links of kMergeTiles tiles");
    uint32_t lu[kTiles], lv[kTiles];
    bool on[kTiles];
#pragma unroll
    for (int i = 0; i < kTiles; ++i) {
        const uint32_t tile = tile_begin + i;
        on[i] = false; lu[i] = 0; lv[i] = 0;
        if (tile < tile_end) {
            const uint32_t ty = tile / tiles_x, tx = tile - ty * tiles_x;
            TileBorder rec;
            if (kCoherent) {
                const ulonglong2 v = __ldcg(reinterpret_cast<const ulonglong2 *>(border + tile));
                rec.right_col = v.x; rec.bottom_row = v.y;
            } else rec = border[tile];
            const uint32_t *pu, *pv;
            unsigned long long mask;
            uint32_t k;
            bool inside = true;
            if (b < kTile) {                                 // right column -- left column of the tile on the right
                k = b; mask = rec.right_col;
                pu = edges[tile].right + k;
                pv = edges[(tx + 1 == tiles_x) ? tile - tx : tile + 1].left + k;
                if (kSuper) inside = tx + 1 != tiles_x;
            } else {                                         // bottom row -- top row of the tile below
                k = b - kTile; mask = rec.bottom_row;
                pu = edges[tile].bottom + k;
                pv = edges[(ty + 1 == tiles_y) ? tx : tile + tiles_x].top + k;
                if (kSuper) inside = ty + 1 != tiles_y;
            }
            on[i] = inside && ((mask >> k) & 1ull);
            if (on[i]) { lu[i] = ld_in<kCoherent>(pu); lv[i] = ld_in<kCoherent>(pv); }
        }
    }
#pragma unroll
    for (int i = 0; i < kTiles; ++i) {
        // the previous border bond joins the same two tile-local components: nothing new to learn
        const uint32_t plu = __shfl_up_sync(0xFFFFFFFFu, lu[i], 1), plv = __shfl_up_sync(0xFFFFFFFFu, lv[i], 1);
        const bool pon = __shfl_up_sync(0xFFFFFFFFu, (uint32_t)on[i], 1) != 0;
        const bool dup = lane != 0 && pon && plu == lu[i] && plv == lv[i];
        const bool keep = on[i] && !dup;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, keep);
        uint32_t base = 0;
        if (lane == 0 && m) base = atomicAdd(&S.n, (uint32_t)__popc(m));
        base = __shfl_sync(0xFFFFFFFFu, base, 0);
        if (keep) S.link[base + __popc(m & ((1u << lane) - 1u))] = make_uint2(lu[i], lv[i]);
    }
    Bar::sync();
    const uint32_t n = S.n;
    uint32_t st[3] = {0, 0, 0};                              // kStats: hops, longest find, lost races
    for (uint32_t k = b; k < n; k += kMergeThreads) {
        const uint2 e = S.link[k];
        if (kSuper) unite<kStats, DomAddr>(labels, e.x, e.y, st, DomAddr(dom));
        else unite<kStats>(labels, e.x, e.y, st);
    }
    if (kStats) {
        const uint32_t hops = __reduce_add_sync(0xFFFFFFFFu, st[0]), deep = __reduce_max_sync(0xFFFFFFFFu, st[1]);
        const uint32_t lost = __reduce_add_sync(0xFFFFFFFFu, st[2]);
        if (lane == 0) {
            atomicAdd(&counters->merge_hops, (unsigned long long)hops);
            atomicAdd(&counters->merge_retries, (unsigned long long)lost);
            atomicMax(&counters->max_merge_depth, deep);
        }
        if (b == 0) atomicAdd(&counters->merge_links, (unsigned long long)n);
    }
}

struct MergeBar {
    static __device__ __forceinline__ void sync() { __syncthreads(); }
};

template <bool kStats, int kTiles>
__global__ void __launch_bounds__(kMergeThreads)
k_tile_merge(uint32_t *labels, const TileBorder *__restrict__ border, const TileEdges *__restrict__ edges,
             Params P, uint32_t n_tiles, PassCounters *__restrict__ counters)
{
    __shared__ MergeShared S;
    tile_merge_body<kStats, false, false, MergeBar, kTiles>(S, labels, border, edges, P, Dom{}, blockIdx.x * kTiles, n_tiles, counters);
}

template <int kTiles>
__global__ void __launch_bounds__(kMergeThreads)
k_tile_merge_super(uint32_t *labels, const TileBorder *__restrict__ border, const TileEdges *__restrict__ edges,
                   Params P, Dom dom, uint32_t n_tiles)
{
    __shared__ MergeShared S;
    tile_merge_body<false, true, false, MergeBar, kTiles>(S, labels, border, edges, P, dom, blockIdx.x * kTiles, n_tiles, nullptr);
}

// ---- kernel 3: flatten to the canonical root + flip --------------------------------------------
// After the merge, the tile-local roots form a forest in labels[] (see the top of this file).  `rootbits` says
// which sites are tile-local roots: each of them is chased ONCE to its canonical root through global memory
// and gets ONE Philox FLIP draw (work spread over the whole CTA); every other site holds the tile-local id
// of its root and needs one shared-memory lookup of (canonical root, new state).
//
// Memory layout of the accesses: a tile row of labels is 256 bytes = 16 lanes x 16 bytes, so one
// warp-wide 16-byte access covers two full tile rows (4 wavefronts of 128 contiguous bytes, the
// minimum).  A CTA of kFlipThreads threads owns a tile; warp w owns kFlipRows = 2 kFlipAcc tile rows;
// its k-th access covers rows kFlipRows w + 2k and + 2k + 1; lane l holds the 4 sites
// x = 4 (l % 16) .. + 3 of row kFlipRows w + 2k + l / 16.

constexpr int kFlipThreads = 256;                                // (tile_draw_masks is written for 256 threads per tile)

template <int NT>
struct FlipShared {
    static constexpr int kAcc = (int)kTileSites / (4 * NT);       // 16-byte accesses per thread
    static constexpr int kRows = 2 * kAcc;                       // tile rows per warp
    uint32_t root[kTileSites];                                   // per tile-local root: its canonical root
    uint8_t state[kTileSites];                                   // per tile-local root: the new state
    uint16_t list[NT / 32][kRows * kTile];                       // per warp: the tile-local roots of its rows
};

// The body of the flip kernel for tile (tx, ty), run by NT threads.
// kLabels: write the canonical labels back (eager mode, or the on-demand flatten of lazy mode);
// kSpins: draw and write the new spins; kCount: leave the number of canonical roots per warp in tile_clusters[]
// (n_clusters of sw_measure without a pass over labels[]; costs 3 % of the kernel, so only the last sweep of a call does it).
// kSuper: one sub-lattice of the super-lattice: label values global, addresses local; a chase ends at a root OR at the
// first link that leaves the piece (after the resolve pass of sw_super.cu such a link points at the canonical root).
// pk_t / pk_n: philox_sweep constants of this sweep and the next (Params::pk_t / pk_n, or made on the device).
// kSizes (sw_sweep_measure with the largest cluster): the tile kernel listed the tile-local components that own a site on
// the border of the tile in btab[tile][] (root's tile-local id | size << 12, k_tile_blocks_sizes; the others are whole
// clusters and were dealt with there); each adds its size to sizes[canonical root] -- one global atomic per such
// component, nothing per site -- so that afterwards sizes[] (all zero before) holds the sizes of the clusters that
// cross a tile border at their canonical roots.
//
// kTma (experiment, SW_FLIP_TMA; k_tile_flip only): the label rows of the tile move by TMA bulk copies (cp.async.bulk,
// SASS UBLKCP) instead of 16-byte cp.async per thread.  A tile row is 256 contiguous bytes in global AND in S.root, so
// each warp fetches its own kRows rows with one bulk copy per row (lanes 0 .. kRows-1 issue one each) that complete on
// the warp's own mbarrier -- no CTA barrier, the warp waits for its own rows only, like cp.async.wait_all did.
// kTma == 2: the canonical labels leave the same way: phase C writes them over the warp's own rows of S.root (a root's
// entry already IS its label; the other entries are read by their owner only, before it overwrites them) and one
// bulk store per row sends them out.  Measured numbers: DESIGN.md sec. 6.
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
                 :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst_smem, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst_smem), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_store(void *dst, uint32_t src_smem, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" :: "l"(dst), "r"(src_smem), "r"(bytes) : "memory");
}

template <bool kLabels, bool kSpins, bool kCount, bool kStats, bool kSuper, int NT, class Bar, bool kSizes = false, int kTma = 0>
__device__ __forceinline__ void
tile_flip_body(FlipShared<NT> &S, const uint32_t tx, const uint32_t ty, uint32_t *labels, const uint16_t *rootbits, uint8_t *spins,
               const Params &P, const uint32_t (&pk_t)[3], const uint32_t (&pk_n)[3], const Dom &dom,
               uint32_t *tile_clusters, uint2 *next_draws, PassCounters *counters, uint32_t *sizes = nullptr,
               const uint32_t *btab = nullptr, unsigned long long *mbar = nullptr)
{
    static_assert(kTma == 0 || !kSuper, "the bulk-copy variant is written for the single lattice");
    constexpr int kAcc = FlipShared<NT>::kAcc, kRows = FlipShared<NT>::kRows;
    const uint32_t tid = threadIdx.x;
    const uint32_t lane = tid & 31u, warp = tid >> 5;
    const uint32_t L = kSuper ? dom.Lg : P.L;                  // row stride of label values (global site indices)
    const uint32_t W = kSuper ? dom.W : P.L;                   // row stride of the arrays
    const uint32_t tiles_x = W >> 6;
    const uint32_t tile = ty * tiles_x + tx;
    const uint32_t origin = kSuper ? (dom.oy + (ty << 6)) * L + dom.ox + (tx << 6) : (ty << 6) * L + (tx << 6);
    const uint32_t x4 = (lane & 15u) << 2;                     // my first column inside the tile
    const uint32_t yk0 = warp * kRows + (lane >> 4);           // my tile row for k = 0 (k-th: + 2k)
    const uint32_t i00 = origin + yk0 * L + x4;                // global index of my first site for k = 0
    const uint32_t a00 = kSuper ? ((ty << 6) + yk0) * W + (tx << 6) + x4 : i00;   // its array offset

    // -- phase A: everything this tile needs from HBM is requested at once: my labels and root flags.
    //    A tile-local root's own entry is its link into the global forest (itself if the merge never hooked
    //    it), so the first step of every chase comes out of this coalesced load instead of a scattered one.
    //    What a site needs afterwards is the tile-local id of its root (12 bits; its own id if it is a root): it stays
    //    in shared memory until phase C.
    uint32_t work = 0;                                         // bit 4k + j: my site j of access k is a tile-local root
    uint32_t rq[kAcc];
    uint32_t tab = 0;                                          // kSizes: my entry of the tile's border table
    if (kSizes) {
        static_assert(!kSizes || NT == 256, "one border-table entry per thread");
        tab = __ldcg(btab + tile * 256u + tid);
    }
    // The labels go straight to shared memory (cp.async, L2 only: 16 bytes per thread and access, no registers held
    // while they are in flight): a root's entry is where its chase starts (and is replaced by the canonical root
    // below), every other site's entry keeps the tile-local id of its root until phase C reads it back -- nothing
    // per site has to stay in registers across the draws and the chases.
    uint32_t bar = 0;
    if (kTma) {
        bar = (uint32_t)__cvta_generic_to_shared(mbar + warp);
        if (lane == 0) { mbar_init(bar, 1); mbar_expect_tx(bar, kRows * kTile * 4); }
        __syncwarp();
        if (lane < (uint32_t)kRows) {                          // one 256-byte row each
            const uint32_t row = warp * kRows + lane;
            bulk_load((uint32_t)__cvta_generic_to_shared(&S.root[row << 6]), labels + origin + row * W, kTile * 4, bar);
        }
    }
#pragma unroll
    for (int k = 0; k < kAcc; ++k) {
        const uint32_t o = a00 + 2 * k * W, id0 = ((yk0 + 2 * k) << 6) + x4;
        if (!kTma) {
            const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&S.root[id0]);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(dst), "l"(labels + o) : "memory");
        }
        rq[k] = rootbits[o >> 4];
    }
    // while those loads are on their way: the bond draws of the NEXT sweep for this tile (pure arithmetic, see above)
    if (kSpins && next_draws) {
#pragma unroll
        for (int u = 0; u < 256; u += NT) tile_draw_masks(next_draws, tile, origin, tid + u, pk_n, P, L);
    }
#pragma unroll
    for (int k = 0; k < kAcc; ++k) work |= ((rq[k] >> (x4 & 12u)) & 15u) << (4 * k);
    if (kTma) mbar_wait(bar, 0); else asm volatile("cp.async.wait_all;" ::: "memory");

    {
        // each warp lists the tile-local roots of its rows (prefix sum over the lanes, no atomics) ...
        const uint32_t n = __popc(work);
        uint32_t incl = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t up = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= (uint32_t)o) incl += up;
        }
        const uint32_t n_warp = __shfl_sync(0xFFFFFFFFu, incl, 31);
        uint32_t pos = incl - n, w = work;
        const uint32_t idb = (yk0 << 6) + x4;
        while (w) {
            const uint32_t j = __ffs(w) - 1u;
            w &= w - 1u;
            S.list[warp][pos++] = (uint16_t)(idb + ((j >> 2) << 7) + (j & 3u));
        }
        __syncwarp();
        // ... and gives each ONE chase and ONE new state (step (3)), 32 roots at a time
        uint32_t hops_all = 0, hops_max = 0;                   // kStats
        for (uint32_t k = lane; k < n_warp; k += 32) {
            const uint32_t id = S.list[warp][k];
            const uint32_t self = origin + (id >> 6) * L + (id & 63u);
            uint32_t hops = 1;                                 // the first hop came with the coalesced load of phase A
            uint32_t g;
            if (kSuper) {
                const DomAddr addr(dom);
                uint32_t a = self;
                g = S.root[id];
                while (g != a && addr.mine(g)) { a = g; g = ld_label(labels, a, addr); }
            } else {
                g = find_root_halving_from<kStats>(labels, self, S.root[id], &hops);
            }
            if (kStats) { hops_all += hops; hops_max = max(hops_max, hops); }
            S.root[id] = g;
            if (kSpins) S.state[id] = (uint8_t)flip_state(g, pk_t, P);
        }
        if (kStats) {
            hops_all = __reduce_add_sync(0xFFFFFFFFu, hops_all);
            hops_max = __reduce_max_sync(0xFFFFFFFFu, hops_max);
            if (lane == 0) { atomicAdd(&counters->chase_hops, (unsigned long long)hops_all); atomicMax(&counters->max_chase_depth, hops_max); }
        }
    }
    Bar::sync();
    if (kSizes && (tab >> 12)) atomicAdd(sizes + S.root[tab & 0xFFFu], tab >> 12);   // (the root's entry holds its canonical root now)

    // -- phase C: every site looks up (canonical root, new state) of its tile-local root
    uint32_t canon = 0;                                        // clusters whose smallest site is one of mine (for sw_measure)
#pragma unroll
    for (int k = 0; k < kAcc; ++k) {
        const uint32_t i0 = i00 + 2 * k * L, o = a00 + 2 * k * W;
        uint32_t st = 0, lab[4], qid[4];
        {
            const uint32_t id0 = ((yk0 + 2 * k) << 6) + x4, rb = (work >> (4 * k)) & 15u;
            const uint4 l = *reinterpret_cast<const uint4 *>(&S.root[id0]);           // my own entries, as phase A left them
            const uint32_t mine[4] = {l.x, l.y, l.z, l.w};
#pragma unroll
            for (int j = 0; j < 4; ++j) qid[j] = ((rb >> j) & 1u) ? id0 + j : mine[j];
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t id = qid[j];
            lab[j] = S.root[id];
            if (kCount) canon += (lab[j] == i0 + j);           // a canonical root is its own label
            if (kSpins) st |= (uint32_t)S.state[id] << (8 * j);
        }
        if (kSpins) *reinterpret_cast<uint32_t *>(spins + o) = st;
        if (kLabels && kTma == 2)
            *reinterpret_cast<uint4 *>(&S.root[((yk0 + 2 * k) << 6) + x4]) = make_uint4(lab[0], lab[1], lab[2], lab[3]);
        else if (kLabels)
            *reinterpret_cast<uint4 *>(labels + o) = make_uint4(lab[0], lab[1], lab[2], lab[3]);
    }
    if (kLabels && kTma == 2) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // my writes to S.root, before the async proxy reads them
        __syncwarp();
        if (lane < (uint32_t)kRows) {
            const uint32_t row = warp * kRows + lane;
            bulk_store(labels + origin + row * W, (uint32_t)__cvta_generic_to_shared(&S.root[row << 6]), kTile * 4);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory must outlive the read
        }
    }
    if (kCount) {
        canon = __reduce_add_sync(0xFFFFFFFFu, canon);
        if (lane == 0) tile_clusters[tile * (NT / 32) + warp] = canon;
    }
}

#ifndef SW_FLIP_CTAS
#define SW_FLIP_CTAS 7
#endif
#ifndef SW_FLIP_TMA
#define SW_FLIP_TMA 0        // 0: 16-byte cp.async per thread (kept: see DESIGN.md sec. 6), 1: TMA bulk loads, 2: bulk loads and stores
#endif
template <bool kLabels, bool kSpins, bool kCount, bool kStats = false>
__global__ void __launch_bounds__(kFlipThreads, SW_FLIP_CTAS)
k_tile_flip(uint32_t *labels, const uint16_t *__restrict__ rootbits, uint8_t *__restrict__ spins, Params P,
            uint32_t *__restrict__ tile_clusters, uint2 *__restrict__ next_draws, PassCounters *__restrict__ counters = nullptr)
{
    __shared__ __align__(128) FlipShared<kFlipThreads> S;
#if SW_FLIP_TMA
    __shared__ unsigned long long mbar[kFlipThreads / 32];     // one mbarrier per warp (its own rows)
    tile_flip_body<kLabels, kSpins, kCount, kStats, false, kFlipThreads, MergeBar, false, SW_FLIP_TMA>(
        S, blockIdx.x, blockIdx.y, labels, rootbits, spins, P, P.pk_t, P.pk_n, Dom{}, tile_clusters, next_draws, counters, nullptr, nullptr, mbar);
#else
    tile_flip_body<kLabels, kSpins, kCount, kStats, false, kFlipThreads, MergeBar>(
        S, blockIdx.x, blockIdx.y, labels, rootbits, spins, P, P.pk_t, P.pk_n, Dom{}, tile_clusters, next_draws, counters);   // grid = (tiles_x, tiles_x): no division
#endif
}

// the flip of a sweep whose cluster sizes are wanted (sw_sweep_measure with SW_OBS_LARGEST): eager labels, spins, cluster
// count, and the sizes (see tile_flip_body, kSizes; the tile kernel of this sweep was k_tile_blocks_sizes)
__global__ void __launch_bounds__(kFlipThreads, SW_FLIP_CTAS)
k_tile_flip_sizes(uint32_t *labels, const uint16_t *__restrict__ rootbits, uint8_t *__restrict__ spins, Params P,
                  uint32_t *__restrict__ tile_clusters, uint2 *__restrict__ next_draws, uint32_t *sizes, const uint32_t *__restrict__ btab)
{
    __shared__ FlipShared<kFlipThreads> S;
    tile_flip_body<true, true, true, false, false, kFlipThreads, MergeBar, true>(
        S, blockIdx.x, blockIdx.y, labels, rootbits, spins, P, P.pk_t, P.pk_n, Dom{}, tile_clusters, next_draws, nullptr, sizes, btab);
}

// one sub-lattice of the super-lattice; grid = (W / 64, H / 64).  `spins` is read by the neighbours' tile kernels of the
// next sweep (their halo), never by this kernel.
template <bool kLabels, bool kSpins, bool kCount>
__global__ void __launch_bounds__(kFlipThreads, SW_FLIP_CTAS)
k_tile_flip_super(uint32_t *labels, const uint16_t *__restrict__ rootbits, uint8_t *spins, Params P, Dom dom,
                  uint32_t *__restrict__ tile_clusters, uint2 *__restrict__ next_draws)
{
    __shared__ FlipShared<kFlipThreads> S;
    tile_flip_body<kLabels, kSpins, kCount, false, true, kFlipThreads, MergeBar>(
        S, blockIdx.x, blockIdx.y, labels, rootbits, spins, P, P.pk_t, P.pk_n, dom, tile_clusters, next_draws, nullptr);
}

}  // namespace sw
