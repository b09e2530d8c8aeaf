// sw_tiled.cuh -- the hot path of libsw.so for L % 64 == 0: three kernels per sweep.
//
//   k_tile_bonds_label  step (1) + tile-local part of step (2)   ("done independently on each site")
//   k_tile_merge        union-find over the bonds that cross a tile border (PAPER.md:66-68 uses the
//                       same boundary-only idea one level up, between GPUs)
//   k_tile_flip         pointer-jumping flatten to the canonical root ("tracks back
//                       the label variable until [it] remains unchanged") fused with step (3)
//
// A tile is 64 x 64 sites; a CTA of 256 threads owns one tile; thread (y = tid/4, c = tid%4) owns
// the 16 consecutive sites x = 16c .. 16c+15 of tile row y: one 16-byte spin load, one Philox call
// per site pair, one 32-bit bond word, four 16-byte label stores.
#pragma once

#include "sw_common.cuh"

namespace sw {

constexpr uint32_t kTile = 64;                       // tile edge
constexpr uint32_t kTileSites = kTile * kTile;       // 4096
constexpr int kTileThreads = 256;
constexpr int kMergeThreads = 128;

// per-tile record of the bonds that leave the tile (written by k_tile_bonds_label, read by k_tile_merge)
struct __align__(16) TileBorder {
    unsigned long long right_col;   // bit y: bond (X0+63, Y0+y) -> (X0+64, Y0+y)
    unsigned long long bottom_row;  // bit x: bond (X0+x, Y0+63) -> (X0+x, Y0+64)
};

// per-tile copy of the tile-local labels of the left and right columns (written by the tile kernel,
// read by k_tile_merge): a column of labels[] is one 32-byte sector per site, these are 256 bytes each
struct __align__(16) TileCols {
    uint32_t left[kTile];           // label of site (X0,      Y0 + y)
    uint32_t right[kTile];          // label of site (X0 + 63, Y0 + y)
};

// ---- shared-memory union-find (tile-local) -----------------------------------------------------
// Nodes are "pieces": maximal runs of right-bonded sites inside one thread's 16-site segment, named
// by their first site.  A node id is the PADDED local index 17 * thread + x (one spare word per 16
// entries, so that the 32 lanes of a warp, which own segments 16 words apart, fall in 32 different
// banks).  Padding keeps the row-major order, so "smaller id" still means "smaller site index".
//
// Links always point to a smaller id, so plain stores that replace a link by a link to an ancestor
// (path halving) are safe next to concurrent atomicMin hooks: nothing that was joined can come
// apart, and the root of a set is always its smallest member ("proper label").

constexpr uint32_t kPad = 17;                               // padded words per 16-site segment
constexpr uint32_t kParentWords = kTileThreads * kPad;      // 4352

__device__ __forceinline__ void unite_s(volatile uint32_t *parent, uint32_t a, uint32_t b)
{
    while (true) {
        // chase both ends together (the loop runs max(depth a, depth b) times, not the sum), halving as we go
        uint32_t pa = parent[a], pb = parent[b];
        while (pa != a || pb != b) {
            const uint32_t ga = parent[pa], gb = parent[pb];
            if (ga != pa) parent[a] = ga;
            if (gb != pb) parent[b] = gb;
            a = ga; b = gb;
            pa = parent[a]; pb = parent[b];
        }
        if (a == b) return;
        if (a < b) { const uint32_t s = a; a = b; b = s; }
        const uint32_t old = atomicMin(const_cast<uint32_t *>(parent) + a, b);
        if (old == a) return;
        a = old;
    }
}

// the four 0x00/0xFF bytes of a __vcmpeq4 result -> 4 bits
__device__ __forceinline__ uint32_t pack4(uint32_t eq) { return ((eq & 0x01010101u) * 0x01020408u) >> 24; }

// position of the piece start (highest set bit of S at or below x)
__device__ __forceinline__ uint32_t run_start(uint32_t S, uint32_t x) { return 31u - __clz(S & ((2u << x) - 1u)); }

// piece-start mask of a segment from its (tile-local) right-bond mask: site x starts a piece unless bonded to x-1
__device__ __forceinline__ uint32_t starts_of(uint32_t r16) { return (~(r16 << 1) | 1u) & 0xFFFFu; }

// An extra link is named by the thread t = 4y + c that owns its LOWER end and a column x of its segment:
// vertical = (piece of site x in row y) -- (piece of site x in row y-1); joint (bit 12) = (first piece of the
// segment) -- (last piece of the segment to its left).  The piece starts are recomputed from the shared
// bond masks, so the list entry stays 16 bits.
__device__ __forceinline__ void unite_link(volatile uint32_t *parent, const uint32_t *rd, uint32_t e)
{
    const uint32_t t = (e >> 4) & 0xFFu, x = e & 15u;
    uint32_t a, b;
    if (e & 0x1000u) {
        a = t * kPad;
        b = (t - 1) * kPad + run_start(starts_of(rd[t - 1] & 0xFFFFu), 15u);
    } else {
        a = t * kPad + run_start(starts_of(rd[t] & 0xFFFFu), x);
        b = (t - 4) * kPad + run_start(starts_of(rd[t - 4] & 0xFFFFu), x);
    }
    unite_s(parent, a, b);
}

// ---- kernel 1: bonds + tile-local labels --------------------------------------------------------
// Labeling in four phases (the idea of label equivalence without the outer iteration: one
// assignment pass, one pass over the leftover equivalences, one resolve pass):
//   A  every piece that has a neighbour piece above it (or to its left, across a segment joint)
//      takes ONE of them as its parent with a plain store: no search, no atomics.  Parents have
//      smaller ids, so this is a forest.
//   B  the remaining links (second and later up-links of a piece, up-links of a piece that took its
//      joint) are real equivalences: united with find + atomicMin, 32 at a time per warp.
//   C  every piece is pointed straight at its root.  A warp walks the pieces of its 8-row strip in
//      row order, so the parent of a piece is almost always resolved already (as in the second
//      pass of a sequential Hoshen-Kopelman labeling).
//   D  each thread reads the roots of its pieces and writes labels, root flags and the border record.
constexpr uint32_t kListCap = 8 * 64 + 32;             // pieces of a strip <= 512; extra links of a strip <= 512 + 24

__global__ void __launch_bounds__(kTileThreads, 8)
k_tile_bonds_label(const uint8_t *__restrict__ spins, uint32_t *__restrict__ bonds,
                   uint32_t *__restrict__ labels, uint16_t *__restrict__ rootbits,
                   TileBorder *__restrict__ border, TileCols *__restrict__ cols, Params P)
{
    __shared__ uint32_t s_parent[kParentWords];
    __shared__ uint32_t s_rd[kTileThreads];                    // per thread: tile-local right bonds | down bonds << 16
    __shared__ uint16_t s_list[kTileThreads / 32][kListCap];   // per warp: extra links (phase B), then pieces (phase C)
    __shared__ uint32_t s_right[2];

    const uint32_t tid = threadIdx.x, y = tid >> 2, c = tid & 3;
    const uint32_t lane = tid & 31u, warp = tid >> 5;
    const uint32_t L = P.L, tiles_x = L >> 6;
    const uint32_t ty = blockIdx.x / tiles_x, tx = blockIdx.x - ty * tiles_x;
    const uint32_t X0 = tx << 6, Y0 = ty << 6;
    const uint32_t gy = Y0 + y, gx = X0 + (c << 4);
    const uint64_t row_off = (uint64_t)gy * L;
    const uint32_t i0 = (uint32_t)(row_off + gx);           // global index of my first site

    if (tid < 2) s_right[tid] = 0;

    // -- spins: my 16 sites, the 16 below them, and the right neighbour of my last site
    const uint4 sv = *reinterpret_cast<const uint4 *>(spins + row_off + gx);
    const uint32_t gyd = (gy + 1 == L) ? 0u : gy + 1;
    const uint4 dv = *reinterpret_cast<const uint4 *>(spins + (uint64_t)gyd * L + gx);
    uint32_t nxt = __shfl_down_sync(0xFFFFFFFFu, sv.x, 1);
    if (c == 3) nxt = spins[row_off + ((X0 + kTile == L) ? 0u : X0 + kTile)];

    const uint32_t w[4] = {sv.x, sv.y, sv.z, sv.w};
    const uint32_t dw[4] = {dv.x, dv.y, dv.z, dv.w};
    uint32_t eq_r = 0, eq_d = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint32_t r = __funnelshift_r(w[k], (k < 3) ? w[k + 1] : nxt, 8);
        eq_r |= pack4(__vcmpeq4(w[k], r)) << (4 * k);
        eq_d |= pack4(__vcmpeq4(w[k], dw[k])) << (4 * k);
    }

    // -- draws: one Philox call per site pair (sites i0+2p, i0+2p+1): words = right, down, right, down
    uint32_t m_r = 0, m_d = 0;
    const uint32_t pair0 = i0 >> 1;
#pragma unroll
    for (int p = 0; p < 8; ++p) {
        const uint4 d = philox4x32_10(pair0 + p, 0u, P.t, kPurposeBond, P);
        m_r |= (uint32_t)(d.x <= P.thr_m1) << (2 * p);
        m_d |= (uint32_t)(d.y <= P.thr_m1) << (2 * p);
        m_r |= (uint32_t)(d.z <= P.thr_m1) << (2 * p + 1);
        m_d |= (uint32_t)(d.w <= P.thr_m1) << (2 * p + 1);
    }
    const uint32_t r16 = eq_r & m_r & P.thr_any;
    const uint32_t d16 = eq_d & m_d & P.thr_any;
    bonds[i0 >> 4] = r16 | (d16 << 16);

    // -- tile-local masks: bonds that leave the tile are recorded in the border record instead
    const uint32_t lr16 = (c == 3) ? (r16 & 0x7FFFu) : r16;
    s_rd[tid] = lr16 | (d16 << 16);                           // (row 63's down bonds are only read for the border record)
    const uint32_t pbase = tid * kPad;                       // padded id of my first site
    const uint32_t S = starts_of(lr16);                      // bit x: site x starts a piece
#pragma unroll
    for (int x = 0; x < 16; ++x)
        if ((S >> x) & 1u) s_parent[pbase + x] = pbase + x;
    __syncthreads();
    if (c == 3 && (r16 >> 15)) atomicOr(&s_right[y >> 5], 1u << (y & 31));

    // -- phase A: one parent per piece, by plain store
    const uint32_t C = S ^ 0xFFFFu;                          // bit x: site x continues the piece of x-1
    uint32_t extra;                                          // up-links that phase B must still unite
    bool joint;                                              // my first piece is bonded to the segment on my left
    {
        const uint32_t up = (y > 0) ? s_rd[tid - 4] : 0u;
        const uint32_t s = up >> 16;                          // bit x: up-link (row y-1, x) -- (row y, x)
        const uint32_t S_up = starts_of(up & 0xFFFFu);
        const uint32_t left = __shfl_up_sync(0xFFFFFFFFu, lr16, 1);
        joint = c > 0 && ((left >> 15) & 1u);
        // first up-link of every piece: carry chain with generate = s, propagate = C gives, for every
        // site, "some up-link at a smaller x of my piece"
        const uint32_t A = s | C;
        const uint32_t cin = (A + s) ^ A ^ s;                 // bit x: carry into x
        uint32_t first = s & ~(cin & C);
        // an up-link whose left neighbour is an up-link between the same two pieces says nothing new
        const uint32_t v = s & ~((s << 1) & C & ~S_up);
        if (joint) {
            const uint32_t second = S & (S - 1u);             // piece starts after the first one
            const uint32_t e0 = (second & (0u - second)) - 1u;   // extent of my first piece (all ones if it is the only one)
            first &= ~e0;                                     // that piece takes the joint; its up-links become extras
            s_parent[pbase] = pbase - kPad + run_start(starts_of(left & 0xFFFFu), 15u);
        }
        extra = v & ~first;
        while (first) {
            const uint32_t x = __ffs(first) - 1;
            first &= first - 1;
            s_parent[pbase + run_start(S, x)] = pbase - 4 * kPad + run_start(S_up, x);
        }
    }
    __syncthreads();

    // -- phase B: the remaining links, gathered per warp (prefix sum over the lanes) and united 32 at a time
    {
        const uint32_t n = (uint32_t)__popc(extra);
        uint32_t incl = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t upv = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= (uint32_t)o) incl += upv;
        }
        const uint32_t n_warp = __shfl_sync(0xFFFFFFFFu, incl, 31);
        uint32_t pos = incl - n;
        uint16_t *mine = s_list[warp];
        while (extra) {
            mine[pos++] = (uint16_t)((tid << 4) | (__ffs(extra) - 1));
            extra &= extra - 1;
        }
        __syncwarp();
        for (uint32_t k = lane; k < n_warp; k += 32) unite_link(s_parent, s_rd, mine[k]);
    }
    __syncthreads();

    if (tid == 0) {
        TileBorder b;
        b.right_col = (unsigned long long)s_right[0] | ((unsigned long long)s_right[1] << 32);
        b.bottom_row = (unsigned long long)(s_rd[252] >> 16) | ((unsigned long long)(s_rd[253] >> 16) << 16) |
                       ((unsigned long long)(s_rd[254] >> 16) << 32) | ((unsigned long long)(s_rd[255] >> 16) << 48);
        border[blockIdx.x] = b;
    }

    // -- phase C: point every piece of my warp's strip at its root, in row order (no hooks happen any more)
    {
        const uint32_t n = (uint32_t)__popc(S);
        uint32_t incl = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t upv = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= (uint32_t)o) incl += upv;
        }
        const uint32_t n_warp = __shfl_sync(0xFFFFFFFFu, incl, 31);
        uint32_t pos = incl - n, m = S;
        uint16_t *mine = s_list[warp];
        while (m) {
            mine[pos++] = (uint16_t)(pbase + __ffs(m) - 1);
            m &= m - 1;
        }
        __syncwarp();
        volatile uint32_t *par = s_parent;
        for (uint32_t k0 = 0; k0 < n_warp; k0 += 32) {
            const uint32_t k = k0 + lane;
            if (k < n_warp) {
                const uint32_t id = mine[k];
                const uint32_t p = par[id];
                if (p != id) {
                    uint32_t r = p, g = par[r];
                    while (g != r) { r = g; g = par[r]; }
                    if (r != p) par[id] = r;
                }
            }
            __syncwarp();
        }
    }

    // -- phase D: labels = global index of the smallest site of my tile-local component; root flags
    const uint32_t origin = Y0 * L + X0;
    uint32_t lab[16];
    uint32_t cur = 0, roots = 0;
#pragma unroll
    for (int x = 0; x < 16; ++x) {
        if ((S >> x) & 1u) {
            const uint32_t r = s_parent[pbase + x];
            const uint32_t t = (r * 61681u) >> 20;           // r / 17 for r < 4352: the thread that owns the root
            cur = origin + (t >> 2) * L + ((t & 3u) << 4) + (r - t * kPad);
            roots |= (r == pbase + x) ? (1u << x) : 0u;
        }
        lab[x] = cur;
    }
    uint4 *lp = reinterpret_cast<uint4 *>(labels + row_off + gx);
    lp[0] = make_uint4(lab[0], lab[1], lab[2], lab[3]);
    lp[1] = make_uint4(lab[4], lab[5], lab[6], lab[7]);
    lp[2] = make_uint4(lab[8], lab[9], lab[10], lab[11]);
    lp[3] = make_uint4(lab[12], lab[13], lab[14], lab[15]);
    rootbits[i0 >> 4] = (uint16_t)roots;
    if (c == 0) cols[blockIdx.x].left[y] = lab[0];
    if (c == 3) cols[blockIdx.x].right[y] = lab[15];
}

// ---- kernel 2: merge across tile borders -------------------------------------------------------
// One thread per border site (64 on the right column, 64 on the bottom row of a tile).  Only about a
// third of them carry a link worth uniting (active bond, not a repeat of its neighbour's link), and a
// unite is a chain of dependent L2 / HBM round trips, so the kernel is latency-bound: a CTA therefore
// gathers the links of kMergeTiles tiles into a dense list first (coalesced loads, all independent)
// and then unites them with every lane busy.

constexpr int kMergeTiles = 4;

__global__ void __launch_bounds__(kMergeThreads)
k_tile_merge(uint32_t *labels, const TileBorder *__restrict__ border, const TileCols *__restrict__ cols,
             Params P, uint32_t n_tiles)
{
    __shared__ uint2 s_link[kMergeTiles * kMergeThreads];
    __shared__ uint32_t s_n;

    const uint32_t b = threadIdx.x, lane = b & 31u;
    const uint32_t L = P.L, tiles_x = L >> 6;
    if (b == 0) s_n = 0;
    __syncthreads();

    uint32_t lu[kMergeTiles], lv[kMergeTiles];
    bool on[kMergeTiles];
#pragma unroll
    for (int i = 0; i < kMergeTiles; ++i) {
        const uint32_t tile = blockIdx.x * kMergeTiles + i;
        on[i] = false; lu[i] = 0; lv[i] = 0;
        if (tile < n_tiles) {
            const uint32_t ty = tile / tiles_x, tx = tile - ty * tiles_x;
            const uint32_t X0 = tx << 6, Y0 = ty << 6;
            const TileBorder rec = border[tile];
            const uint32_t *pu, *pv;
            unsigned long long mask;
            uint32_t k;
            if (b < kTile) {                                 // right column -- left column of the tile on the right
                k = b; mask = rec.right_col;
                pu = cols[tile].right + k;
                pv = cols[(tx + 1 == tiles_x) ? tile - tx : tile + 1].left + k;
            } else {                                         // bottom row -- top row of the tile below
                k = b - kTile; mask = rec.bottom_row;
                pu = labels + (uint64_t)(Y0 + kTile - 1) * L + X0 + k;
                pv = labels + (uint64_t)((Y0 + kTile == L) ? 0u : Y0 + kTile) * L + X0 + k;
            }
            on[i] = (mask >> k) & 1ull;
            if (on[i]) { lu[i] = __ldcg(pu); lv[i] = __ldcg(pv); }
        }
    }
#pragma unroll
    for (int i = 0; i < kMergeTiles; ++i) {
        // the previous border bond joins the same two tile-local components: nothing new to learn
        const uint32_t plu = __shfl_up_sync(0xFFFFFFFFu, lu[i], 1), plv = __shfl_up_sync(0xFFFFFFFFu, lv[i], 1);
        const bool pon = __shfl_up_sync(0xFFFFFFFFu, (uint32_t)on[i], 1) != 0;
        const bool dup = lane != 0 && pon && plu == lu[i] && plv == lv[i];
        const bool keep = on[i] && !dup;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, keep);
        uint32_t base = 0;
        if (lane == 0 && m) base = atomicAdd(&s_n, (uint32_t)__popc(m));
        base = __shfl_sync(0xFFFFFFFFu, base, 0);
        if (keep) s_link[base + __popc(m & ((1u << lane) - 1u))] = make_uint2(lu[i], lv[i]);
    }
    __syncthreads();
    const uint32_t n = s_n;
    for (uint32_t k = b; k < n; k += kMergeThreads) {
        const uint2 e = s_link[k];
        unite(labels, e.x, e.y);
    }
}

// ---- kernel 3: flatten to the canonical root + flip --------------------------------------------
// After the merge, labels[] is a forest: a site that is not the root of its tile-local component
// points at that root (inside the tile); a tile-local root points at itself or, if the merge hooked
// it, at a smaller root anywhere.  `rootbits` says which sites are tile-local roots, so each
// distinct root seen by the tile is chased and drawn ONCE (work spread over the whole CTA) and
// every other site needs one shared-memory lookup.
//
// Memory layout of the accesses: a tile row of labels is 256 bytes = 16 lanes x 16 bytes, so one
// warp-wide 16-byte access covers two full tile rows (4 wavefronts of 128 contiguous bytes, the
// minimum).  A CTA of kFlipThreads threads owns a tile; warp w owns kFlipRows = 2 kFlipAcc tile rows;
// its k-th access covers rows kFlipRows w + 2k and + 2k + 1; lane l holds the 4 sites
// x = 4 (l % 16) .. + 3 of row kFlipRows w + 2k + l / 16.

#ifndef SW_FLIP_THREADS
#define SW_FLIP_THREADS 256
#endif
#ifndef SW_FLIP_MINB
#define SW_FLIP_MINB 5
#endif
constexpr int kFlipThreads = SW_FLIP_THREADS;
constexpr int kFlipAcc = (int)kTileSites / (4 * kFlipThreads);   // 16-byte accesses per thread
constexpr int kFlipRows = 2 * kFlipAcc;                          // tile rows per warp

template <bool kPow2>
__global__ void __launch_bounds__(kFlipThreads, SW_FLIP_MINB)
k_tile_flip(uint32_t *labels, const uint16_t *__restrict__ rootbits, uint8_t *__restrict__ spins,
            Params P, int write_labels)
{
    __shared__ uint32_t s_root[kTileSites];                   // per tile-local root: its canonical root
    __shared__ uint8_t s_state[kTileSites];                   // per tile-local root: the new state
    __shared__ uint16_t s_list[kFlipThreads / 32][kFlipRows * kTile];   // per warp: the tile-local roots of its rows

    const uint32_t tid = threadIdx.x;
    const uint32_t lane = tid & 31u, warp = tid >> 5;
    const uint32_t L = P.L, tiles_x = L >> 6;
    const uint32_t ty = blockIdx.x / tiles_x, tx = blockIdx.x - ty * tiles_x;
    const uint32_t X0 = tx << 6, Y0 = ty << 6;
    const uint32_t origin = Y0 * L + X0;
    const uint32_t x4 = (lane & 15u) << 2;                     // my first column inside the tile
    const uint32_t yk0 = warp * kFlipRows + (lane >> 4);       // my tile row for k = 0 (k-th: + 2k)
    const uint32_t i00 = origin + yk0 * L + x4;                // global index of my first site for k = 0

    // -- phase A: everything this tile needs from HBM is requested at once: my labels and root flags.
    //    A tile-local root's own entry is its link into the global forest (itself if the merge never hooked
    //    it), so the first step of every chase comes out of this coalesced load instead of a scattered one.
    uint32_t lab[4 * kFlipAcc];
    uint32_t work = 0;                                         // bit 4k + j: my site j of access k is a tile-local root
#pragma unroll
    for (int k = 0; k < kFlipAcc; ++k) {
        const uint32_t i0 = i00 + 2 * k * L;
        const uint4 l = __ldcg(reinterpret_cast<const uint4 *>(labels + i0));
        lab[4 * k] = l.x; lab[4 * k + 1] = l.y; lab[4 * k + 2] = l.z; lab[4 * k + 3] = l.w;
        const uint32_t rb = rootbits[i0 >> 4];
        work |= ((rb >> (x4 & 12u)) & 15u) << (4 * k);
    }
    // each warp lists the tile-local roots of its strip (prefix sum over the lanes, no atomics)
    uint32_t n_warp;
    {
        const uint32_t n = __popc(work);
        uint32_t incl = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t up = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= (uint32_t)o) incl += up;
        }
        n_warp = __shfl_sync(0xFFFFFFFFu, incl, 31);
        uint32_t pos = incl - n;
#pragma unroll
        for (int j = 0; j < 4 * kFlipAcc; ++j) {
            if ((work >> j) & 1u) {
                const uint32_t id = ((yk0 + 2 * (j >> 2)) << 6) + x4 + (j & 3);
                s_list[warp][pos++] = (uint16_t)id;
                s_root[id] = lab[j];                          // where the chase of this root starts
            }
        }
    }
    __syncwarp();

    // -- phase B: one chase + one Philox call per tile-local root, 32 at a time per warp
    for (uint32_t k = lane; k < n_warp; k += 32) {
        const uint32_t id = s_list[warp][k];
        const uint32_t self = origin + (id >> 6) * L + (id & 63u);
        const uint32_t g = find_root_halving_from(labels, self, s_root[id]);
        s_root[id] = g;
        s_state[id] = (uint8_t)flip_state(g, P);
    }
    __syncthreads();

    // -- phase C: every site looks its tile-local root up; consecutive sites with the same label share a lookup
#pragma unroll
    for (int k = 0; k < kFlipAcc; ++k) {
        const uint32_t i0 = i00 + 2 * k * L;
        const uint32_t id0 = ((yk0 + 2 * k) << 6) + x4;
        uint32_t st = 0, prev = 0, root = 0, state = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const bool isroot = (work >> (4 * k + j)) & 1u;     // a tile-local root stands for itself
            const uint32_t le = isroot ? i0 + j : lab[4 * k + j];
            if (j == 0 || le != prev) {
                const uint32_t d = le - origin;
                const uint32_t dy = kPow2 ? (d >> P.log2L) : (uint32_t)(((uint64_t)d * P.divL_magic) >> 40);
                const uint32_t id = isroot ? id0 + j : (dy << 6) + (d - dy * L);
                root = s_root[id];
                state = s_state[id];
                prev = le;
            }
            lab[4 * k + j] = root;
            st |= state << (8 * j);
        }
        *reinterpret_cast<uint32_t *>(spins + i0) = st;
        if (write_labels)
            *reinterpret_cast<uint4 *>(labels + i0) = make_uint4(lab[4 * k], lab[4 * k + 1], lab[4 * k + 2], lab[4 * k + 3]);
    }
}

}  // namespace sw
