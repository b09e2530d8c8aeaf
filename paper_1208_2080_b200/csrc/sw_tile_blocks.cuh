// sw_tile_blocks.cuh -- bond activation + tile-local labeling, one thread per 8 x 4 block of sites.
//
//   k_tile_blocks   step (1) + the tile-local part of step (2) of the sweep ("the
//                   calculation [is] done independently on each site"; :42 "proper label" = the
//                   smallest site of the cluster).  In: spins, and the "draw < T" bits of this sweep's
//                   bonds (made one sweep ahead, sw_tiled.cuh).  Out, for k_tile_merge / k_tile_flip:
//                   bonds, labels (tile-local roots: their own global index; other sites: the 12-bit
//                   tile-local id of their root), root bitmap, border record, edge record.
//
// A tile is 64 x 64 sites, a CTA of 128 threads owns it; thread (bx = tid % 8, by = tid / 8) owns the
// block of 8 columns x 4 rows at (8 bx, 4 by): its 32 sites are the 32 bits of one register (bit
// j = 8 r + c is row r, column c of the block).  Everything inside a block is bit-parallel register
// arithmetic -- no shared memory, no atomics:
//   * horizontal closure of a site set along active right bonds is one carry chain (an add) towards
//     higher columns and three shift-and-mask steps towards lower columns;
//   * a component of the block is flood-filled from its smallest unvisited site: vertical step,
//     horizontal closure, until nothing new appears;
//   * "which component is site j in" is kept bit-sliced in five plane registers.
// Only the components of the blocks (about 0.2 per site at q = 2, K_c instead of 0.53 horizontal
// runs per site) go through the shared-memory union-find, over the bonds that cross a block edge
// (0.16 per site): first up-link of every component by plain store, the rest with an atomic minimum.
#pragma once

#include "sw_common.cuh"
#include "sw_tiled.cuh"

namespace sw {

constexpr int kBlkThreads = 128;
constexpr int kBlkSlots = 26;                 // components of an 8 x 4 block that can have a link: <= 20 border singles + 6 pairs
constexpr int kBlkExtraCap = 32 * 11;         // per warp: <= 7 up-links + 4 left-links per thread go through atomics
constexpr uint32_t kDecodeMul = (1u << 24) | (1u << 17) | (1u << 10) | (1u << 3);

struct BlkShared {
    uint16_t parent[kTileSites];              // union-find over tile-local site ids (y * 64 + x): component seeds are linked; a site of
                                              // the right column of a block points at its seed (the block on its right links to the site)
    uint32_t list[kBlkSlots][kBlkThreads];    // per thread, slot k: component mask -> seed id | seed bit << 16 -> tile-local id of its root
    uint16_t pub_bottom[8][kBlkThreads];      // seed id of the component of my bottom-row site c
    uint32_t edge[kBlkThreads];               // what the blocks below / to the right need to know about a block: bits 0-7 down
                                              // bonds of row 3, 8-15 right bonds of row 3, 16-19 right bonds of column 7,
                                              // 20-22 down bonds of column 7 (rows 0-2)
    uint32_t n_extra[kBlkThreads / 32];
};
// The links that need the atomic pass are buffered per warp in list slots kBlkBufSlot .. kBlkSlots-1, which are
// free unless some block of the tile has more than kBlkBufSlot components (then they are united unbuffered).
constexpr int kBlkBufSlot = 14;
static_assert((kBlkSlots - kBlkBufSlot) * kBlkThreads >= (kBlkThreads / 32) * kBlkExtraCap, "link buffer too small");

// ---- union-find on 16-bit parents ------------------------------------------------------------------
// Links point to smaller ids, plain stores only ever replace a link
// by a link to an ancestor, hooks are an atomic minimum (here a CAS on the 32-bit word that holds the entry:
// a plain 16-bit store to either half in between makes the CAS fail and retry).
__device__ __forceinline__ uint32_t atomic_min_u16(uint16_t *base, uint32_t idx, uint32_t val)
{
    uint32_t *w = reinterpret_cast<uint32_t *>(base) + (idx >> 1);
    const uint32_t sh = (idx & 1u) << 4;
    uint32_t old = *reinterpret_cast<volatile uint32_t *>(w);
    while (true) {
        const uint32_t cur = (old >> sh) & 0xFFFFu;
        if (cur <= val) return cur;
        const uint32_t got = atomicCAS(w, old, (old & ~(0xFFFFu << sh)) | (val << sh));
        if (got == old) return cur;
        old = got;
    }
}

__device__ __forceinline__ void unite_s16(uint16_t *parent_, uint32_t a, uint32_t b)
{
    volatile uint16_t *parent = parent_;
    {   // two unconditional hops on both sides first (a root points at itself): most chases end here, branch-free
        const uint32_t a1 = parent[a], b1 = parent[b];
        const uint32_t a2 = parent[a1], b2 = parent[b1];
        if (a2 != a1) parent[a] = (uint16_t)a2;
        if (b2 != b1) parent[b] = (uint16_t)b2;
        a = a2; b = b2;
    }
    while (true) {
        uint32_t pa = parent[a], pb = parent[b];
        while (pa != a || pb != b) {
            const uint32_t ga = parent[pa], gb = parent[pb];
            if (ga != pa) parent[a] = (uint16_t)ga;
            if (gb != pb) parent[b] = (uint16_t)gb;
            a = ga; b = gb;
            pa = parent[a]; pb = parent[b];
        }
        if (a == b) return;
        if (a < b) { const uint32_t t = a; a = b; b = t; }
        const uint32_t old = atomic_min_u16(parent_, a, b);
        if (old == a) return;
        a = old;
    }
}

// all sites reachable from n along active right bonds (A: bit j = bond j -- j+1, never set in column 7)
__device__ __forceinline__ uint32_t hclose(uint32_t n, uint32_t A, uint32_t A2, uint32_t A4)
{
    const uint32_t g = n & A;
    n |= (A + g) ^ A ^ g;                     // carry chain: every site above a member through consecutive bonds
    n |= (n >> 1) & A;
    n |= (n >> 2) & A2;
    n |= (n >> 4) & A4;
    return n;
}

// the four plane bytes of block row r as one word (byte b = plane b)
__device__ __forceinline__ uint32_t plane_row(uint32_t P0, uint32_t P1, uint32_t P2, uint32_t P3, uint32_t r)
{
    const uint32_t sel = r | ((4u + r) << 4);
    return __byte_perm(__byte_perm(P0, P1, sel), __byte_perm(P2, P3, sel), 0x5410);
}

// component slot of column c from the row words (W: planes 0-3, V: plane 4 of the row shifted left by 4)
__device__ __forceinline__ uint32_t slot_of(uint32_t W, uint32_t V, uint32_t c)
{
    return ((((W >> c) & 0x01010101u) | ((V >> c) & 0x10u)) * kDecodeMul) >> 24;
}
__device__ __forceinline__ uint32_t slot_of4(uint32_t W, uint32_t c)
{
    return (((W >> c) & 0x01010101u) * kDecodeMul) >> 24;
}

// The body of the tile kernel for tile (tx, ty) of a piece of the lattice, run by kBlkThreads threads.
//   kSuper     the piece is a sub-lattice of the super-lattice (label values global, addresses local: `dom`);
//              false: the whole lattice, dom is not looked at
//   kCoherent  see ld_in
//   Bar        the CTA-wide barrier of those kBlkThreads threads
template <bool kSuper, bool kCoherent, class Bar>
__device__ __forceinline__ void
tile_blocks_body(BlkShared &S, const uint32_t tx, const uint32_t ty, const uint8_t *spins, uint32_t *bonds,
                 uint32_t *labels, uint16_t *rootbits, TileBorder *border, TileEdges *edges, const uint2 *draws,
                 const Params &P, const Dom &dom)
{
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t bx = tid & 7u, by = tid >> 3;
    const uint32_t L = kSuper ? dom.Lg : P.L;                  // row stride of label values (global site indices)
    const uint32_t W = kSuper ? dom.W : P.L;                   // row stride of the arrays
    const uint32_t tiles_x = W >> 6;
    const uint32_t tile = ty * tiles_x + tx;
    const uint32_t X0 = tx << 6, Y0 = ty << 6;
    const uint32_t x0 = X0 + (bx << 3), y0 = Y0 + (by << 2);
    const uint32_t origin = kSuper ? (dom.oy + Y0) * L + dom.ox + X0 : Y0 * L + X0;   // global index of the tile's first site
    const uint32_t idbase = (by << 8) + (bx << 3);             // tile-local id of my first site
    const uint32_t i0 = origin + idbase / 64u * L + (bx << 3); // global index of my first site (mod 2^32 exact: N <= 2^32)
    const uint32_t a0 = kSuper ? y0 * W + x0 : i0;             // its array offset

    // -- union-find array: identity
    {
        uint4 *p4 = reinterpret_cast<uint4 *>(S.parent);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint32_t e = (i * kBlkThreads + tid) * 8u, e2 = e * 0x00010001u + 0x00010000u;   // (e, e + 1) as two halves
            p4[i * kBlkThreads + tid] = make_uint4(e2, e2 + 0x00020002u, e2 + 0x00040004u, e2 + 0x00060006u);
        }
        if (lane == 0) S.n_extra[warp] = 0;
    }

    // -- spins: my 4 rows of 8, the row below (from the lane 8 up, or from memory), the column to the right
    uint2 s[5];
#pragma unroll
    for (int r = 0; r < 4; ++r)
        s[r] = ld_in<kCoherent>(reinterpret_cast<const uint2 *>(spins + (uint64_t)(y0 + r) * W + x0));
    s[4].x = __shfl_down_sync(0xFFFFFFFFu, s[0].x, 8);
    s[4].y = __shfl_down_sync(0xFFFFFFFFu, s[0].y, 8);
    if ((lane >> 3) == 3u) {
        if (kSuper && y0 + 4u == dom.H) {                      // row 0 of the piece below
            s[4] = ld_in<true>(reinterpret_cast<const uint2 *>(dom.down + x0));
        } else {
            const uint32_t yd = (!kSuper && y0 + 4u == L) ? 0u : y0 + 4u;
            s[4] = ld_in<kCoherent>(reinterpret_cast<const uint2 *>(spins + (uint64_t)yd * W + x0));
        }
    }
    uint32_t nx = __byte_perm(__byte_perm(s[0].x, s[1].x, 0x0040), __byte_perm(s[2].x, s[3].x, 0x0040), 0x5410);
    nx = __shfl_down_sync(0xFFFFFFFFu, nx, 1);                // column 0 of the block on my right, one byte per row
    if (bx == 7u) {
        nx = 0;
        if (kSuper && X0 + kTile == W) {                       // column 0 of the piece on the right
#pragma unroll
            for (int r = 0; r < 4; ++r) nx |= (uint32_t)ld_in<true>(dom.right + (uint64_t)(y0 + r) * dom.right_W) << (8 * r);
        } else {
            const uint32_t xr = (!kSuper && X0 + kTile == L) ? 0u : X0 + kTile;
#pragma unroll
            for (int r = 0; r < 4; ++r) nx |= (uint32_t)ld_in<kCoherent>(spins + (uint64_t)(y0 + r) * W + xr) << (8 * r);
        }
    }

    // -- step (1): a bond is active iff the spins are equal and its draw is below the threshold
    uint32_t R = 0, D = 0;
    {
        // The threshold tests of this sweep's draws were made ahead of time (tile_draw_masks in sw_tiled.cuh: by the flip
        // kernel of the previous sweep while it waited for its loads, or by k_draws): bit 8r + c of dm.x / dm.y says
        // whether the right / down draw of my site (r, c) is below the threshold.
        const uint2 dm = ld_in<kCoherent>(draws + tile * kBlkThreads + tid);
        if (P.q == 2u) {                                       // spins are 0 / 1: "equal" is bit 0 of the XNOR (pack4 looks at bit 0 only)
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const uint32_t a0 = s[r].x, a1 = s[r].y;
                const uint32_t n0 = __funnelshift_r(a0, a1, 8), n1 = __funnelshift_r(a1, nx >> (8 * r), 8);
                R |= (pack4(~(a0 ^ n0)) | (pack4(~(a1 ^ n1)) << 4)) << (8 * r);
                D |= (pack4(~(a0 ^ s[r + 1].x)) | (pack4(~(a1 ^ s[r + 1].y)) << 4)) << (8 * r);
            }
        } else {
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const uint32_t a0 = s[r].x, a1 = s[r].y;
                const uint32_t n0 = __funnelshift_r(a0, a1, 8), n1 = __funnelshift_r(a1, nx >> (8 * r), 8);
                const uint32_t eq_r = pack4(__vcmpeq4(a0, n0)) | (pack4(__vcmpeq4(a1, n1)) << 4);
                const uint32_t eq_d = pack4(__vcmpeq4(a0, s[r + 1].x)) | (pack4(__vcmpeq4(a1, s[r + 1].y)) << 4);
                R |= eq_r << (8 * r);
                D |= eq_d << (8 * r);
            }
        }
        R &= dm.x;
        D &= dm.y;
    }
    R &= P.thr_any;
    D &= P.thr_any;
    S.edge[tid] = (D >> 24) | ((R >> 24) << 8) | (pack4((R >> 7) & 0x01010101u) << 16) | (pack4((D >> 7) & 0x00010101u) << 20);

    // bond words cover 16 sites = my row and my lane-pair partner's: the even lane stores rows 0-1, the odd lane rows 2-3
    const uint32_t odd = bx & 1u;
    {
        const uint32_t pR = __shfl_xor_sync(0xFFFFFFFFu, R, 1), pD = __shfl_xor_sync(0xFFFFFFFFu, D, 1);
        const uint32_t Re = odd ? pR : R, Ro = odd ? R : pR, De = odd ? pD : D, Do = odd ? D : pD;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint32_t r = 2u * odd + h, sel = r | ((4u + r) << 4);
            const uint32_t word = __byte_perm(__byte_perm(Re, Ro, sel), __byte_perm(De, Do, sel), 0x5410);
            bonds[(a0 + r * W) >> 4] = word;
        }
    }
    Bar::sync();                                               // B1: parent[], edge[] visible

    // -- the bonds that leave the tile (warp 0): right bonds of block column 7, down bonds of block row 15
    if (warp == 0) {
        const uint32_t nib = (S.edge[((lane & 15u) << 3) + 7u] >> 16) & 15u;          // block (7, lane): bit r = right bond of its row r
        const uint32_t dn = S.edge[120u + (lane & 7u)] & 0xFFu;                       // block (lane, 15): down bonds of columns 8 lane .. + 7
        const uint32_t r_lo = __reduce_or_sync(0xFFFFFFFFu, lane < 8u ? nib << (4u * lane) : 0u);
        const uint32_t r_hi = __reduce_or_sync(0xFFFFFFFFu, (lane >= 8u && lane < 16u) ? nib << (4u * (lane - 8u)) : 0u);
        const uint32_t b_lo = __reduce_or_sync(0xFFFFFFFFu, lane < 4u ? dn << (8u * lane) : 0u);
        const uint32_t b_hi = __reduce_or_sync(0xFFFFFFFFu, (lane >= 4u && lane < 8u) ? dn << (8u * (lane - 4u)) : 0u);
        if (lane == 0) {
            TileBorder b;
            b.right_col = (unsigned long long)r_lo | ((unsigned long long)r_hi << 32);
            b.bottom_row = (unsigned long long)b_lo | ((unsigned long long)b_hi << 32);
            border[tile] = b;
        }
    }

    // -- masks of my block.  Site sets are 32-bit masks, bit j = 8 r + c.
    const uint32_t A = R & 0x7F7F7F7Fu;                        // bit j: bond j -- j+1 inside the block
    const uint32_t A2 = A & (A >> 1), A4 = A2 & (A2 >> 2);
    const uint32_t Dl = D & 0x00FFFFFFu;                       // bit j: bond j -- j+8 inside the block
    const uint32_t Ds = Dl << 8;
    // links to other blocks of the tile, as masks over MY sites
    const uint32_t e_up = by > 0u ? S.edge[tid - 8u] : 0u, e_left = bx > 0u ? S.edge[tid - 1u] : 0u;
    const uint32_t up_row3 = e_up & 0xFFu;                                            // bit c: (block above, row 3, c) -- my (0, c)
    const uint32_t left_c7 = (((e_left >> 16) & 15u) * 0x00204081u) & 0x01010101u;    // bit 8r: (left block, r, 7) -- my (r, 0)
    const uint32_t out = (by < 15u ? D & 0xFF000000u : 0u) | (bx < 7u ? R & 0x80808080u : 0u);
    // sites that belong to a component worth a slot: any bond inside the block, or a link to another block
    const uint32_t todo = A | (A << 1) | Dl | Ds | up_row3 | left_c7 | out;

    // -- flood fill, component by component, smallest unvisited site first
    uint32_t n = 0;                                            // components found
    {
        uint32_t rem = todo;
        uint32_t m = rem & (0u - rem);
        while (m) {
            m = hclose(m, A, A2, A4);
            const uint32_t v = (((m << 8) & Ds) | ((m >> 8) & Dl)) & ~m;
            if (v) {
                m |= v;
            } else {
                S.list[n][tid] = m;
                ++n;
                rem &= ~m;
                m = rem & (0u - rem);
            }
        }
    }

    // -- bit-sliced slot numbers (plane b holds bit b of the slot of every site) and the seed of every component
    uint32_t P0 = 0, P1 = 0, P2 = 0, P3 = 0, P4 = 0;
    {
        const uint32_t n_max = __reduce_max_sync(0xFFFFFFFFu, n);
#pragma unroll
        for (int k = 0; k < kBlkSlots; ++k) {
            if ((uint32_t)k >= n_max) break;                  // warp-uniform
            if ((uint32_t)k < n) {
                const uint32_t m = S.list[k][tid];
                if (k & 1) P0 |= m;
                if (k & 2) P1 |= m;
                if (k & 4) P2 |= m;
                if (k & 8) P3 |= m;
                if (k & 16) P4 |= m;
                const uint32_t j = __ffs(m) - 1u;
                S.list[k][tid] = (idbase + ((j >> 3) << 6) + (j & 7u)) | (j << 16);
            }
        }
    }

    // -- publish the seeds of my bottom row for the block below (its up-links become plain-store parents); the sites
    //    of my right column point at the seed of their component, and the block on my right links to those SITES
    //    (one more hop in its finds; those links go through the atomic pass anyway)
    {
        const uint32_t W3 = plane_row(P0, P1, P2, P3, 3u), V3 = (P4 >> 24) << 4;
#pragma unroll
        for (int c = 0; c < 8; ++c)
            S.pub_bottom[c][tid] = (uint16_t)S.list[slot_of(W3, V3, c)][tid];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const uint32_t Wr = plane_row(P0, P1, P2, P3, r), Vr = ((P4 >> (8 * r)) & 0xFFu) << 4;
            if ((todo >> (8 * r + 7)) & 1u) S.parent[idbase + (r << 6) + 7u] = (uint16_t)S.list[slot_of(Wr, Vr, 7u)][tid];
        }
    }

    // -- links between blocks.  A link that repeats its neighbour's (same two components) is dropped.  The first
    //    up-link of every component becomes its parent by plain store (the seed above is a smaller id, and a
    //    component is written once: a forest); every other link needs the atomic pass after the barrier.
    auto walk_links = [&](auto &&on_first, auto &&on_other) {
        if (up_row3) {
            const uint32_t W0 = plane_row(P0, P1, P2, P3, 0u), V0 = (P4 & 0xFFu) << 4;
            const uint32_t R_up = (e_up >> 8) & 0xFFu;
            uint32_t u = up_row3 & ~((up_row3 & A & R_up & 0x7Fu) << 1);
            uint32_t seen = 0;
            while (u) {
                const uint32_t c = __ffs(u) - 1u;
                u &= u - 1u;
                const uint32_t k = slot_of(W0, V0, c);
                const uint32_t a = S.list[k][tid] & 0xFFFFu, b = S.pub_bottom[c][tid - 8u];
                if (!((seen >> k) & 1u)) {
                    seen |= 1u << k;
                    on_first(a, b);
                } else {
                    on_other(a, b);
                }
            }
        }
        if (left_c7) {
            const uint32_t D_left = (((e_left >> 20) & 7u) * 0x00204081u) & 0x00010101u;
            uint32_t l = left_c7 & ~((left_c7 & Dl & D_left) << 8);
            while (l) {
                const uint32_t j = __ffs(l) - 1u, r = j >> 3;
                l &= l - 1u;
                const uint32_t Wr = plane_row(P0, P1, P2, P3, r), Vr = ((P4 >> j) & 0xFFu) << 4;
                on_other(S.list[slot_of(Wr, Vr, 0u)][tid] & 0xFFFFu, idbase + (r << 6) - 1u);   // the site on my left
            }
        }
    };
    const bool crowded = Bar::sync_or(n > (uint32_t)kBlkBufSlot);   // B2: seeds of all blocks visible
    uint32_t *const buf = &S.list[kBlkBufSlot][0] + warp * kBlkExtraCap;
    if (!crowded) {
        walk_links([&](uint32_t a, uint32_t b) { S.parent[a] = (uint16_t)b; },
                   [&](uint32_t a, uint32_t b) { buf[atomicAdd(&S.n_extra[warp], 1u)] = a | (b << 16); });
    } else {
        walk_links([&](uint32_t a, uint32_t b) { S.parent[a] = (uint16_t)b; }, [](uint32_t, uint32_t) {});
    }
    Bar::sync();                                               // B3: the plain-store forest is complete
    if (!crowded) {
        const uint32_t n_warp = S.n_extra[warp];
        for (uint32_t k = lane; k < n_warp; k += 32) {
            const uint32_t e = buf[k];
            unite_s16(S.parent, e & 0xFFFFu, e >> 16);
        }
    } else {
        walk_links([](uint32_t, uint32_t) {}, [&](uint32_t a, uint32_t b) { unite_s16(S.parent, a, b); });
    }
    Bar::sync();                                               // B4: no hooks happen any more

    // -- every component: its root (chase; compress my own entry only) and root flag
    uint32_t rootm = ~todo;                                    // a site without any bond is its own cluster
    {
        volatile uint16_t *par = S.parent;
        for (uint32_t k = 0; k < n; ++k) {
            const uint32_t e = S.list[k][tid], id = e & 0xFFFFu;
            // three unconditional hops (a root points at itself, so hopping on is harmless), then the rare long chain
            const uint32_t r1 = par[id], r2 = par[r1];
            uint32_t r = r2, g = par[r2];
            while (g != r) { r = g; g = par[r]; }
            if (r != r1) par[id] = (uint16_t)r;
            rootm |= (uint32_t)(r == id) << (e >> 16);
            S.list[k][tid] = r;
        }
    }

    // -- labels: a tile-local root keeps its own global index (the merge links it from there), every other site
    //    gets the tile-local id of its root; root bitmap; roots of the edge sites as global indices for the merge
    const bool five = __any_sync(0xFFFFFFFFu, n > 16u);
    auto global_of = [&](uint32_t v) { return origin + (v >> 6) * L + (v & 63u); };
    uint32_t col_l[4], col_r[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const uint32_t Wr = plane_row(P0, P1, P2, P3, r), Vr = ((P4 >> (8 * r)) & 0xFFu) << 4;
        const uint32_t self = i0 + r * L;
        uint32_t lab[8];
        if (!five) {
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const uint32_t v = S.list[slot_of4(Wr, c)][tid];
                lab[c] = ((rootm >> (8 * r + c)) & 1u) ? self + c : v;
            }
        } else {
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const uint32_t v = S.list[slot_of(Wr, Vr, c)][tid];
                lab[c] = ((rootm >> (8 * r + c)) & 1u) ? self + c : v;
            }
        }
        uint4 *lp = reinterpret_cast<uint4 *>(labels + (uint64_t)(y0 + r) * W + x0);
        lp[0] = make_uint4(lab[0], lab[1], lab[2], lab[3]);
        lp[1] = make_uint4(lab[4], lab[5], lab[6], lab[7]);
        col_l[r] = lab[0];
        col_r[r] = lab[7];
        if ((r == 0 && by == 0u) || (r == 3 && by == 15u)) {   // top / bottom row of the tile
            uint32_t g[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) g[c] = ((rootm >> (8 * r + c)) & 1u) ? lab[c] : global_of(lab[c]);
            uint4 *ep = reinterpret_cast<uint4 *>((r == 0 ? edges[tile].top : edges[tile].bottom) + 8u * bx);
            ep[0] = make_uint4(g[0], g[1], g[2], g[3]);
            ep[1] = make_uint4(g[4], g[5], g[6], g[7]);
        }
    }
    {
        const uint32_t pm = __shfl_xor_sync(0xFFFFFFFFu, rootm, 1);
        const uint32_t me = odd ? pm : rootm, mo = odd ? rootm : pm;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint32_t r = 2u * odd + h;
            rootbits[(a0 + r * W) >> 4] = (uint16_t)(((me >> (8 * r)) & 0xFFu) | (((mo >> (8 * r)) & 0xFFu) << 8));
        }
    }
    if (bx == 0u || bx == 7u) {                               // left / right column of the tile
        const uint32_t c = bx == 0u ? 0u : 7u;
        uint32_t g[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const uint32_t v = bx == 0u ? col_l[r] : col_r[r];
            g[r] = ((rootm >> (8 * r + c)) & 1u) ? v : global_of(v);
        }
        *reinterpret_cast<uint4 *>((bx == 0u ? edges[tile].left : edges[tile].right) + 4u * by) = make_uint4(g[0], g[1], g[2], g[3]);
    }
}

struct CtaBar {
    static __device__ __forceinline__ void sync() { __syncthreads(); }
    static __device__ __forceinline__ bool sync_or(bool p) { return __syncthreads_or(p) != 0; }
};

__global__ void __launch_bounds__(kBlkThreads, 9)
k_tile_blocks(const uint8_t *__restrict__ spins, uint32_t *__restrict__ bonds,
              uint32_t *__restrict__ labels, uint16_t *__restrict__ rootbits,
              TileBorder *__restrict__ border, TileEdges *__restrict__ edges, const uint2 *__restrict__ draws, Params P)
{
    __shared__ BlkShared S;
    tile_blocks_body<false, false, CtaBar>(S, blockIdx.x, blockIdx.y, spins, bonds, labels, rootbits, border, edges, draws, P, Dom{});   // grid = (tiles_x, tiles_x): no division
}

// the same for one sub-lattice of the super-lattice (sw_super.cu); grid = (W / 64, H / 64)
__global__ void __launch_bounds__(kBlkThreads, 9)
k_tile_blocks_super(const uint8_t *spins, uint32_t *__restrict__ bonds,
                    uint32_t *__restrict__ labels, uint16_t *__restrict__ rootbits,
                    TileBorder *__restrict__ border, TileEdges *__restrict__ edges, const uint2 *__restrict__ draws, Params P, Dom dom)
{
    __shared__ BlkShared S;
    tile_blocks_body<true, false, CtaBar>(S, blockIdx.x, blockIdx.y, spins, bonds, labels, rootbits, border, edges, draws, P, dom);
}

}  // namespace sw
