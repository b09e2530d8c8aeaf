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
//   * "which component is site j in" is kept bit-sliced in plane registers, transposed into one slot
//     nibble per site once all components are known.
// Only the components of the blocks (about 0.2 per site at q = 2, K_c instead of 0.53 horizontal
// runs per site) go through the shared-memory union-find, whose nodes ARE those components, over the
// bonds that cross a block edge (0.16 per site): first up-link of every component by plain store,
// the rest with a native 32-bit atomic minimum.
#pragma once

#include <type_traits>

#include "sw_common.cuh"
#include "sw_tiled.cuh"

namespace sw {

constexpr int kBlkThreads = 128;
constexpr int kBlkSlots = 26;                 // components of an 8 x 4 block that can have a link: <= 20 border singles + 6 pairs
constexpr int kBlkExtraCap = 32 * 11;         // per warp: <= 7 up-links + 4 left-links per thread go through atomics
constexpr uint32_t kOffMask = 0xFFFFu;        // the address half of a node entry

// The union-find of a tile runs over the COMPONENTS OF THE BLOCKS, not over sites: node (k, tid) = slot k of the block of
// thread tid, &node[k][tid].  Its entry is (seed id << 16) | the low 16 bits of the shared-memory address of its PARENT
// (the seed = smallest site of the component, as a tile-local id y * 64 + x; static shared memory lies in the first
// 64 KB of the CTA's window, so 16 bits hold the address and a hop is one logic instruction + one load; the upper
// bits `win` of a shared address are the same for the whole CTA: zero, or the rank of the CTA in its cluster); a
// root holds its own.  Entries are unique per node and ordered like the seeds, so hooking the larger root under the
// smaller is one native 32-bit atomicMin, the root of a tile-local component is its smallest site, and
// the upper half of a root's entry IS the label of the component's other sites.
struct BlkShared {
    uint32_t node[kBlkSlots][kBlkThreads];    // flood fill: component masks; then the entries (see above); rows >= kBlkBufSlot double as link buffer
    uint4 pub[kBlkThreads];                   // what the blocks below / to the right need to know about my components:
                                              //   .x  slots of my bottom row, nibble p(c) = 2 (c % 4) + c / 4 for column c
                                              //   .y  byte r = 5-bit slot of my site (r, 7)
                                              //   .z  bit p(c) = fifth slot bit of my bottom-row site c (blocks with > 16 components)
    uint32_t edge[kBlkThreads];               // bits 0-7 down bonds of row 3, 8-15 right bonds of row 3, 16-19 right bonds of
                                              // column 7, 20-22 down bonds of column 7 (rows 0-2)
    uint32_t n_extra[kBlkThreads / 32];
    uint32_t five;                            // some block of the tile has more than 16 components (slots need a fifth bit)
};
// what the kSizes instantiation needs on top (sw_sweep_measure with the largest cluster): per node, bits 0-12 the number
// of its sites -- summed into the root of its tile-local component after the last hook (a tile has 4096 sites) -- and
// bit 15: the component owns a site on the border of the tile
struct BlkSizesShared {
    uint16_t size[kBlkSlots][kBlkThreads];
    uint32_t n_tab;
};
constexpr uint32_t kBorderTabEntries = 256;   // per tile: <= 252 components can own one of the 252 border sites

// The links that need the atomic pass are buffered per warp in node rows kBlkBufSlot .. kBlkSlots-1, which are
// free unless some block of the tile has more than kBlkBufSlot components (then they are united unbuffered).
constexpr int kBlkBufSlot = 14;
static_assert((kBlkSlots - kBlkBufSlot) * kBlkThreads >= (kBlkThreads / 32) * kBlkExtraCap, "link buffer too small");

// shared-memory accesses by 32-bit shared address (volatile: other threads hook and re-point nodes concurrently)
__device__ __forceinline__ uint32_t ld_node(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void st_node(uint32_t addr, uint32_t e)
{
    asm volatile("st.volatile.shared.u32 [%0], %1;" :: "r"(addr), "r"(e) : "memory");
}
__device__ __forceinline__ uint32_t min_node(uint32_t addr, uint32_t e)
{
    uint32_t old;
    asm volatile("atom.shared.min.u32 %0, [%1], %2;" : "=r"(old) : "r"(addr), "r"(e) : "memory");
    return old;
}
// after the last hook: entries only ever change to the root's, either value ends the chase at the same root
__device__ __forceinline__ uint32_t ld_node_quiet(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t and_opaque(uint32_t a, uint32_t m)
{
    uint32_t v;
    asm("and.b32 %0, %1, %2;" : "=r"(v) : "r"(a), "r"(m));
    return v;
}
__device__ __forceinline__ uint32_t ld_label_half(uint32_t addr)
{
    uint16_t v;
    asm volatile("ld.shared.u16 %0, [%1+2];" : "=h"(v) : "r"(addr) : "memory");
    return v;
}

// Join the components of nodes a and b (shared-memory addresses).  A node is named by its own entry value s (s & kOffMask is
// where it lives); links point to smaller entries, plain stores only ever replace a link by a link to an ancestor,
// hooks are an atomic minimum: if the word hit was no longer a root, the link it held is not lost, we carry on
// uniting its old target (one pass over all links yields the complete partition).
__device__ __forceinline__ void unite_nodes(uint32_t a, uint32_t b, const uint32_t win)
{
    auto at = [win](uint32_t e) { return (e & kOffMask) | win; };     // where the node named by entry e lives
    uint32_t sa = ld_node(a), sb = ld_node(b);
    {   // one more unconditional hop on both sides (a root points at itself): most chases end here, branch-free
        const uint32_t na = ld_node(at(sa)), nb = ld_node(at(sb));
        if (na != sa) st_node(a, na);
        if (nb != sb) st_node(b, nb);
        sa = na; sb = nb;
    }
    while (true) {
        uint32_t pa = ld_node(at(sa)), pb = ld_node(at(sb));
        while (pa != sa || pb != sb) {
            const uint32_t ga = ld_node(at(pa)), gb = ld_node(at(pb));
            if (ga != pa) st_node(at(sa), ga);
            if (gb != pb) st_node(at(sb), gb);
            sa = ga; sb = gb;
            pa = ld_node(at(sa)); pb = ld_node(at(sb));
        }
        if (sa == sb) return;
        if (sa < sb) { const uint32_t t = sa; sa = sb; sb = t; }
        const uint32_t old = min_node(at(sa), sb);
        if (old == sa) return;
        sa = old;
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

// bit c of an 8-bit column mask -> bit p(c) = 2 (c % 4) + c / 4 (the order of the slot nibbles of a row)
__device__ __forceinline__ uint32_t perm8(uint32_t x)
{
    uint32_t t = (x & 0x0Fu) | ((x & 0xF0u) << 4);            // columns 0-3 in bits 0-3, columns 4-7 in bits 8-11
    t = (t | (t << 2)) & 0x3333u;
    t = (t | (t << 1)) & 0x5555u;
    return (t | (t >> 7)) & 0xFFu;
}

// exchange the bits of hi selected by m << s with the bits of lo selected by m (delta swap across two registers)
__device__ __forceinline__ void delta_swap(uint32_t &lo, uint32_t &hi, uint32_t s, uint32_t m)
{
    const uint32_t t = ((lo >> s) ^ hi) & m;
    hi ^= t;
    lo ^= t << s;
}

// The body of the tile kernel for tile (tx, ty) of a piece of the lattice, run by kBlkThreads threads.
//   kSuper     the piece is a sub-lattice of the super-lattice (label values global, addresses local: `dom`);
//              false: the whole lattice, dom is not looked at
//   kCoherent  see ld_in
//   Bar        the CTA-wide barrier of those kBlkThreads threads
//   kSizes     also count the sites of every tile-local component.  A component that owns no site on the border of the
//              tile IS a whole cluster: its size only raises row[2] (the largest cluster so far).  The others go to the
//              tile's border table btab[tile][0..255] as (root's tile-local id | size << 12; 0 = unused entry) for the
//              flip kernel, which adds them up per cluster (k_tile_flip_sizes); whole lattice only
template <bool kSuper, bool kCoherent, class Bar, bool kSizes = false>
__device__ __forceinline__ void
tile_blocks_body(BlkShared &S, const uint32_t tx, const uint32_t ty, const uint8_t *spins, uint32_t *bonds,
                 uint32_t *labels, uint16_t *rootbits, TileBorder *border, TileEdges *edges, const uint2 *draws,
                 const Params &P, const Dom &dom, BlkSizesShared *Zs = nullptr, uint32_t *btab = nullptr,
                 unsigned long long *row = nullptr)
{
    static_assert(!(kSizes && kSuper), "the size counts are made for the whole lattice only");
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
    const uint32_t mybase = (uint32_t)__cvta_generic_to_shared(&S.node[0][tid]);   // shared address of my column of node[][]
    // its window bits (only a CTA of a multi-CTA cluster has any: the kCoherent instantiation) / its 16 address bits in an entry
    const uint32_t win = kCoherent ? mybase & ~kOffMask : 0u, my16 = mybase & kOffMask;

    if (tid < kBlkThreads / 32) S.n_extra[tid] = 0;
    if (tid == 32) S.five = 0;
    if (kSizes && tid == 64) Zs->n_tab = 0;
    // kSizes: my sites on the border of the tile
    const uint32_t bmask = !kSizes ? 0u : (by == 0u ? 0x000000FFu : 0u) | (by == 15u ? 0xFF000000u : 0u) |
                                          (bx == 0u ? 0x01010101u : 0u) | (bx == 7u ? 0x80808080u : 0u);

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
        } else if (P.q <= 4u) {                                // states are two bits: equal iff the XOR has neither (bit 0 of the NOR)
            auto eq2 = [](uint32_t a, uint32_t b) { const uint32_t d = a ^ b; return ~(d | (d >> 1)); };
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const uint32_t a0 = s[r].x, a1 = s[r].y;
                const uint32_t n0 = __funnelshift_r(a0, a1, 8), n1 = __funnelshift_r(a1, nx >> (8 * r), 8);
                R |= (pack4(eq2(a0, n0)) | (pack4(eq2(a1, n1)) << 4)) << (8 * r);
                D |= (pack4(eq2(a0, s[r + 1].x)) | (pack4(eq2(a1, s[r + 1].y)) << 4)) << (8 * r);
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
    Bar::sync();                                               // B1: edge[], n_extra[], five visible

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
                S.node[n][tid] = m;
                ++n;
                rem &= ~m;
                m = rem & (0u - rem);
            }
        }
    }
    if (n > 16u) S.five = 1u;

    // -- bit-sliced slot numbers (plane b holds bit b of the slot of every site); every component becomes a root node
    uint32_t Q0 = 0, Q1 = 0, Q2 = 0, Q3 = 0, P4 = 0;
    {
        const uint32_t n_max = __reduce_max_sync(0xFFFFFFFFu, n);
#pragma unroll
        for (int k = 0; k < kBlkSlots; ++k) {
            if ((uint32_t)k >= n_max) break;                  // warp-uniform
            if ((uint32_t)k < n) {
                const uint32_t m = S.node[k][tid];
                if (k & 1) Q0 |= m;
                if (k & 2) Q1 |= m;
                if (k & 4) Q2 |= m;
                if (k & 8) Q3 |= m;
                if (k & 16) P4 |= m;
                if (kSizes) Zs->size[k][tid] = (uint16_t)(__popc(m) | ((m & bmask) ? 0x8000u : 0u));
                const uint32_t j = __ffs(m) - 1u;
                S.node[k][tid] = ((idbase + ((j >> 3) << 6) + (j & 7u)) << 16) + ((uint32_t)k * 512u + my16);
            }
        }
    }
    // planes 0-3 -> slot nibbles: afterwards nibble g of Q_i is the slot (mod 16) of site 4 g + i, i.e. of (r, c) with
    // i = c % 4, g = 2 r + c / 4 (a 4 x 4 bit transpose across the four registers)
    delta_swap(Q0, Q1, 1u, 0x55555555u);
    delta_swap(Q2, Q3, 1u, 0x55555555u);
    delta_swap(Q0, Q2, 2u, 0x33333333u);
    delta_swap(Q1, Q3, 2u, 0x33333333u);

    // -- publish the slots of my bottom row and of my right column for the blocks below / to the right
    {
        const uint32_t bottom = __byte_perm(__byte_perm(Q0, Q1, 0x0073), __byte_perm(Q2, Q3, 0x0073), 0x5410);   // byte i = top byte of Q_i
        const uint32_t col7 = ((Q3 >> 4) & 0x0F0F0F0Fu) | (((P4 >> 7) & 0x01010101u) << 4);
        S.pub[tid] = make_uint4(bottom, col7, P4 ? perm8(P4 >> 24) : 0u, 0u);
    }
    const uint32_t N0 = __byte_perm(__byte_perm(Q0, Q1, 0x0040), __byte_perm(Q2, Q3, 0x0040), 0x5410);           // slots of my row 0, nibble p(c)

    // -- links between blocks.  A link that repeats its neighbour's (same two components) is dropped.  The first
    //    up-link of every component becomes its parent by plain store (the component above has a smaller seed, and a
    //    component is written once: a forest); every other link needs the atomic pass after the barrier.
    auto walk_links = [&](auto five_, auto &&on_first, auto &&on_other) {
        constexpr bool kFive = decltype(five_)::value;
        if (up_row3) {
            const uint4 pu = S.pub[tid - 8u];
            const uint32_t R_up = (e_up >> 8) & 0xFFu;
            uint32_t u = perm8(up_row3 & ~((up_row3 & A & R_up & 0x7Fu) << 1));
            const uint32_t p4a = kFive ? perm8(P4 & 0xFFu) : 0u;
            uint32_t seen = 0;
            while (u) {
                const uint32_t p = __ffs(u) - 1u, sh = p << 2;
                u &= u - 1u;
                uint32_t ka = (N0 >> sh) & 15u, kb = (pu.x >> sh) & 15u;
                if (kFive) { ka |= ((p4a >> p) & 1u) << 4; kb |= ((pu.z >> p) & 1u) << 4; }
                const uint32_t a = (ka << 9) + mybase, b = (kb << 9) + mybase - 32u;
                if (!((seen >> ka) & 1u)) {
                    seen |= 1u << ka;
                    on_first(a, b);
                } else {
                    on_other(a, b);
                }
            }
        }
        if (left_c7) {
            const uint32_t pl = S.pub[tid - 1u].y;
            const uint32_t D_left = (((e_left >> 20) & 7u) * 0x00204081u) & 0x00010101u;
            uint32_t l = left_c7 & ~((left_c7 & Dl & D_left) << 8);
            while (l) {
                const uint32_t j = __ffs(l) - 1u;              // = 8 r
                l &= l - 1u;
                uint32_t ka = (Q0 >> j) & 15u;                 // site (r, 0) is nibble 2 r of Q0
                if (kFive) ka |= ((P4 >> j) & 1u) << 4;
                const uint32_t kb = (pl >> j) & 31u;
                on_other((ka << 9) + mybase, (kb << 9) + mybase - 4u);
            }
        }
    };
    const bool crowded = Bar::sync_or(n > (uint32_t)kBlkBufSlot);   // B2: the nodes and the published slots of all blocks visible
    const bool five = S.five != 0u;
    uint32_t *const buf = &S.node[kBlkBufSlot][0] + warp * kBlkExtraCap;
    auto first = [&](uint32_t a, uint32_t b) { st_node(a, ld_node(b)); };   // b's entry, or already its parent's: an ancestor either way
    if (!crowded) {
        walk_links(std::false_type{}, first, [&](uint32_t a, uint32_t b) { buf[atomicAdd(&S.n_extra[warp], 1u)] = (a & kOffMask) | (b << 16); });
    } else if (!five) {
        walk_links(std::false_type{}, first, [](uint32_t, uint32_t) {});
    } else {
        walk_links(std::true_type{}, first, [](uint32_t, uint32_t) {});
    }
    Bar::sync();                                               // B3: the plain-store forest is complete
    if (!crowded) {
        const uint32_t n_warp = S.n_extra[warp];
        for (uint32_t k = lane; k < n_warp; k += 32) {
            const uint32_t e = buf[k];
            unite_nodes((e & kOffMask) | win, (e >> 16) | win, win);
        }
    } else if (!five) {
        walk_links(std::false_type{}, [](uint32_t, uint32_t) {}, [&](uint32_t a, uint32_t b) { unite_nodes(a, b, win); });
    } else {
        walk_links(std::true_type{}, [](uint32_t, uint32_t) {}, [&](uint32_t a, uint32_t b) { unite_nodes(a, b, win); });
    }
    Bar::sync();                                               // B4: no hooks happen any more

    // -- every component: its root (chase, then point my node straight at it: the labels below read it from there)
    uint32_t rootm = ~todo;                                    // a site without any bond is its own cluster
    uint32_t rootk = 0;                                        // kSizes: bit k = my node k is a root
    for (uint32_t k = 0; k < n; ++k) {
        const uint32_t me = (k << 9) + mybase;
        auto at = [win](uint32_t e) { return (e & kOffMask) | win; };
        // three unconditional hops (a root points at itself, so hopping on is harmless), then the rare long chain
        const uint32_t r1 = ld_node_quiet(me), r2 = ld_node_quiet(at(r1));
        uint32_t r = r2, g = ld_node_quiet(at(r2));
        while (g != r) { r = g; g = ld_node_quiet(at(r)); }
        if (r != r1) st_node(me, r);
        if (at(r) == me) {
            rootm |= 1u << (((r >> 19) & 24u) | ((r >> 16) & 7u));   // my seed (y * 64 + x): bit 8 (y % 4) + x % 8
            if (kSizes) rootk |= 1u << k;
        } else if (kSizes) {                                   // my sites count for the root (two 16-bit fields per word)
            const uint32_t idx = (at(r) - (mybase - (tid << 2))) >> 2;            // node index 128 k' + tid' of the root
            uint32_t *const word = reinterpret_cast<uint32_t *>(&Zs->size[0][0]) + (idx >> 1);
            const uint32_t sh = (idx & 1u) << 4, mine = Zs->size[k][tid];
            atomicAdd(word, (mine & 0x1FFFu) << sh);
            if (mine & 0x8000u) atomicOr(word, 0x8000u << sh);
        }
    }
    if (kSizes) {
        Bar::sync();                                           // all counts are in; pub[] is free (the table is built there)
        uint32_t *const tab = reinterpret_cast<uint32_t *>(&S.pub[0]);
        uint32_t whole = 0;                                    // largest component of mine that lies inside the tile
        while (rootk) {
            const uint32_t k = __ffs(rootk) - 1u;
            rootk &= rootk - 1u;
            const uint32_t f = Zs->size[k][tid], total = f & 0x1FFFu;
            if (f & 0x8000u) tab[atomicAdd(&Zs->n_tab, 1u)] = (S.node[k][tid] >> 16) | (total << 12);   // a root holds its own entry: its seed
            else whole = max(whole, total);
        }
        uint32_t lone = ~todo & bmask;                         // border sites without a bond inside the tile: components of one
        while (lone) {
            const uint32_t j = __ffs(lone) - 1u;
            lone &= lone - 1u;
            tab[atomicAdd(&Zs->n_tab, 1u)] = (idbase + ((j >> 3) << 6) + (j & 7u)) | (1u << 12);
        }
        whole = __reduce_max_sync(0xFFFFFFFFu, whole);
        if (lane == 0 && whole) atomicMax(row + 2, (unsigned long long)whole);
        Bar::sync();
        const uint32_t n_tab = Zs->n_tab;
#pragma unroll
        for (uint32_t e = tid; e < kBorderTabEntries; e += kBlkThreads) btab[tile * kBorderTabEntries + e] = e < n_tab ? tab[e] : 0u;
    }

    // -- labels: a tile-local root keeps its own global index (the merge links it from there), every other site
    //    gets the tile-local id of its root (the upper half of its component's node); root bitmap; roots of the edge
    //    sites as global indices for the merge
    const bool five_w = __any_sync(0xFFFFFFFFu, n > 16u);      // (also reconverges the warp after the chases)
    auto global_of = [&](uint32_t v) { return origin + (v >> 6) * L + (v & 63u); };
    uint32_t col_l[4], col_r[4];
    auto write_labels = [&](auto five_) {
        constexpr bool kFive = decltype(five_)::value;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const uint32_t self = i0 + r * L, rb = __byte_perm(rootm, 0, 0x4440 + r);
            uint32_t lab[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                // my slot nibble sits at bit sh of Q_(c % 4); * 512 = the row of node[][].  (The AND is opaque to the
                // compiler so that it stays in front of the shift: mask, then one shift-and-add.)
                const uint32_t Qi = (c & 3) == 0 ? Q0 : (c & 3) == 1 ? Q1 : (c & 3) == 2 ? Q2 : Q3;
                constexpr int kZero = 0;
                const int sh = 4 * (2 * r + (c >> 2)) + kZero;
                const uint32_t x = and_opaque(Qi, 0xFu << sh);
                uint32_t o = mybase + (sh <= 9 ? x << (9 - sh) : x >> (sh - 9));
                if (kFive) o += ((P4 >> (8 * r + c)) & 1u) << 13;
                uint32_t v = ld_label_half(o);
                if (rb & (1u << c)) v = self + c;
                lab[c] = v;
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
    };
    if (!five_w) write_labels(std::false_type{});
    else write_labels(std::true_type{});
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

#ifndef SW_BLK_CTAS
#define SW_BLK_CTAS 12
#endif
__global__ void __launch_bounds__(kBlkThreads, SW_BLK_CTAS)
k_tile_blocks(const uint8_t *__restrict__ spins, uint32_t *__restrict__ bonds,
              uint32_t *__restrict__ labels, uint16_t *__restrict__ rootbits,
              TileBorder *__restrict__ border, TileEdges *__restrict__ edges, const uint2 *__restrict__ draws, Params P)
{
    __shared__ BlkShared S;
    tile_blocks_body<false, false, CtaBar>(S, blockIdx.x, blockIdx.y, spins, bonds, labels, rootbits, border, edges, draws, P, Dom{});   // grid = (tiles_x, tiles_x): no division
}

// the same, and the sizes of the tile-local components (see kSizes)
__global__ void __launch_bounds__(kBlkThreads, 9)
k_tile_blocks_sizes(const uint8_t *__restrict__ spins, uint32_t *__restrict__ bonds,
                    uint32_t *__restrict__ labels, uint16_t *__restrict__ rootbits,
                    TileBorder *__restrict__ border, TileEdges *__restrict__ edges, const uint2 *__restrict__ draws, Params P,
                    uint32_t *__restrict__ btab, unsigned long long *__restrict__ row)
{
    __shared__ BlkShared S;
    __shared__ BlkSizesShared Z;
    tile_blocks_body<false, false, CtaBar, true>(S, blockIdx.x, blockIdx.y, spins, bonds, labels, rootbits, border, edges, draws, P, Dom{}, &Z, btab, row);
}

// the same for one sub-lattice of the super-lattice (sw_super.cu); grid = (W / 64, H / 64)
__global__ void __launch_bounds__(kBlkThreads, SW_BLK_CTAS)
k_tile_blocks_super(const uint8_t *spins, uint32_t *__restrict__ bonds,
                    uint32_t *__restrict__ labels, uint16_t *__restrict__ rootbits,
                    TileBorder *__restrict__ border, TileEdges *__restrict__ edges, const uint2 *__restrict__ draws, Params P, Dom dom)
{
    __shared__ BlkShared S;
    tile_blocks_body<true, false, CtaBar>(S, blockIdx.x, blockIdx.y, spins, bonds, labels, rootbits, border, edges, draws, P, dom);
}

}  // namespace sw
