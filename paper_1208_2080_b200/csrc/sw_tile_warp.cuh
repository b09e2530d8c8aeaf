// sw_tile_warp.cuh -- bonds + tile-local labeling with ONE WARP per 64 x 64 tile.
//
//   step (1) of the sweep and the tile-local part of step (2)   ("done
//   independently on each site").  The labeling is a Hoshen-Kopelman scan (labels are
//   handed out row by row, equivalences go into a label[label] table, "proper label" = the smallest
//   label of the cluster) run by every thread on its own 16 x 8 block, followed by the boundary-only
//   merge of PAPER.md:66-68 one level down: blocks of a tile instead of sub-lattices of GPUs.
//
// Thread (by = lane / 4, bx = lane % 4) owns the block of rows 8 by .. 8 by + 7, columns
// 16 bx .. 16 bx + 15 of its warp's tile.
//   bonds    per row: one 16-byte spin load (+ the row below, + 4 halo bytes), byte-wise SIMD
//            compares, 8 Philox calls (one per site pair), one 32-bit bond word.
//   level 0  sequential over the 7 inner row boundaries of the block: the first up-link of a piece
//            gives it the root of the piece above by a plain store, every further up-link is a
//            find + hook inside the thread's own entries.  No atomics, no barriers, depth stays
//            small because pieces are attached to ROOTS.
//   level 1  the links that cross block borders (<= 16 + 8 per thread, ~9 survive the duplicate
//            filter): lock-step rounds of find / hook by plain 16-bit store / verify, separated by
//            __syncwarp.  A hook that lost a same-address race is retried from the winner.
//   resolve  every piece of the thread is pointed straight at its tile root.
//   output   labels (global index of the tile-local minimum), tile-root bitmap, border record.
//
// Node ids are plain tile-local site indices y * 64 + x in a uint16 table (8 KB per tile), so
// "smaller id" is "smaller site index" and the root of a set is its smallest member.
#pragma once

#include "sw_tiled.cuh"

namespace sw {

constexpr int kTwWarps = 4;                                  // tiles (= warps) per CTA
constexpr int kTwThreads = kTwWarps * 32;
constexpr uint32_t kFull = 0xFFFFFFFFu;

__device__ __forceinline__ uint32_t find16(const uint16_t *par, uint32_t a)
{
    uint32_t p = par[a];
    while (p != a) { a = p; p = par[a]; }
    return a;
}

__global__ void __launch_bounds__(kTwThreads, 6)
k_tile_warp(const uint8_t *__restrict__ spins, uint32_t *__restrict__ bonds,
            uint32_t *__restrict__ labels, uint16_t *__restrict__ rootbits,
            TileBorder *__restrict__ border, TileCols *__restrict__ cols, Params P, uint32_t n_tiles)
{
    __shared__ __align__(16) uint16_t s_par_all[kTwWarps][kTileSites];
    __shared__ uint32_t s_rd_all[kTwWarps][kTile * 4];       // [row][bx]: tile-local right bonds | down bonds << 16

    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t tile = blockIdx.x * kTwWarps + warp;
    if (tile >= n_tiles) return;                             // whole warp leaves; nothing below is CTA-wide
    uint16_t *par = s_par_all[warp];
    uint32_t *s_rd = s_rd_all[warp];

    const uint32_t bx = lane & 3u, by = lane >> 2;
    const uint32_t L = P.L, tiles_x = L >> 6;
    const uint32_t ty = tile / tiles_x, tx = tile - ty * tiles_x;
    const uint32_t X0 = tx << 6, Y0 = ty << 6;
    const uint32_t y0 = by << 3;                             // first tile row of my block
    const uint32_t gx = X0 + (bx << 4);
    const uint32_t gxn = (gx + 16 == L) ? 0u : gx + 16;      // column of the right neighbour of my last site
    const uint32_t base0 = (y0 << 6) + (bx << 4);            // node id of my block's first site

    // ---- bonds: 8 rows, software-pipelined loads ------------------------------------------------
    {
        uint32_t gy = Y0 + y0;
        uint4 cur = *reinterpret_cast<const uint4 *>(spins + (uint64_t)gy * L + gx);
        uint32_t nxt = *reinterpret_cast<const uint32_t *>(spins + (uint64_t)gy * L + gxn);
        uint32_t rc = 0;                                     // right-column border bits of my 8 rows (bx == 3)
#pragma unroll 1
        for (uint32_t r = 0; r < 8; ++r) {
            const uint64_t row_off = (uint64_t)gy * L;
            const uint32_t gyd = (gy + 1 == L) ? 0u : gy + 1;
            const uint4 dn = *reinterpret_cast<const uint4 *>(spins + (uint64_t)gyd * L + gx);
            const uint32_t nxt_dn = *reinterpret_cast<const uint32_t *>(spins + (uint64_t)gyd * L + gxn);
            const uint32_t i0 = (uint32_t)(row_off + gx);

            // draws first: they do not depend on the loads
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
            const uint32_t w[4] = {cur.x, cur.y, cur.z, cur.w};
            const uint32_t dw[4] = {dn.x, dn.y, dn.z, dn.w};
            uint32_t eq_r = 0, eq_d = 0;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t rr = __funnelshift_r(w[k], (k < 3) ? w[k + 1] : nxt, 8);
                eq_r |= pack4(__vcmpeq4(w[k], rr)) << (4 * k);
                eq_d |= pack4(__vcmpeq4(w[k], dw[k])) << (4 * k);
            }
            const uint32_t r16 = eq_r & m_r & P.thr_any;
            const uint32_t d16 = eq_d & m_d & P.thr_any;
            bonds[i0 >> 4] = r16 | (d16 << 16);
            rc |= (r16 >> 15) << r;
            const uint32_t lr16 = (bx == 3) ? (r16 & 0x7FFFu) : r16;   // the bond that leaves the tile goes to the border record
            s_rd[((y0 + r) << 2) + bx] = lr16 | (d16 << 16);
            // every entry of my row segment starts as its own root (only piece starts are ever used)
            const uint32_t id0 = base0 + (r << 6);
            const uint32_t pk = id0 * 0x10001u;
            uint4 *pp = reinterpret_cast<uint4 *>(par + id0);
            pp[0] = make_uint4(pk + 0x00010000u, pk + 0x00030002u, pk + 0x00050004u, pk + 0x00070006u);
            pp[1] = make_uint4(pk + 0x00090008u, pk + 0x000B000Au, pk + 0x000D000Cu, pk + 0x000F000Eu);
            if (by == 7 && r == 7)
                reinterpret_cast<uint16_t *>(&border[tile].bottom_row)[bx] = (uint16_t)d16;
            cur = dn; nxt = nxt_dn; gy = gyd;
        }
        if (bx == 3) reinterpret_cast<uint8_t *>(&border[tile].right_col)[by] = (uint8_t)rc;
    }
    // (from here on a thread only reads its OWN s_rd / par entries until level 1)

    // ---- level 0: Hoshen-Kopelman scan of my block ----------------------------------------------
    {
        uint32_t up = s_rd[(y0 << 2) + bx];
#pragma unroll 1
        for (uint32_t r = 1; r < 8; ++r) {
            const uint32_t me = s_rd[((y0 + r) << 2) + bx];
            const uint32_t s = up >> 16;                          // bit x: up-link (row r-1, x) -- (row r, x)
            const uint32_t S_up = starts_of(up & 0xFFFFu), S = starts_of(me & 0xFFFFu);
            const uint32_t C = S ^ 0xFFFFu;                      // bit x: site x continues the piece of x-1
            // first up-link of every piece (carry chain: generate = s, propagate = C)
            const uint32_t A = s | C;
            const uint32_t cin = (A + s) ^ A ^ s;
            const uint32_t first = s & ~(cin & C);
            // an up-link whose left neighbour is an up-link between the same two pieces says nothing new
            uint32_t v = s & ~((s << 1) & C & ~S_up);
            const uint32_t b_up = base0 + ((r - 1) << 6), b_me = base0 + (r << 6);
            while (v) {
                const uint32_t bit = v & (0u - v);
                v ^= bit;
                const uint32_t below = (bit << 1) - 1u;          // bits 0..x
                const uint32_t a = find16(par, b_up + 31u - __clz(S_up & below));
                const uint32_t id = b_me + 31u - __clz(S & below);
                if (first & bit) {
                    par[id] = (uint16_t)a;
                } else {
                    const uint32_t b = find16(par, id);
                    if (a != b) par[max(a, b)] = (uint16_t)min(a, b);
                }
            }
            up = me;
        }
    }
    __syncwarp();

    // ---- level 1: links across block borders ------------------------------------------------------
    {
        uint32_t m = 0;
        if (by < 7) {                                            // my row 7 -- row 0 of the block below
            const uint32_t me = s_rd[((y0 + 7) << 2) + bx], lo = s_rd[((y0 + 8) << 2) + bx];
            const uint32_t s = me >> 16;
            const uint32_t C7 = starts_of(me & 0xFFFFu) ^ 0xFFFFu, Cl = starts_of(lo & 0xFFFFu) ^ 0xFFFFu;
            m = s & ~((s << 1) & C7 & Cl);
        }
#pragma unroll
        for (uint32_t r = 0; r < 8; ++r)                         // my last site -- first site of the block on my right
            m |= ((s_rd[((y0 + r) << 2) + bx] >> 15) & 1u) << (16 + r);

        uint32_t a = 0, b = 0;
        bool retry = false;
        while (true) {
            bool hook = false;
            if (retry) { a = find16(par, a); b = find16(par, b); hook = (a != b); retry = false; }
            while (!hook && m) {
                const uint32_t k = __ffs(m) - 1;
                m &= m - 1;
                if (k < 16) {
                    const uint32_t below = (2u << k) - 1u;
                    const uint32_t S7 = starts_of(s_rd[((y0 + 7) << 2) + bx] & 0xFFFFu);
                    const uint32_t Sl = starts_of(s_rd[((y0 + 8) << 2) + bx] & 0xFFFFu);
                    a = base0 + (7u << 6) + 31u - __clz(S7 & below);
                    b = base0 + (8u << 6) + 31u - __clz(Sl & below);
                } else {
                    const uint32_t r = k - 16;
                    const uint32_t Sr = starts_of(s_rd[((y0 + r) << 2) + bx] & 0xFFFFu);
                    a = base0 + (r << 6) + 31u - __clz(Sr);
                    b = base0 + (r << 6) + 16u;
                }
                a = find16(par, a); b = find16(par, b);
                hook = (a != b);
            }
            if (!__any_sync(kFull, hook)) break;
            const uint32_t hi = max(a, b), lo = min(a, b);
            __syncwarp();                                        // all finds of this round are done
            if (hook) par[hi] = (uint16_t)lo;
            __syncwarp();
            if (hook && par[hi] != lo) { retry = true; a = lo; b = hi; }   // lost a same-root race: go on from the winner
        }
    }
    __syncwarp();

    // ---- resolve: my pieces -> tile roots ------------------------------------------------------------
#pragma unroll
    for (uint32_t j = 0; j < 4; ++j) {
        uint32_t mm = starts_of(s_rd[((y0 + 2 * j) << 2) + bx] & 0xFFFFu) |
                      (starts_of(s_rd[((y0 + 2 * j + 1) << 2) + bx] & 0xFFFFu) << 16);
        const uint32_t jb = base0 + (j << 7);
        while (mm) {
            const uint32_t k = __ffs(mm) - 1;
            mm &= mm - 1;
            const uint32_t id = jb + ((k & 16u) << 2) + (k & 15u);
            const uint32_t p = par[id];
            if (p != id) {
                uint32_t rt = par[p];
                if (rt != p) {
                    uint32_t g = par[rt];
                    while (g != rt) { rt = g; g = par[rt]; }
                    par[id] = (uint16_t)rt;
                    par[p] = (uint16_t)rt;                       // the next piece that hangs under p gets there in two loads
                }
            }
        }
    }
    __syncwarp();

    // ---- output: labels, root flags ----------------------------------------------------------------
    {
        const uint32_t origin = Y0 * L + X0;
#pragma unroll 1
        for (uint32_t r = 0; r < 8; ++r) {
            const uint32_t S = starts_of(s_rd[((y0 + r) << 2) + bx] & 0xFFFFu);
            const uint32_t id0 = base0 + (r << 6);
            const uint4 q0 = *reinterpret_cast<const uint4 *>(par + id0);
            const uint4 q1 = *reinterpret_cast<const uint4 *>(par + id0 + 8);
            const uint32_t qq[8] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w};
            uint32_t lab[16];
            uint32_t curl = 0, roots = 0;
#pragma unroll
            for (int x = 0; x < 16; ++x) {
                if ((S >> x) & 1u) {
                    const uint32_t e = (x & 1) ? (qq[x >> 1] >> 16) : (qq[x >> 1] & 0xFFFFu);
                    curl = origin + (e >> 6) * L + (e & 63u);
                    roots |= (e == id0 + x) ? (1u << x) : 0u;
                }
                lab[x] = curl;
            }
            const uint64_t row_off = (uint64_t)(Y0 + y0 + r) * L;
            uint4 *lp = reinterpret_cast<uint4 *>(labels + row_off + gx);
            lp[0] = make_uint4(lab[0], lab[1], lab[2], lab[3]);
            lp[1] = make_uint4(lab[4], lab[5], lab[6], lab[7]);
            lp[2] = make_uint4(lab[8], lab[9], lab[10], lab[11]);
            lp[3] = make_uint4(lab[12], lab[13], lab[14], lab[15]);
            rootbits[(uint32_t)(row_off + gx) >> 4] = (uint16_t)roots;
            if (bx == 0) cols[tile].left[y0 + r] = lab[0];
            if (bx == 3) cols[tile].right[y0 + r] = lab[15];
        }
    }
}

}  // namespace sw
