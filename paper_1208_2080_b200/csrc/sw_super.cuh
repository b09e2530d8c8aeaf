// sw_super.cu -- the paper's own contribution, re-thought for NVLink-connected B200s: the lattice is cut into a
// gx x gy "super-lattice" of sub-lattices, one per GPU (Fig. 1), and labeled in two stages:
//
//   stage 1  inside every sub-lattice: the three kernels of the single-GPU path (bonds + tile-local labels, tile-border
//            merge, later the flatten + flip), with the bonds that leave the sub-lattice recorded but not united;
//   stage 2  between sub-lattices: only the 2 (W + H) boundary sites of each piece are looked at ("we use
//            only the 4 N_x sites of the boundary").
//
// What differs from the paper (Fermi + MPI, 2012), and why:
//   * No halo copies, no host staging (PAPER.md:54 GPU -> CPU -> MPI -> CPU -> GPU): the bond kernel of a piece reads the
//     first column / row of its right / lower neighbour directly through a peer pointer (NVLink P2P; the same pointer
//     arithmetic when the pieces share a device), 2 (W + H) bytes per sweep.
//   * No iterated label diffusion with a global "flag" gathered and broadcast every round (the number of
//     rounds grows with the number of GPUs): stage 2 is ONE pass of the same lock-free union-find the tile
//     merge uses -- find by peer loads, hook the larger root under the smaller with a system-scope atomicMin in the
//     owner's memory -- so the "flag" degenerates to one barrier: all pieces have finished stage 2.
//   * No new-state exchange and no state / bond bits packed into the label word (Fig. 2): the new state of
//     a cluster is drawn from the Philox key of its canonical root, the smallest GLOBAL site index, so every piece
//     computes it on its own.  Label values are global site indices; with N = L^2 <= 2^32 they fit the paper's 32-bit
//     `label`, and the (owner, local offset) pair of its 64-bit `label_total_lattice` is what
//     SuperGeo::locate() computes from a label value whenever a link is followed into another piece.
//   * After stage 2 a RESOLVE pass over the boundary sites re-points every link that leaves a piece at the canonical
//     root ("the update of label_total_lattice for the whole sub-lattice", reduced to the boundary
//     components), so the flatten + flip kernel of a piece never reads another piece's memory: its root chases end at a
//     root or at the first link that leaves the piece.
// The result is bit-identical to the single-lattice path and to the CPU oracle (tests/test_super_gpu.py): the same
// bonds, canonical labels, spins and observables.
//
// This file (compiled as part of sw_api.cu, one translation unit) drives all pieces from ONE process (streams + events; pieces may share a device, which is how the
// path is verified on a single B200).  One process per GPU is the same launch sequence with the three event waits
// replaced by a barrier of the process group and the peer pointers opened through CUDA IPC.
#pragma once

#include "../../include/sw.h"

#include <algorithm>
#include <cstdio>
#include <new>
#include <string>
#include <vector>

#include "sw_host.h"
#include "sw_common.cuh"
#include "sw_generic.cuh"
#include "sw_observe.cuh"
#include "sw_tiled.cuh"
#include "sw_tile_blocks.cuh"

namespace sw {

constexpr int kMaxPieces = 64;

// every piece's label array and edge records, by owner id (kernel parameter; peer pointers where the devices differ)
struct SuperGeo {
    uint32_t Lg, log2Lg, gx, gy, W, H;
    uint32_t *labels[kMaxPieces];
    const TileEdges *edges[kMaxPieces];
    uint32_t *sizes[kMaxPieces];            // cluster-size scratch (sw_super_measure of the largest cluster)

    // label value (global site index) -> (owner, local offset): the pair PAPER.md:64 keeps in label_total_lattice
    __device__ __forceinline__ void locate(uint32_t g, uint32_t &owner, uint32_t &off) const
    {
        uint32_t x, y;
        if (log2Lg != 0xFFFFFFFFu) { y = g >> log2Lg; x = g & (Lg - 1u); } else { y = g / Lg; x = g - y * Lg; }
        const uint32_t px = x / W, py = y / H;
        owner = py * gx + px;
        off = (y - py * H) * W + (x - px * W);
    }
    __device__ __forceinline__ uint32_t *entry(uint32_t g) const
    {
        uint32_t o, off;
        locate(g, o, off);
        return labels[o] + off;
    }
    __device__ __forceinline__ uint32_t load(uint32_t g) const { return __ldcg(entry(g)); }
    // read-only find: stage 2 never re-points a link on the way (only roots are hooked), so that afterwards the
    // links that leave a piece sit exactly at the hooked roots of boundary components (what the resolve pass relies on)
    __device__ __forceinline__ uint32_t find(uint32_t a, uint32_t &hops) const
    {
        uint32_t p = load(a);
        ++hops;
        while (p != a) { a = p; p = load(a); ++hops; }
        return a;
    }
};

struct SuperCounters {
    unsigned long long links;       // active bonds between pieces that were united (after the duplicate filter)
    unsigned long long hops;        // label loads of stage 2 (finds of the merge and of the resolve pass), local or peer
    unsigned long long retries;     // hooks that lost the race for a root
    unsigned long long resolved;    // links that leave their piece, re-pointed at the canonical root
};

__global__ void k_init_random_super(uint8_t *__restrict__ spins, Params P, Dom dom)
{
    const uint64_t total = (uint64_t)dom.W * dom.H, stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += stride) {
        const uint32_t ly = (uint32_t)(i / dom.W), lx = (uint32_t)(i - (uint64_t)ly * dom.W);
        const uint32_t g = (dom.oy + ly) * dom.Lg + dom.ox + lx;
        spins[i] = (uint8_t)state_from_draw(philox4x32_10(g, 0u, 0u, kPurposeInit, P).x, P.q);
    }
}

// ---- stage 2: unite across the borders between pieces --------------------------------------------
// One thread per site of the right column (H of them) and of the bottom row (W) of piece `me`; the partner is the
// left column of the piece on the right / the top row of the piece below (periodic in the super-lattice).
__global__ void __launch_bounds__(128)
k_super_merge(SuperGeo geo, uint32_t me, uint32_t right, uint32_t down, const TileBorder *__restrict__ border, SuperCounters *counters)
{
    const uint32_t tiles_x = geo.W >> 6, tiles_y = geo.H >> 6;
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31u;
    bool on = false;
    uint32_t u = 0, v = 0;
    if (p < geo.H) {                                         // right column, row p
        const uint32_t ty = p >> 6, k = p & 63u, tile = ty * tiles_x + tiles_x - 1u;
        on = (border[tile].right_col >> k) & 1ull;
        if (on) { u = geo.edges[me][tile].right[k]; v = __ldcg(&geo.edges[right][ty * tiles_x].left[k]); }
    } else if (p < geo.H + geo.W) {                          // bottom row, column p - H
        const uint32_t x = p - geo.H, tx = x >> 6, k = x & 63u, tile = (tiles_y - 1u) * tiles_x + tx;
        on = (border[tile].bottom_row >> k) & 1ull;
        if (on) { u = geo.edges[me][tile].bottom[k]; v = __ldcg(&geo.edges[down][tx].top[k]); }
    }
    // the previous boundary bond joins the same two tile-local components: nothing new
    const uint32_t pu = __shfl_up_sync(0xFFFFFFFFu, u, 1), pv = __shfl_up_sync(0xFFFFFFFFu, v, 1);
    const bool pon = __shfl_up_sync(0xFFFFFFFFu, (uint32_t)on, 1) != 0;
    if (lane != 0 && pon && pu == u && pv == v) on = false;
    uint32_t hops = 0, lost = 0;
    if (on) {
        uint32_t a = geo.find(u, hops), b = geo.find(v, hops);
        while (a != b) {
            if (a < b) { const uint32_t s = a; a = b; b = s; }
            const uint32_t old = atomicMin_system(geo.entry(a), b);      // the larger root goes under the smaller; the word lives in its owner's memory
            if (old == a) break;
            ++lost;
            a = geo.find(old, hops);
            b = geo.find(b, hops);
        }
    }
    const uint32_t n_on = __popc(__ballot_sync(0xFFFFFFFFu, on));
    hops = __reduce_add_sync(0xFFFFFFFFu, hops);
    lost = __reduce_add_sync(0xFFFFFFFFu, lost);
    if (lane == 0 && (n_on | hops)) {
        atomicAdd(&counters->links, (unsigned long long)n_on);
        atomicAdd(&counters->hops, (unsigned long long)hops);
        atomicAdd(&counters->retries, (unsigned long long)lost);
    }
}

// ---- resolve: every link that leaves piece `me` is re-pointed at the canonical root ------------------------------------
// One thread per boundary site (left and right column, top and bottom row).  From the site's tile-local root the local
// links are followed to the last node inside the piece; if its link leaves the piece, the canonical root is found through
// the other pieces (read-only) and written there.  Links that leave a piece only exist at roots stage 2 hooked, and
// every such root belongs to a component that touches the boundary, so all of them are reached.
__global__ void __launch_bounds__(128)
k_super_resolve(SuperGeo geo, Dom dom, SuperCounters *counters)
{
    const uint32_t tiles_x = geo.W >> 6, tiles_y = geo.H >> 6, me = dom.me;
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31u;
    uint32_t hops = 0, done = 0;
    if (p < 2u * (geo.H + geo.W)) {
        uint32_t a;
        const TileEdges *e = geo.edges[me];
        if (p < geo.H) a = e[(p >> 6) * tiles_x].left[p & 63u];
        else if (p < 2u * geo.H) { const uint32_t y = p - geo.H; a = e[(y >> 6) * tiles_x + tiles_x - 1u].right[y & 63u]; }
        else if (p < 2u * geo.H + geo.W) { const uint32_t x = p - 2u * geo.H; a = e[x >> 6].top[x & 63u]; }
        else { const uint32_t x = p - 2u * geo.H - geo.W; a = e[(tiles_y - 1u) * tiles_x + (x >> 6)].bottom[x & 63u]; }
        const DomAddr addr(dom);
        uint32_t *mine = geo.labels[me];
        uint32_t q = __ldcg(mine + addr(a));
        ++hops;
        while (q != a && addr.mine(q)) { a = q; q = __ldcg(mine + addr(a)); ++hops; }
        if (q != a) {                                        // the link of `a` leaves the piece
            const uint32_t root = geo.find(q, hops);
            if (root != q) { atomicMin(mine + addr(a), root); done = 1; }
        }
    }
    hops = __reduce_add_sync(0xFFFFFFFFu, hops);
    done = __reduce_add_sync(0xFFFFFFFFu, done);
    if (lane == 0 && (hops | done)) {
        atomicAdd(&counters->hops, (unsigned long long)hops);
        atomicAdd(&counters->resolved, (unsigned long long)done);
    }
}

// ---- observables of one piece (a6): equal pairs with the neighbours across the piece border, state histogram ------------
__global__ void __launch_bounds__(kObsThreads)
k_super_observe(const uint8_t *__restrict__ spins, Params P, Dom dom, uint32_t want, unsigned long long *row)
{
    __shared__ unsigned int s_hist[256];
    __shared__ unsigned long long s_scratch[kObsThreads / 32];
    for (int k = threadIdx.x; k < 256; k += blockDim.x) s_hist[k] = 0;
    __syncthreads();
    const uint64_t total = (uint64_t)dom.W * dom.H, stride = (uint64_t)gridDim.x * blockDim.x;
    unsigned long long e = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += stride) {
        const uint32_t ly = (uint32_t)(i / dom.W), lx = (uint32_t)(i - (uint64_t)ly * dom.W);
        const uint8_t s = spins[i];
        if (want & 1u) {
            const uint8_t r = (lx + 1u < dom.W) ? spins[i + 1] : __ldcg(dom.right + (uint64_t)ly * dom.right_W);
            const uint8_t d = (ly + 1u < dom.H) ? spins[i + dom.W] : __ldcg(dom.down + lx);
            e += (s == r) + (s == d);
        }
        if (want & 2u) atomicAdd(&s_hist[s], 1u);
    }
    __syncthreads();
    if (want & 2u)
        for (int k = threadIdx.x; k < (int)P.q; k += blockDim.x)
            if (s_hist[k]) atomicAdd(row + 3 + k, (unsigned long long)s_hist[k]);
    if (want & 1u) block_add_u64(e, row + 0, s_scratch);
}

// sizes[owner(root)][offset(root)] += members, run-length aggregated along the rows of the piece (labels are canonical)
__global__ void k_super_sizes(SuperGeo geo, uint32_t me)
{
    const uint64_t n_groups = ((uint64_t)geo.W * geo.H) >> 4, stride = (uint64_t)gridDim.x * blockDim.x;
    const uint32_t *labels = geo.labels[me];
    for (uint64_t g = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; g < n_groups; g += stride) {
        uint32_t cur = 0, run = 0;
        const uint4 *lp = reinterpret_cast<const uint4 *>(labels + (g << 4));
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint4 l = lp[k];
            const uint32_t lab[4] = {l.x, l.y, l.z, l.w};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (run && lab[j] == cur) { ++run; continue; }
                if (run) { uint32_t o, off; geo.locate(cur, o, off); atomicAdd_system(geo.sizes[o] + off, run); }
                cur = lab[j]; run = 1;
            }
        }
        if (run) { uint32_t o, off; geo.locate(cur, o, off); atomicAdd_system(geo.sizes[o] + off, run); }
    }
}

}  // namespace sw

// ------------------------------------------------------------------------------------------------ host side

namespace {

using sw::Dom;
using sw::Params;

struct Piece {
    bool local = true;              // false: another process owns it; only the peer pointers (opened through CUDA IPC) are known
    void *ipc_base = nullptr;       // what cudaIpcOpenMemHandle returned for a remote piece
    int device = 0;
    uint32_t px = 0, py = 0;
    cudaStream_t stream = nullptr;
    cudaEvent_t ev_stage1 = nullptr, ev_stage2 = nullptr, ev_flip = nullptr;
    uint8_t *ws = nullptr;
    size_t ws_bytes = 0;
    uint8_t *spins = nullptr, *stage = nullptr;
    uint32_t *bonds = nullptr, *labels = nullptr, *tile_clusters = nullptr, *flag = nullptr, *sizes = nullptr;
    uint16_t *rootbits = nullptr;
    sw::TileBorder *border = nullptr;
    sw::TileEdges *edges = nullptr;
    uint2 *draws = nullptr;
    unsigned long long *row = nullptr;
    sw::SuperCounters *counters = nullptr;
    size_t stage_bytes = 0;
    Dom dom{};
};

}  // namespace

struct sw_super {
    uint32_t L = 0, q = 0, gx = 0, gy = 0, W = 0, H = 0;
    uint64_t N = 0, seed = 0, T = 0, t = 0, draws_t = ~0ull;
    double K = 0;
    bool have_spins = false, have_labels = false;
    int rank_piece = -1;            // >= 0: one process per GPU, this process owns that piece only (sw_create_super_rank)
    uint64_t launches = 0, sweeps = 0;
    std::vector<Piece> pieces;
    sw::SuperGeo geo{};
    std::string err;
};

namespace {

int sfail(sw_super *s, int code, const char *what)
{
    if (s) s->err = what;
    return code;
}

int scuda(sw_super *s, cudaError_t e, const char *what)
{
    if (s) s->err = std::string(what) + ": " + cudaGetErrorString(e);
    return SW_ERR_CUDA;
}

#define SS_CUDA(s, call)                                          \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return scuda((s), e_, #call);      \
    } while (0)

struct DevSwitch {
    int prev = -1;
    DevSwitch() { cudaGetDevice(&prev); }
    void to(int d) { cudaSetDevice(d); }
    ~DevSwitch() { if (prev >= 0) cudaSetDevice(prev); }
};

Params piece_params(const sw_super *s, uint64_t t)
{
    // P.L is the global size (the generic helpers that look at it are not used on pieces); P.N = sites of one piece
    return swh::make_params(s->L, s->q, (uint64_t)s->W * s->H, s->seed, s->T, t);
}

uint32_t right_of(const sw_super *s, uint32_t d) { const uint32_t px = d % s->gx, py = d / s->gx; return py * s->gx + (px + 1) % s->gx; }
uint32_t down_of(const sw_super *s, uint32_t d) { const uint32_t px = d % s->gx, py = d / s->gx; return ((py + 1) % s->gy) * s->gx + px; }

int grid_cap(uint64_t items, int threads) { return (int)std::max<uint64_t>(1, std::min<uint64_t>((items + threads - 1) / threads, 148 * 16)); }

// byte offsets of a piece's arrays inside its one allocation: the same for every piece, so a process that opened
// another piece's allocation through CUDA IPC knows where its spins, labels and edge records are
struct PieceLayout { size_t spins, bonds, labels, rootbits, border, edges, tc, draws, row, flag, cnt, stage, stage_bytes, sizes, total; };

PieceLayout piece_layout(const sw_super *s)
{
    const uint64_t Np = (uint64_t)s->W * s->H, tiles = Np / sw::kTileSites;
    PieceLayout o{};
    size_t off = 0;
    auto carve = [&](size_t bytes) { const size_t at = off; off = swh::align_up(off + bytes); return at; };
    o.spins = carve(Np); o.bonds = carve((Np / 16) * 4); o.labels = carve(Np * 4); o.rootbits = carve((Np / 16) * 2);
    o.border = carve(tiles * sizeof(sw::TileBorder)); o.edges = carve(tiles * sizeof(sw::TileEdges));
    o.tc = carve(tiles * (sw::kFlipThreads / 32) * 4); o.draws = carve((Np / 32) * sizeof(uint2));
    o.row = carve((3 + (size_t)s->q) * 8); o.flag = carve(4); o.cnt = carve(sizeof(sw::SuperCounters));
    o.stage_bytes = (size_t)std::min<uint64_t>(Np, std::max<uint64_t>(s->W, 32ull << 20));
    o.stage = carve(o.stage_bytes);
    o.sizes = carve(Np * 4);                                 // cluster-size scratch: other pieces add to it (sw_super_measure of the largest cluster)
    o.total = off;
    return o;
}

void set_piece_pointers(Piece &p, uint8_t *base, const PieceLayout &o)
{
    p.ws = base; p.ws_bytes = o.total; p.stage_bytes = o.stage_bytes;
    p.spins = base + o.spins; p.bonds = (uint32_t *)(base + o.bonds); p.labels = (uint32_t *)(base + o.labels);
    p.rootbits = (uint16_t *)(base + o.rootbits); p.border = (sw::TileBorder *)(base + o.border); p.edges = (sw::TileEdges *)(base + o.edges);
    p.tile_clusters = (uint32_t *)(base + o.tc); p.draws = (uint2 *)(base + o.draws); p.row = (unsigned long long *)(base + o.row);
    p.flag = (uint32_t *)(base + o.flag); p.counters = (sw::SuperCounters *)(base + o.cnt); p.stage = base + o.stage;
    p.sizes = (uint32_t *)(base + o.sizes);
}

// (re)build the tables the kernels take by value: every piece's labels / edge records / size scratch, the neighbours' spins
void refresh_geo(sw_super *s)
{
    const uint32_t n = (uint32_t)s->pieces.size();
    s->geo.Lg = s->L; s->geo.log2Lg = swh::log2_exact(s->L); s->geo.gx = s->gx; s->geo.gy = s->gy; s->geo.W = s->W; s->geo.H = s->H;
    for (uint32_t d = 0; d < n; ++d) {
        Piece &p = s->pieces[d];
        s->geo.labels[d] = p.labels; s->geo.edges[d] = p.edges; s->geo.sizes[d] = p.sizes;
        const Piece &r = s->pieces[right_of(s, d)], &dn = s->pieces[down_of(s, d)];
        p.dom.W = s->W; p.dom.H = s->H; p.dom.Lg = s->L; p.dom.log2Lg = s->geo.log2Lg;
        p.dom.ox = p.px * s->W; p.dom.oy = p.py * s->H;
        p.dom.right = r.spins; p.dom.down = dn.spins; p.dom.right_W = s->W; p.dom.me = d;
    }
}

// why the last sw_create_super / sw_create_super_rank of this thread failed (there is no context to hold the text then)
thread_local const char *g_create_err = "";

// rank mode: unmap the pieces of the other processes (their pointers are dead afterwards)
void close_imported(sw_super *s)
{
    for (auto &p : s->pieces) {
        if (p.local || !p.ipc_base) continue;
        cudaIpcCloseMemHandle(p.ipc_base);
        p.ipc_base = nullptr;
        p.ws = nullptr; p.spins = nullptr; p.labels = nullptr; p.edges = nullptr; p.sizes = nullptr;
    }
}

void destroy_pieces(sw_super *s)
{
    DevSwitch sw_;
    for (auto &p : s->pieces) if (p.local && p.stream) { sw_.to(p.device); cudaStreamSynchronize(p.stream); }   // nothing of mine still reads a peer
    close_imported(s);
    for (auto &p : s->pieces) {
        if (!p.local) continue;
        sw_.to(p.device);
        if (p.stream) cudaStreamSynchronize(p.stream);
        if (p.ws) cudaFree(p.ws);
        if (p.ev_stage1) cudaEventDestroy(p.ev_stage1);
        if (p.ev_stage2) cudaEventDestroy(p.ev_stage2);
        if (p.ev_flip) cudaEventDestroy(p.ev_flip);
        if (p.stream) cudaStreamDestroy(p.stream);
    }
    s->pieces.clear();
}

// The three phases of a sweep.  In one process (all pieces local) they are ordered by events: a phase of a piece waits for
// the previous phase of EVERY piece.  With one process per GPU (rank mode) the caller puts a barrier of the process group
// between the phases (after sw_super_synchronize) and the event waits fall away.
//   phase 0  stage 1: bonds + tile-local labels + tile-border merge inside the piece
//   phase 1  stage 2: union over the bonds between pieces (boundary sites only)
//   phase 2  resolve, flatten to the canonical root, flip
int super_phase(sw_super *s, int phase, bool count_clusters)
{
    DevSwitch sw_;
    const Params P = piece_params(s, s->t);
    const uint32_t n = (uint32_t)s->pieces.size();
    const dim3 tgrid(s->W / sw::kTile, s->H / sw::kTile);
    const uint32_t tiles = tgrid.x * tgrid.y;
    for (uint32_t d = 0; d < n; ++d) {
        Piece &p = s->pieces[d];
        if (!p.local) continue;
        sw_.to(p.device);
        for (uint32_t o = 0; o < n; ++o) {
            const Piece &other = s->pieces[o];
            if (o == d || !other.local) continue;
            // phase 0 waits for every piece's last flip: the neighbours' new spins must be written, and nobody may still be
            // following links into my labels of the last sweep (the resolve pass of ANY piece can)
            SS_CUDA(s, cudaStreamWaitEvent(p.stream, phase == 0 ? other.ev_flip : phase == 1 ? other.ev_stage1 : other.ev_stage2, 0));
        }
        if (phase == 0) {
            if (s->draws_t != s->t) { sw::k_draws_super<<<tgrid, 256, 0, p.stream>>>(p.draws, P, p.dom); s->launches += 1; }
            sw::k_tile_blocks_super<<<tgrid, sw::kBlkThreads, 0, p.stream>>>(p.spins, p.bonds, p.labels, p.rootbits, p.border, p.edges, p.draws, P, p.dom);
            const unsigned per = (unsigned)sw::merge_tiles_per_cta(tiles);
            auto merge = per == 2 ? sw::k_tile_merge_super<2> : sw::k_tile_merge_super<4>;
            merge<<<(tiles + per - 1) / per, sw::kMergeThreads, 0, p.stream>>>(p.labels, p.border, p.edges, P, p.dom, tiles);
            SS_CUDA(s, cudaEventRecord(p.ev_stage1, p.stream));
            s->launches += 2;
        } else if (phase == 1) {
            sw::k_super_merge<<<(s->W + s->H + 127) / 128, 128, 0, p.stream>>>(s->geo, d, right_of(s, d), down_of(s, d), p.border, p.counters);
            SS_CUDA(s, cudaEventRecord(p.ev_stage2, p.stream));
            s->launches += 1;
        } else {
            sw::k_super_resolve<<<(2 * (s->W + s->H) + 127) / 128, 128, 0, p.stream>>>(s->geo, p.dom, p.counters);
            auto flip = count_clusters ? sw::k_tile_flip_super<true, true, true> : sw::k_tile_flip_super<true, true, false>;
            flip<<<tgrid, sw::kFlipThreads, 0, p.stream>>>(p.labels, p.rootbits, p.spins, P, p.dom, p.tile_clusters, p.draws);
            SS_CUDA(s, cudaEventRecord(p.ev_flip, p.stream));
            s->launches += 2;
        }
    }
    SS_CUDA(s, cudaGetLastError());
    if (phase == 2) {
        s->draws_t = s->t + 1;
        s->t += 1; s->sweeps += 1;
        s->have_labels = true;
    }
    return SW_OK;
}

int super_sweep_once(sw_super *s, bool count_clusters)
{
    for (int phase = 0; phase < 3; ++phase) {
        const int rc = super_phase(s, phase, count_clusters);
        if (rc != SW_OK) return rc;
    }
    return SW_OK;
}

int sync_all(sw_super *s)
{
    DevSwitch sw_;
    for (auto &p : s->pieces) { if (!p.local) continue; sw_.to(p.device); SS_CUDA(s, cudaStreamSynchronize(p.stream)); }
    return SW_OK;
}

// after a host-side change of all spins: the next tile kernels must see it
int mark_spins_ready(sw_super *s)
{
    DevSwitch sw_;
    for (auto &p : s->pieces) { if (!p.local) continue; sw_.to(p.device); SS_CUDA(s, cudaEventRecord(p.ev_flip, p.stream)); }
    return SW_OK;
}

}  // namespace

extern "C" {

static int create_super_common(sw_super **out, uint32_t L, uint32_t q, double K, uint64_t seed, uint32_t gx, uint32_t gy,
                               const int *devices, int rank_piece)
{
    if (!out) return SW_ERR_INVALID_ARG;
    *out = nullptr;
    g_create_err = "";
    uint64_t T = 0;
    if (L < 64 || L > 65536 || q < 2 || q > 255 || !swh::host_threshold(K, &T)) return SW_ERR_INVALID_ARG;
    if (gx < 1 || gy < 1 || gx * gy > (uint32_t)sw::kMaxPieces || L % (gx * sw::kTile) || L % (gy * sw::kTile)) return SW_ERR_INVALID_ARG;
    if (rank_piece >= (int)(gx * gy)) return SW_ERR_INVALID_ARG;
    sw_super *s = new (std::nothrow) sw_super();
    if (!s) return SW_ERR_OOM;
    s->L = L; s->q = q; s->K = K; s->seed = seed; s->T = T; s->gx = gx; s->gy = gy;
    s->W = L / gx; s->H = L / gy; s->N = (uint64_t)L * L;
    s->rank_piece = rank_piece;
    const uint32_t n = gx * gy;
    const PieceLayout lay = piece_layout(s);
    DevSwitch sw_;
    int cur = 0, count = 0;
    if (cudaGetDevice(&cur) != cudaSuccess || cudaGetDeviceCount(&count) != cudaSuccess) { delete s; return SW_ERR_CUDA; }
    s->pieces.resize(n);
    int rc = SW_OK;
    for (uint32_t d = 0; d < n && rc == SW_OK; ++d) {
        Piece &p = s->pieces[d];
        p.px = d % gx; p.py = d / gx;
        p.local = rank_piece < 0 || (int)d == rank_piece;
        if (!p.local) continue;                              // its pointers arrive through sw_super_ipc_import
        p.device = (devices && rank_piece < 0) ? devices[d] : cur;
        if (p.device < 0 || p.device >= count) { rc = SW_ERR_INVALID_ARG; break; }
        sw_.to(p.device);
        uint8_t *base = nullptr;
        if (cudaMalloc(&base, lay.total) != cudaSuccess) { cudaGetLastError(); rc = SW_ERR_OOM; break; }
        set_piece_pointers(p, base, lay);
        if (cudaStreamCreateWithFlags(&p.stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&p.ev_stage1, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&p.ev_stage2, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&p.ev_flip, cudaEventDisableTiming) != cudaSuccess ||
            cudaMemsetAsync(p.counters, 0, sizeof(sw::SuperCounters), p.stream) != cudaSuccess) { cudaGetLastError(); rc = SW_ERR_CUDA; break; }
    }
    // peer access between the devices in use (NVLink P2P); pieces on one device need none
    for (uint32_t a = 0; a < n && rc == SW_OK && rank_piece < 0; ++a)
        for (uint32_t b = 0; b < n && rc == SW_OK; ++b) {
            const int da = s->pieces[a].device, db = s->pieces[b].device;
            if (da == db) continue;
            int can = 0, native_atomics = 0;
            cudaDeviceCanAccessPeer(&can, da, db);
            if (!can) { g_create_err = "sw_create_super: two of the devices have no peer access to each other"; rc = SW_ERR_CUDA; break; }
            // stage 2 and the size count hook roots with atomicMin_system / atomicAdd_system in the owner's memory: over a link
            // without native atomics (PCIe-only P2P) those are not atomic and labels or sizes would be silently wrong
            if (cudaDeviceGetP2PAttribute(&native_atomics, cudaDevP2PAttrNativeAtomicSupported, da, db) != cudaSuccess) { cudaGetLastError(); native_atomics = 0; }
            if (!native_atomics) {
                g_create_err = "sw_create_super: the link between two of the devices has no native atomics (cudaDevP2PAttrNativeAtomicSupported = 0; "
                               "NVLink is needed): the inter-piece union-find cannot run over it";
                rc = SW_ERR_CUDA; break;
            }
            sw_.to(da);
            const cudaError_t e = cudaDeviceEnablePeerAccess(db, 0);
            if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) rc = SW_ERR_CUDA;
            cudaGetLastError();
        }
    if (rc != SW_OK) { destroy_pieces(s); delete s; return rc; }
    refresh_geo(s);
    *out = s;
    return SW_OK;
}

int sw_create_super(sw_super **out, uint32_t L, uint32_t q, double K, uint64_t seed, uint32_t gx, uint32_t gy, const int *devices)
{
    return create_super_common(out, L, q, K, seed, gx, gy, devices, -1);
}

int sw_create_super_rank(sw_super **out, uint32_t L, uint32_t q, double K, uint64_t seed, uint32_t gx, uint32_t gy, uint32_t my_piece)
{
    if (my_piece >= gx * gy) return SW_ERR_INVALID_ARG;
    return create_super_common(out, L, q, K, seed, gx, gy, nullptr, (int)my_piece);
}

int sw_super_ipc_export(sw_super *s, void *handle_out)
{
    if (!s || !handle_out || s->rank_piece < 0) return sfail(s, SW_ERR_INVALID_ARG, "sw_super_ipc_export: not a rank context");
    static_assert(sizeof(cudaIpcMemHandle_t) == SW_IPC_HANDLE_BYTES, "handle size");
    DevSwitch sw_;
    Piece &p = s->pieces[s->rank_piece];
    sw_.to(p.device);
    SS_CUDA(s, cudaIpcGetMemHandle((cudaIpcMemHandle_t *)handle_out, p.ws));
    return SW_OK;
}

int sw_super_ipc_import(sw_super *s, uint32_t piece, const void *handle)
{
    if (!s || !handle || s->rank_piece < 0 || piece >= s->pieces.size() || (int)piece == s->rank_piece)
        return sfail(s, SW_ERR_INVALID_ARG, "sw_super_ipc_import: bad argument");
    Piece &p = s->pieces[piece];
    if (p.ipc_base) return sfail(s, SW_ERR_STATE, "sw_super_ipc_import: piece already imported");
    DevSwitch sw_;
    sw_.to(s->pieces[s->rank_piece].device);
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, sizeof(h));
    void *base = nullptr;
    SS_CUDA(s, cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess));
    p.ipc_base = base;
    set_piece_pointers(p, (uint8_t *)base, piece_layout(s));
    refresh_geo(s);
    return SW_OK;
}

int sw_super_phase(sw_super *s, int phase)
{
    if (!s || phase < 0 || phase > 2) return SW_ERR_INVALID_ARG;
    if (!s->have_spins) return sfail(s, SW_ERR_STATE, "sw_super_phase: no spins");
    if (s->t + 1 > 0x100000000ull) return sfail(s, SW_ERR_STATE, "sw_super_phase: sweep counter would pass 2^32");
    for (auto &p : s->pieces) if (!p.spins) return sfail(s, SW_ERR_STATE, "sw_super_phase: a piece has not been imported");
    return super_phase(s, phase, true);
}

void sw_super_destroy(sw_super *s)
{
    if (!s) return;
    destroy_pieces(s);
    delete s;
}

int sw_super_init(sw_super *s, int mode)
{
    if (!s) return SW_ERR_INVALID_ARG;
    if (mode != SW_INIT_ORDERED && mode != SW_INIT_RANDOM) return sfail(s, SW_ERR_INVALID_ARG, "sw_super_init: unknown mode");
    DevSwitch sw_;
    const Params P = piece_params(s, 0);
    for (auto &p : s->pieces) {
        if (!p.local) continue;
        sw_.to(p.device);
        if (mode == SW_INIT_ORDERED) SS_CUDA(s, cudaMemsetAsync(p.spins, 0, (size_t)s->W * s->H, p.stream));
        else { sw::k_init_random_super<<<grid_cap((uint64_t)s->W * s->H, 256), 256, 0, p.stream>>>(p.spins, P, p.dom); s->launches += 1; }
    }
    SS_CUDA(s, cudaGetLastError());
    s->t = 0; s->have_spins = true; s->have_labels = false;
    return mark_spins_ready(s);
}

int sw_super_set_state(sw_super *s, const uint8_t *src, uint64_t t)
{
    if (!s || !src || t > 0xFFFFFFFFull) return sfail(s, SW_ERR_INVALID_ARG, "sw_super_set_state: bad argument");
    DevSwitch sw_;
    Params P = piece_params(s, 0);
    for (auto &p : s->pieces) {
        if (!p.local) continue;
        sw_.to(p.device);
        const uint8_t *from = src + (uint64_t)p.dom.oy * s->L + p.dom.ox;
        SS_CUDA(s, cudaMemcpy2DAsync(p.spins, s->W, from, s->L, s->W, s->H, cudaMemcpyHostToDevice, p.stream));
        SS_CUDA(s, cudaMemsetAsync(p.flag, 0, 4, p.stream));
        sw::k_validate_spins<<<grid_cap(P.N, 256), 256, 0, p.stream>>>(p.spins, P, p.flag);
        s->launches += 1;
    }
    bool bad = false;
    for (auto &p : s->pieces) {
        if (!p.local) continue;
        sw_.to(p.device);
        uint32_t f = 0;
        SS_CUDA(s, cudaMemcpyAsync(&f, p.flag, 4, cudaMemcpyDeviceToHost, p.stream));
        SS_CUDA(s, cudaStreamSynchronize(p.stream));
        bad |= f != 0;
    }
    s->have_labels = false;
    if (bad) { s->have_spins = false; return sfail(s, SW_ERR_INVALID_ARG, "sw_super_set_state: spin value >= q"); }
    s->t = t; s->have_spins = true;
    return mark_spins_ready(s);
}

int sw_super_sweep(sw_super *s, uint64_t n)
{
    if (!s) return SW_ERR_INVALID_ARG;
    if (s->rank_piece >= 0) return sfail(s, SW_ERR_STATE, "sw_super_sweep: one process per GPU: drive the sweep with sw_super_phase and a barrier between the phases");
    if (!s->have_spins) return sfail(s, SW_ERR_STATE, "sw_super_sweep: no spins (call sw_super_init or sw_super_set_state)");
    if (s->t + n > 0x100000000ull) return sfail(s, SW_ERR_STATE, "sw_super_sweep: sweep counter would pass 2^32");
    for (uint64_t k = 0; k < n; ++k) {
        const int rc = super_sweep_once(s, k + 1 == n);
        if (rc != SW_OK) return rc;
    }
    return SW_OK;
}

// The three phases of a measurement, over the local pieces (a barrier between them in rank mode, a sync here otherwise):
//   0  zero the rows and, for the largest cluster, the size counters
//   1  equal pairs + histogram, cluster count, sizes[owner(root)] += members (into other pieces' memory too)
//   2  maximum of the local size counters; the local partial row comes back in `part` (sum columns; column 2 is a maximum)
static int measure_phase(sw_super *s, int phase, uint32_t what, uint64_t *part)
{
    DevSwitch sw_;
    const Params P = piece_params(s, s->t);
    const uint64_t Np = (uint64_t)s->W * s->H;
    const uint32_t n = (uint32_t)s->pieces.size();
    const bool cl = s->have_labels && (what & (SW_OBS_CLUSTERS | SW_OBS_LARGEST)), big = s->have_labels && (what & SW_OBS_LARGEST);
    const uint32_t want = what & 3u;
    const size_t cols = 3 + (size_t)s->q;
    if (phase == 2 && part) for (size_t k = 0; k < cols; ++k) part[k] = 0;
    for (uint32_t d = 0; d < n; ++d) {
        Piece &p = s->pieces[d];
        if (!p.local) continue;
        sw_.to(p.device);
        if (phase == 0) {
            SS_CUDA(s, cudaMemsetAsync(p.row, 0, cols * 8, p.stream));
            if (big) SS_CUDA(s, cudaMemsetAsync(p.sizes, 0, Np * 4, p.stream));
        } else if (phase == 1) {
            if (want) { sw::k_super_observe<<<grid_cap(Np, sw::kObsThreads), sw::kObsThreads, 0, p.stream>>>(p.spins, P, p.dom, want, p.row); s->launches += 1; }
            if (cl) {
                const uint32_t entries = (uint32_t)(Np / sw::kTileSites) * (sw::kFlipThreads / 32);
                sw::k_sum_tile_clusters<<<grid_cap(entries, sw::kObsThreads), sw::kObsThreads, 0, p.stream>>>(p.tile_clusters, entries, p.row);
                s->launches += 1;
            }
            if (big) { sw::k_super_sizes<<<grid_cap(Np / 16, 256), 256, 0, p.stream>>>(s->geo, d); s->launches += 1; }
        } else {
            if (big) { sw::k_max_size<<<grid_cap(Np, 256), 256, 0, p.stream>>>(p.sizes, P, p.row); s->launches += 1; }
            std::vector<uint64_t> row(cols);
            SS_CUDA(s, cudaMemcpyAsync(row.data(), p.row, cols * 8, cudaMemcpyDeviceToHost, p.stream));
            SS_CUDA(s, cudaStreamSynchronize(p.stream));
            if (part) for (size_t k = 0; k < cols; ++k) part[k] = (k == 2) ? std::max(part[k], row[k]) : part[k] + row[k];
        }
    }
    SS_CUDA(s, cudaGetLastError());
    return sync_all(s);
}

int sw_super_measure_phase(sw_super *s, int phase, uint32_t what, uint64_t *part)
{
    if (!s || phase < 0 || phase > 2 || (what & ~(uint32_t)SW_OBS_ALL) || (phase == 2 && !part)) return SW_ERR_INVALID_ARG;
    if (!s->have_spins) return sfail(s, SW_ERR_STATE, "sw_super_measure_phase: no spins");
    for (auto &p : s->pieces) if (!p.spins) return sfail(s, SW_ERR_STATE, "sw_super_measure_phase: a piece has not been imported");
    return measure_phase(s, phase, what, part);
}

int sw_super_measure(sw_super *s, uint64_t *energy_bonds, uint64_t *mag_counts, uint64_t *n_clusters, uint64_t *largest_cluster)
{
    if (!s) return SW_ERR_INVALID_ARG;
    if (s->rank_piece >= 0) return sfail(s, SW_ERR_STATE, "sw_super_measure: one process per GPU: use sw_super_measure_phase with a barrier between the phases");
    if (!s->have_spins) return sfail(s, SW_ERR_STATE, "sw_super_measure: no spins");
    const uint32_t what = (energy_bonds ? SW_OBS_ENERGY : 0u) | (mag_counts ? SW_OBS_MAG : 0u) | (n_clusters ? SW_OBS_CLUSTERS : 0u) |
                          (largest_cluster ? SW_OBS_LARGEST : 0u);
    std::vector<uint64_t> total(3 + s->q, 0);
    int rc = sync_all(s);                                     // the spins of all pieces are final
    for (int phase = 0; phase < 3 && rc == SW_OK; ++phase) rc = measure_phase(s, phase, what, total.data());
    if (rc != SW_OK) return rc;
    if (total[1] == 1) total[2] = s->N;                       // a uint32 size counter wraps only when one cluster holds 2^32 sites
    if (energy_bonds) *energy_bonds = total[0];
    if (n_clusters) *n_clusters = s->have_labels ? total[1] : 0;
    if (largest_cluster) *largest_cluster = s->have_labels ? total[2] : 0;
    if (mag_counts) for (uint32_t k = 0; k < s->q; ++k) mag_counts[k] = total[3 + k];
    return SW_OK;
}

static int super_get(sw_super *s, int what, void *dst)
{
    if (!s || !dst) return sfail(s, SW_ERR_INVALID_ARG, "sw_super_get: bad argument");
    if (what == 0 ? !s->have_spins : !s->have_labels) return sfail(s, SW_ERR_STATE, what == 0 ? "no spins" : "no sweep since sw_super_init");
    DevSwitch sw_;
    for (auto &p : s->pieces) {
        if (!p.local) continue;                              // rank mode: only my piece's part of dst is written
        sw_.to(p.device);
        const uint64_t first = (uint64_t)p.dom.oy * s->L + p.dom.ox;
        if (what == 0) {
            SS_CUDA(s, cudaMemcpy2DAsync((uint8_t *)dst + first, s->L, p.spins, s->W, s->W, s->H, cudaMemcpyDeviceToHost, p.stream));
        } else if (what == 1) {
            SS_CUDA(s, cudaMemcpy2DAsync((uint32_t *)dst + first, (size_t)s->L * 4, p.labels, (size_t)s->W * 4, (size_t)s->W * 4, s->H, cudaMemcpyDeviceToHost, p.stream));
        } else {
            const uint32_t rows_per = (uint32_t)std::max<uint64_t>(1, p.stage_bytes / s->W);
            for (uint32_t y = 0; y < s->H; y += rows_per) {
                const uint32_t nr = std::min(rows_per, s->H - y);
                sw::k_expand_bonds<<<grid_cap((uint64_t)nr * s->W, 256), 256, 0, p.stream>>>(p.bonds, p.stage, (uint64_t)y * s->W, (uint64_t)nr * s->W);
                s->launches += 1;
                SS_CUDA(s, cudaMemcpy2DAsync((uint8_t *)dst + first + (uint64_t)y * s->L, s->L, p.stage, s->W, s->W, nr, cudaMemcpyDeviceToHost, p.stream));
                SS_CUDA(s, cudaStreamSynchronize(p.stream));
            }
        }
    }
    return sync_all(s);
}

int sw_super_get_spins(sw_super *s, uint8_t *dst) { return super_get(s, 0, dst); }
int sw_super_get_labels(sw_super *s, uint32_t *dst) { return super_get(s, 1, dst); }
int sw_super_get_bonds(sw_super *s, uint8_t *dst) { return super_get(s, 2, dst); }

int sw_super_get_time(sw_super *s, uint64_t *t)
{
    if (!s || !t) return SW_ERR_INVALID_ARG;
    *t = s->t;
    return SW_OK;
}

int sw_super_synchronize(sw_super *s) { return s ? sync_all(s) : SW_ERR_INVALID_ARG; }

int sw_super_get_stats(sw_super *s, sw_super_stats *out)
{
    if (!s || !out) return SW_ERR_INVALID_ARG;
    DevSwitch sw_;
    *out = sw_super_stats{};
    out->gx = s->gx; out->gy = s->gy; out->piece_w = s->W; out->piece_h = s->H;
    out->sweeps = s->sweeps; out->kernel_launches = s->launches;
    out->boundary_sites_per_piece = 2ull * (s->W + s->H);
    std::vector<int> seen;
    for (auto &p : s->pieces) {
        if (!p.local) continue;
        sw_.to(p.device);
        sw::SuperCounters c;
        SS_CUDA(s, cudaMemcpyAsync(&c, p.counters, sizeof(c), cudaMemcpyDeviceToHost, p.stream));
        SS_CUDA(s, cudaStreamSynchronize(p.stream));
        out->inter_links += c.links; out->inter_hops += c.hops; out->inter_retries += c.retries; out->resolved_links += c.resolved;
        out->device_bytes += p.ws_bytes;
        if (std::find(seen.begin(), seen.end(), p.device) == seen.end()) seen.push_back(p.device);
    }
    out->devices = (uint32_t)seen.size();
    return SW_OK;
}

const char *sw_super_last_error(const sw_super *s) { return s ? s->err.c_str() : g_create_err; }

int sw_super_ipc_close_all(sw_super *s)
{
    if (!s || s->rank_piece < 0) return sfail(s, SW_ERR_INVALID_ARG, "sw_super_ipc_close_all: not a rank context");
    DevSwitch sw_;
    Piece &mine = s->pieces[s->rank_piece];
    sw_.to(mine.device);
    SS_CUDA(s, cudaStreamSynchronize(mine.stream));
    close_imported(s);
    s->have_spins = false;              // no phase can run any more: sw_super_phase refuses a context with a piece missing
    return SW_OK;
}

}  // extern "C"
