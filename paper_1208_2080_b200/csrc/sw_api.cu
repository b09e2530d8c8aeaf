// sw_api.cu -- host side of libsw.so: the context, memory plan, launch sequence and the C ABI of
// include/sw.h.  Every step of the sweep runs in the kernels of sw_tiled.cuh / sw_generic.cuh /
// sw_observe.cuh; there is no CPU fallback: without a CUDA device every entry point that needs
// one returns SW_ERR_CUDA.
#include "../../include/sw.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "sw_host.h"
#include "sw_common.cuh"
#include "sw_generic.cuh"
#include "sw_observe.cuh"
#include "sw_tiled.cuh"
#include "sw_tile_blocks.cuh"
#include "sw_cluster.cuh"

namespace {

using sw::Params;

enum Slot { SLOT_TILE = 0, SLOT_MERGE = 1, SLOT_FLIP = 2, SLOT_G_BONDS = 3, SLOT_G_INIT = 4,
            SLOT_G_UNION = 5, SLOT_G_FLATTEN = 6, SLOT_G_FLIP = 7 };   // the cluster path's one kernel is timed in SLOT_TILE
const char *const kSlotNames[SW_MAX_KERNEL_SLOTS] = {
    "k_tile_blocks", "k_tile_merge", "k_tile_flip", "k_bonds_generic", "k_label_identity",
    "k_union_generic", "k_flatten_generic", "k_flip_generic"};

constexpr size_t kAlign = 256;
inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

struct Plan {
    size_t spins, bonds, labels, rootbits, border, edges, btab, tile_clusters, draws, row, flag, rows, stage, counters, sizes, total;   // byte offsets into the workspace
    size_t rows_cap, stage_bytes;      // rows of the sw_sweep_measure ring; bytes of the sw_get_bonds staging buffer
};

constexpr uint32_t kAllFlags = SW_FLAG_FORCE_GENERIC | SW_FLAG_LAZY_LABELS | SW_FLAG_LABEL_EQUIVALENCE | SW_FLAG_WS_CLUSTER_SIZES |
                               SW_FLAG_PASS_COUNTERS | SW_FLAG_NO_CLUSTER_PATH;

bool tiled_ok(uint32_t L, uint32_t flags) { return (L % sw::kTile == 0) && !(flags & (SW_FLAG_FORCE_GENERIC | SW_FLAG_LABEL_EQUIVALENCE)); }

Plan make_plan(uint32_t L, uint32_t q, uint32_t flags)
{
    const uint64_t N = (uint64_t)L * L;
    Plan p{};
    size_t off = 0;
    p.spins = off;  off = align_up(off + N);
    p.bonds = off;  off = align_up(off + ((N + 15) / 16) * 4);
    p.labels = off; off = align_up(off + N * 4);
    p.rootbits = off; off = align_up(off + (tiled_ok(L, flags) ? (N / 16) * 2 : 0));
    p.border = off; off = align_up(off + (tiled_ok(L, flags) ? (N / sw::kTileSites) * sizeof(sw::TileBorder) : 0));
    p.edges = off; off = align_up(off + (tiled_ok(L, flags) ? (N / sw::kTileSites) * sizeof(sw::TileEdges) : 0));
    p.btab = off; off = align_up(off + (tiled_ok(L, flags) ? (N / sw::kTileSites) * sw::kBorderTabEntries * 4 : 0));
    p.tile_clusters = off; off = align_up(off + (tiled_ok(L, flags) ? (N / sw::kTileSites) * (sw::kFlipThreads / 32) * 4 : 0));
    p.draws = off;  off = align_up(off + (tiled_ok(L, flags) ? (N / 32) * sizeof(uint2) : 0));   // one uint2 per 8 x 4 block
    p.row = off;    off = align_up(off + (3 + (size_t)q + 2) * 8);   // + the two words of sum |c|^2 (sw_measure_clusters)
    p.flag = off;   off = align_up(off + 4);
    // scratch the read-back / measurement calls need, owned by the context (no cudaMalloc behind the caller's back):
    // a ring of observable rows for sw_sweep_measure, a staging buffer for sw_get_bonds, the pass counters of sw_get_stats
    p.rows_cap = std::max<size_t>(16, std::min<size_t>(4096, (256u << 10) / ((3 + (size_t)q) * 8)));
    p.rows = off;   off = align_up(off + p.rows_cap * (3 + (size_t)q) * 8);
    p.stage_bytes = (size_t)std::max<uint64_t>(512, (std::min<uint64_t>(N, 32ull << 20) + 511) / 512 * 512);   // two 256-byte-aligned halves
    p.stage = off;  off = align_up(off + p.stage_bytes);
    p.counters = off; off = align_up(off + sizeof(sw::PassCounters));
    // the 4N-byte cluster-size scratch of sw_measure(largest_cluster): part of the workspace only on request
    // (SW_FLAG_WS_CLUSTER_SIZES); otherwise it is allocated once, on the first call that needs it
    p.sizes = off;  off = align_up(off + ((flags & SW_FLAG_WS_CLUSTER_SIZES) ? N * 4 : 0));
    p.total = off;
    return p;
}

}  // namespace

struct sw_ctx {
    uint32_t L = 0, q = 0, flags = 0;
    uint64_t N = 0, seed = 0, T = 0, t = 0;
    double K = 0;
    bool tiled = false, lazy = false, label_equiv = false;
    bool cluster = false;                 // small lattice: all sweeps of a call in ONE launch of k_cluster_sweeps (sw_cluster.cuh)
    uint32_t counts_per_tile = sw::kFlipThreads / 32;   // entries per tile the last flip left in d_tile_clusters
    uint64_t counts_t = ~0ull;            // == t: d_tile_clusters holds the root counts of the last sweep (a flip with kCount ran)
    uint64_t le_rounds_last = 0, le_rounds_total = 0;
    bool have_spins = false, have_labels = false, labels_flat = false;
    bool owns_ws = false, owns_stream = false;
    int device = 0;
    cudaStream_t stream = nullptr;
    uint8_t *ws = nullptr;
    size_t ws_bytes = 0;
    uint8_t *d_spins = nullptr;
    uint32_t *d_bonds = nullptr, *d_labels = nullptr, *d_flag = nullptr, *d_tile_clusters = nullptr;
    uint2 *d_draws = nullptr;             // bond-draw masks of sweep draws_t (tiled path), made one sweep ahead
    uint64_t draws_t = ~0ull;
    uint16_t *d_rootbits = nullptr;
    sw::TileBorder *d_border = nullptr;
    sw::TileEdges *d_edges = nullptr;
    uint32_t *d_btab = nullptr;          // per tile: the components that own a site on the tile border (k_tile_blocks_sizes)
    unsigned long long *d_row = nullptr;
    unsigned long long *d_rows = nullptr; // ring of observable rows for sw_sweep_measure (rows_cap rows)
    size_t rows_cap = 0;
    uint8_t *d_stage = nullptr;           // staging buffer of sw_get_bonds (stage_bytes)
    size_t stage_bytes = 0;
    sw::PassCounters *d_counters = nullptr;   // SW_FLAG_PASS_COUNTERS
    bool count_passes = false;
    uint32_t *d_sizes = nullptr;          // 4N-byte scratch for cluster sizes: in the workspace (SW_FLAG_WS_CLUSTER_SIZES) or
    bool owns_sizes = false;              // allocated once by the first sw_measure(largest_cluster)
    bool sizes_zero = false;              // d_sizes is all zero (k_max_size_zero leaves it so; the counting sweeps rely on it)
    uint64_t sizes_t = ~0ull;             // == t: d_sizes holds the cluster sizes of the last sweep, counted by k_tile_blocks_sizes + k_tile_flip_sizes
    uint64_t launches = 0, sweeps = 0;
    int num_sms = 148;
    // profiling: events are created once and reused (no cudaEventCreate inside a timed region after the first pass)
    bool profiling = false;
    struct Ev { int slot; uint64_t sweep; cudaEvent_t a, b; };
    std::vector<Ev> events;               // recorded since sw_profile_begin
    std::vector<cudaEvent_t> event_pool;  // idle events
    std::vector<double> series;           // per-sweep device time of the last profiled region (sw_profile_series)
    std::string err;
};

// every ABI call runs on the device the context was created on, whatever the caller's current device is
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const sw_ctx *c) {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) cudaSetDevice(c->device); else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

namespace {

int fail(sw_ctx *c, int code, const char *what)
{
    if (c) c->err = what;
    return code;
}

int cuda_fail(sw_ctx *c, cudaError_t e, const char *what)
{
    if (c) c->err = std::string(what) + ": " + cudaGetErrorString(e);
    return SW_ERR_CUDA;
}

#define SW_CUDA(c, call)                                            \
    do {                                                            \
        cudaError_t e_ = (call);                                    \
        if (e_ != cudaSuccess) return cuda_fail((c), e_, #call);    \
    } while (0)

using swh::host_threshold;   // T = floor(p * 2^32), p = 1 - exp(-K), computed once on the host (sw_host.h; R10)

Params make_params(const sw_ctx *c, uint64_t t)
{
    return swh::make_params(c->L, c->q, c->N, c->seed, c->T, t);
}

int grid_for(const sw_ctx *c, uint64_t items, int threads)
{
    const uint64_t want = (items + threads - 1) / threads;
    const uint64_t cap = (uint64_t)c->num_sms * 16;
    return (int)(want < 1 ? 1 : (want > cap ? cap : want));
}

cudaEvent_t take_event(sw_ctx *c)
{
    cudaEvent_t e = nullptr;
    if (!c->event_pool.empty()) { e = c->event_pool.back(); c->event_pool.pop_back(); return e; }
    return cudaEventCreate(&e) == cudaSuccess ? e : nullptr;
}

struct Timed {
    sw_ctx *c; int slot; cudaEvent_t a = nullptr, b = nullptr;
    Timed(sw_ctx *c_, int slot_) : c(c_), slot(slot_) {
        c->launches += 1;
        if (c->profiling && (a = take_event(c)) && (b = take_event(c))) cudaEventRecord(a, c->stream);
    }
    ~Timed() {
        if (a && b) { cudaEventRecord(b, c->stream); c->events.push_back({slot, c->sweeps, a, b}); }
    }
};

// Small lattices: n sweeps in one launch (sw_cluster.cuh).  what != 0: the observables of every sweep go to d_rows
// (zeroed here), one row per sweep; the caller keeps n <= rows_cap then.
int sweep_cluster(sw_ctx *c, uint64_t n, uint32_t what, unsigned long long *d_rows)
{
    const Params P = make_params(c, c->t);
    const dim3 tgrid(c->L / sw::kTile, c->L / sw::kTile);
    if (c->draws_t != c->t) {
        c->launches += 1;
        sw::k_draws<<<tgrid, 256, 0, c->stream>>>(c->d_draws, P);
    }
    if (what) SW_CUDA(c, cudaMemsetAsync(d_rows, 0, (size_t)n * (3 + (size_t)c->q) * 8, c->stream));
    if ((what & SW_OBS_LARGEST) && !c->d_sizes) {
        SW_CUDA(c, cudaMalloc(&c->d_sizes, c->N * 4));
        c->owns_sizes = true;
    }
    if (what & SW_OBS_LARGEST) c->sizes_zero = false;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = tgrid; cfg.blockDim = dim3(sw::kClusterThreads); cfg.dynamicSmemBytes = 0; cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = tgrid.x; attr[0].val.clusterDim.y = tgrid.y; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    {
        Timed tm(c, SLOT_TILE);
        const uint32_t n32 = (uint32_t)n;
        cudaError_t e = what ? cudaLaunchKernelEx(&cfg, sw::k_cluster_sweeps<true>, c->d_spins, c->d_bonds, c->d_labels, c->d_rootbits, c->d_border,
                                                  c->d_edges, c->d_draws, c->d_tile_clusters, P, n32, what, d_rows, c->d_sizes)
                             : cudaLaunchKernelEx(&cfg, sw::k_cluster_sweeps<false>, c->d_spins, c->d_bonds, c->d_labels, c->d_rootbits, c->d_border,
                                                  c->d_edges, c->d_draws, c->d_tile_clusters, P, n32, 0u, (unsigned long long *)nullptr, (uint32_t *)nullptr);
        if (e != cudaSuccess) return cuda_fail(c, e, "k_cluster_sweeps launch");
    }
    c->t += n; c->sweeps += n;
    c->draws_t = c->t;
    c->have_labels = true; c->labels_flat = true;
    c->counts_per_tile = sw::kClusterThreads / 32;
    c->counts_t = c->t;                  // the cluster kernel counts the roots of every sweep
    return SW_OK;
}

// can a cluster of all the tiles be co-scheduled on this device?
bool cluster_path_ok(sw_ctx *c)
{
    const unsigned tiles = (unsigned)(c->N / sw::kTileSites);
    if (!c->tiled || tiles > sw::kClusterMaxTiles || c->lazy || c->count_passes) return false;
    for (int m = 0; m < 2; ++m) {
        const void *fn = m ? (const void *)sw::k_cluster_sweeps<true> : (const void *)sw::k_cluster_sweeps<false>;
        if (tiles > 8 && cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) { cudaGetLastError(); return false; }
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(c->L / sw::kTile, c->L / sw::kTile); cfg.blockDim = dim3(sw::kClusterThreads);
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = cfg.gridDim.x; attr[0].val.clusterDim.y = cfg.gridDim.y; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        int n_clusters = 0;
        if (cudaOccupancyMaxActiveClusters(&n_clusters, fn, &cfg) != cudaSuccess || n_clusters < 1) { cudaGetLastError(); return false; }
    }
    return true;
}

// the cluster-size counters: there, and all zero
int ensure_sizes_zero(sw_ctx *c)
{
    if (!c->d_sizes) {                   // not part of the workspace (no SW_FLAG_WS_CLUSTER_SIZES): allocated once, kept until sw_destroy
        SW_CUDA(c, cudaMalloc(&c->d_sizes, c->N * 4));
        c->owns_sizes = true;
        c->sizes_zero = false;
    }
    if (!c->sizes_zero) {
        SW_CUDA(c, cudaMemsetAsync(c->d_sizes, 0, c->N * 4, c->stream));
        c->sizes_zero = true;
    }
    return SW_OK;
}

// count_clusters: the flip kernel also counts the canonical roots (wanted for the last sweep before a measurement);
// sizes_row != nullptr (a zeroed row of observables): the sweep counts the cluster sizes as well.  The tile kernel counts
// the sites of its tile-local components: those inside one tile are whole clusters and only raise sizes_row[2], the
// others go through the tile's border table to the flip kernel, which adds them up in d_sizes at the canonical roots for
// k_max_size_zero (k_tile_blocks_sizes, k_tile_flip_sizes)
int sweep_once(sw_ctx *c, bool count_clusters, unsigned long long *sizes_row = nullptr)
{
    const Params P = make_params(c, c->t);
    if (c->tiled) {
        const unsigned tiles = (unsigned)(c->N / sw::kTileSites);
        const dim3 tgrid(c->L / sw::kTile, c->L / sw::kTile);      // one CTA per tile, (tx, ty)
        if (c->draws_t != c->t) {        // first sweep after sw_init / sw_set_state: nobody has made this sweep's bond draws yet
            c->launches += 1;
            sw::k_draws<<<tgrid, 256, 0, c->stream>>>(c->d_draws, P);
        }
        const bool with_sizes = sizes_row && !c->lazy && !c->count_passes;
        if (with_sizes) {
            const int rc = ensure_sizes_zero(c);
            if (rc != SW_OK) return rc;
            Timed tm(c, SLOT_TILE);
            sw::k_tile_blocks_sizes<<<tgrid, sw::kBlkThreads, 0, c->stream>>>(c->d_spins, c->d_bonds, c->d_labels, c->d_rootbits, c->d_border, c->d_edges, c->d_draws, P, c->d_btab, sizes_row);
            c->sizes_zero = false;
        } else
        { Timed tm(c, SLOT_TILE);
          sw::k_tile_blocks<<<tgrid, sw::kBlkThreads, 0, c->stream>>>(c->d_spins, c->d_bonds, c->d_labels, c->d_rootbits, c->d_border, c->d_edges, c->d_draws, P); }
        { Timed tm(c, SLOT_MERGE);
          const unsigned per = (unsigned)sw::merge_tiles_per_cta(tiles);
          auto merge = per == 2 ? (c->count_passes ? sw::k_tile_merge<true, 2> : sw::k_tile_merge<false, 2>)
                                : (c->count_passes ? sw::k_tile_merge<true, 4> : sw::k_tile_merge<false, 4>);
          merge<<<(tiles + per - 1) / per, sw::kMergeThreads, 0, c->stream>>>(c->d_labels, c->d_border, c->d_edges, P, tiles, c->d_counters); }
        if (with_sizes) {
            Timed tm(c, SLOT_FLIP);
            sw::k_tile_flip_sizes<<<tgrid, sw::kFlipThreads, 0, c->stream>>>(c->d_labels, c->d_rootbits, c->d_spins, P, c->d_tile_clusters, c->d_draws, c->d_sizes, c->d_btab);
            c->sizes_t = c->t + 1;
        } else
        { Timed tm(c, SLOT_FLIP);
          auto flip = c->count_passes ? (c->lazy ? sw::k_tile_flip<false, true, true, true> : sw::k_tile_flip<true, true, true, true>)
                    : c->lazy ? (count_clusters ? sw::k_tile_flip<false, true, true> : sw::k_tile_flip<false, true, false>)
                              : (count_clusters ? sw::k_tile_flip<true, true, true> : sw::k_tile_flip<true, true, false>);
          flip<<<tgrid, sw::kFlipThreads, 0, c->stream>>>(c->d_labels, c->d_rootbits, c->d_spins, P, c->d_tile_clusters, c->d_draws, c->d_counters); }
        c->draws_t = c->t + 1;           // the flip kernel made the draws of the next sweep on the side
        c->labels_flat = !c->lazy;
        if (with_sizes || count_clusters || c->count_passes) {     // the flip instantiations with kCount
            c->counts_per_tile = sw::kFlipThreads / 32;
            c->counts_t = c->t + 1;
        }
    } else if (c->label_equiv) {
        // the loop of scanning and analysis kernels "is iterated up to the point when the information of
        // the labeling needs no more process of scanning function"; as in the paper the host looks at a flag every round
        const int th = 256;
        { Timed tm(c, SLOT_G_BONDS);
          sw::k_bonds_generic<<<grid_for(c, (c->N + 15) / 16, th), th, 0, c->stream>>>(c->d_spins, c->d_bonds, P); }
        { Timed tm(c, SLOT_G_INIT);
          sw::k_label_identity<<<grid_for(c, c->N, th), th, 0, c->stream>>>(c->d_labels, P); }
        c->le_rounds_last = 0;
        for (uint32_t changed = 1; changed;) {
            SW_CUDA(c, cudaMemsetAsync(c->d_flag, 0, 4, c->stream));
            { Timed tm(c, SLOT_G_UNION);       // slot names in this mode: k_le_scan / k_le_analysis (sw_kernel_name)
              sw::k_le_scan<<<grid_for(c, c->N, th), th, 0, c->stream>>>(c->d_bonds, c->d_labels, P, c->d_flag); }
            { Timed tm(c, SLOT_G_FLATTEN);
              sw::k_le_analysis<<<grid_for(c, c->N, th), th, 0, c->stream>>>(c->d_labels, P); }
            SW_CUDA(c, cudaMemcpyAsync(&changed, c->d_flag, 4, cudaMemcpyDeviceToHost, c->stream));
            SW_CUDA(c, cudaStreamSynchronize(c->stream));
            c->le_rounds_last += 1;
        }
        c->le_rounds_total += c->le_rounds_last;
        { Timed tm(c, SLOT_G_FLIP);
          sw::k_flip_generic<<<grid_for(c, c->N, th), th, 0, c->stream>>>(c->d_labels, c->d_spins, P); }
        c->labels_flat = true;
    } else {
        const int th = 256;
        { Timed tm(c, SLOT_G_BONDS);
          sw::k_bonds_generic<<<grid_for(c, (c->N + 15) / 16, th), th, 0, c->stream>>>(c->d_spins, c->d_bonds, P); }
        { Timed tm(c, SLOT_G_INIT);
          sw::k_label_identity<<<grid_for(c, c->N, th), th, 0, c->stream>>>(c->d_labels, P); }
        { Timed tm(c, SLOT_G_UNION);
          sw::k_union_generic<<<grid_for(c, c->N, th), th, 0, c->stream>>>(c->d_bonds, c->d_labels, P); }
        if (!c->lazy) {
            Timed tm(c, SLOT_G_FLATTEN);
            sw::k_flatten_generic<<<grid_for(c, c->N, th), th, 0, c->stream>>>(c->d_labels, P);
        }
        { Timed tm(c, SLOT_G_FLIP);
          sw::k_flip_generic<<<grid_for(c, c->N, th), th, 0, c->stream>>>(c->d_labels, c->d_spins, P); }
        c->labels_flat = !c->lazy;
    }
    c->t += 1;
    c->sweeps += 1;
    c->have_labels = true;
    return SW_OK;
}

int ensure_flat(sw_ctx *c)
{
    if (c->labels_flat) return SW_OK;
    const Params P = make_params(c, c->t);
    c->launches += 1;
    if (c->tiled)       // lazy mode: the forest of the last sweep is still in place (tile-local ids + root links)
        sw::k_tile_flip<true, false, false><<<dim3(c->L / sw::kTile, c->L / sw::kTile), sw::kFlipThreads, 0, c->stream>>>(c->d_labels, c->d_rootbits, c->d_spins, P, c->d_tile_clusters, nullptr, nullptr);
    else
        sw::k_flatten_generic<<<grid_for(c, c->N, 256), 256, 0, c->stream>>>(c->d_labels, P);
    SW_CUDA(c, cudaGetLastError());
    c->labels_flat = true;
    return SW_OK;
}

// Enqueue the observable kernels for the current state into the device row `row` (zeroed here).
// row_is_zero: the caller zeroed the row already
int enqueue_observe(sw_ctx *c, unsigned long long *row, bool want_e, bool want_m, bool want_nc, bool want_big, unsigned long long *c2 = nullptr,
                    bool row_is_zero = false)
{
    const Params P = make_params(c, c->t);
    if (!row_is_zero) SW_CUDA(c, cudaMemsetAsync(row, 0, (3 + (size_t)c->q) * 8, c->stream));
    const bool cl = c->have_labels;
    uint32_t want = (want_e ? 1u : 0u) | (want_m ? 2u : 0u) | ((cl && (want_nc || want_big)) ? 4u : 0u);
    if ((want & 4u) && c->tiled && c->counts_t != c->t) {
        // the last sweep ran without the count (sw_sweep_measure_ex without SW_OBS_CLUSTERS / SW_OBS_LARGEST): d_tile_clusters is
        // stale or was never written; count the roots (labels[i] == i) in the observe pass below, on flat labels
        const int rc = ensure_flat(c);
        if (rc != SW_OK) return rc;
    } else if ((want & 4u) && c->tiled) {      // the flip kernel of the last sweep left one count per tile: no pass over labels[]
        want &= ~4u;
        c->launches += 1;
        const unsigned tiles = (unsigned)(c->N / sw::kTileSites) * c->counts_per_tile;   // one count per warp of the last flip
        sw::k_sum_tile_clusters<<<grid_for(c, tiles, sw::kObsThreads), sw::kObsThreads, 0, c->stream>>>(c->d_tile_clusters, tiles, row);
    }
    if (want) {
        c->launches += 1;
        if (c->L % 16 == 0)
            sw::k_observe_vec16<<<grid_for(c, c->N / 64, sw::kObsThreads), sw::kObsThreads, 0, c->stream>>>(c->d_spins, c->d_labels, P, want, row);
        else
            sw::k_observe_scalar<<<grid_for(c, c->N, sw::kObsThreads), sw::kObsThreads, 0, c->stream>>>(c->d_spins, c->d_labels, P, want, row);
    }
    if (cl && want_big && c->tiled && c->sizes_t == c->t && !c2) {
        // the kernels of the last sweep counted the sizes: clusters inside one tile are in row[2] already, the others in d_sizes
        c->launches += 1;
        sw::k_max_size_zero<<<grid_for(c, c->N / 4, 256), 256, 0, c->stream>>>(c->d_sizes, P, row);
        c->sizes_zero = true;
        c->sizes_t = ~0ull;
    } else if (cl && want_big) {
        if (c->tiled) {          // cluster sizes need root pointers: on the tiled path labels[] holds tile-local ids until flattened
            const int rc = ensure_flat(c);
            if (rc != SW_OK) return rc;
        }
        c->sizes_t = ~0ull;
        const int rc = ensure_sizes_zero(c);
        if (rc != SW_OK) return rc;
        c->launches += 2;
        c->sizes_zero = false;
        sw::k_cluster_sizes<<<grid_for(c, (c->N + 15) / 16, 256), 256, 0, c->stream>>>(c->d_labels, c->d_sizes, P);
        if (c2) {
            SW_CUDA(c, cudaMemsetAsync(c2, 0, 16, c->stream));
            sw::k_size_moments<<<grid_for(c, c->N, 256), 256, 0, c->stream>>>(c->d_sizes, P, row, c2);
        } else if (c->N % 4 == 0) {
            sw::k_max_size_zero<<<grid_for(c, c->N / 4, 256), 256, 0, c->stream>>>(c->d_sizes, P, row);
            c->sizes_zero = true;
        } else sw::k_max_size<<<grid_for(c, c->N, 256), 256, 0, c->stream>>>(c->d_sizes, P, row);
    }
    SW_CUDA(c, cudaGetLastError());
    return SW_OK;
}

// a uint32 size counter wraps to 0 only when one cluster holds all 2^32 sites
void fix_row(const sw_ctx *c, uint64_t *row)
{
    if (row[1] == 1) row[2] = c->N;
}

int create_common(sw_ctx **out, uint32_t L, uint32_t q, double K, uint64_t seed, uint32_t flags,
                  void *dev_ws, size_t ws_bytes, void *stream, bool external)
{
    if (!out) return SW_ERR_INVALID_ARG;
    *out = nullptr;
    uint64_t T = 0;
    if (L < 2 || L > 65536 || q < 2 || q > 255 || !host_threshold(K, &T)) return SW_ERR_INVALID_ARG;
    if (flags & ~kAllFlags) return SW_ERR_INVALID_ARG;
    sw_ctx *c = new (std::nothrow) sw_ctx();
    if (!c) return SW_ERR_OOM;
    c->L = L; c->q = q; c->K = K; c->seed = seed; c->T = T; c->flags = flags;
    c->N = (uint64_t)L * L;
    c->tiled = tiled_ok(L, flags);
    c->label_equiv = (flags & SW_FLAG_LABEL_EQUIVALENCE) != 0;
    c->lazy = (flags & SW_FLAG_LAZY_LABELS) != 0 && !c->label_equiv;   // the analysis kernel leaves flat labels anyway
    const Plan plan = make_plan(L, q, flags);
    cudaError_t e = cudaGetDevice(&c->device);
    if (e != cudaSuccess) { delete c; return SW_ERR_CUDA; }
    cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device);
    if (external) {
        if (!dev_ws || ws_bytes < plan.total || ((uintptr_t)dev_ws % kAlign) != 0) { delete c; return dev_ws ? SW_ERR_OOM : SW_ERR_INVALID_ARG; }
        c->ws = (uint8_t *)dev_ws; c->stream = (cudaStream_t)stream;
    } else {
        if (cudaMalloc(&c->ws, plan.total) != cudaSuccess) { cudaGetLastError(); delete c; return SW_ERR_OOM; }
        c->owns_ws = true;
        if (cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) != cudaSuccess) { cudaFree(c->ws); delete c; return SW_ERR_CUDA; }
        c->owns_stream = true;
    }
    c->ws_bytes = plan.total;
    c->d_spins = c->ws + plan.spins;
    c->d_bonds = (uint32_t *)(c->ws + plan.bonds);
    c->d_labels = (uint32_t *)(c->ws + plan.labels);
    c->d_rootbits = (uint16_t *)(c->ws + plan.rootbits);
    c->d_border = (sw::TileBorder *)(c->ws + plan.border);
    c->d_edges = (sw::TileEdges *)(c->ws + plan.edges);
    c->d_btab = (uint32_t *)(c->ws + plan.btab);
    c->d_tile_clusters = (uint32_t *)(c->ws + plan.tile_clusters);
    c->d_draws = (uint2 *)(c->ws + plan.draws);
    c->d_row = (unsigned long long *)(c->ws + plan.row);
    c->d_flag = (uint32_t *)(c->ws + plan.flag);
    c->d_rows = (unsigned long long *)(c->ws + plan.rows); c->rows_cap = plan.rows_cap;
    c->d_stage = c->ws + plan.stage; c->stage_bytes = plan.stage_bytes;
    c->d_counters = (sw::PassCounters *)(c->ws + plan.counters);
    c->count_passes = (flags & SW_FLAG_PASS_COUNTERS) != 0 && c->tiled;
    c->cluster = !(flags & SW_FLAG_NO_CLUSTER_PATH) && cluster_path_ok(c);
    if (flags & SW_FLAG_WS_CLUSTER_SIZES) c->d_sizes = (uint32_t *)(c->ws + plan.sizes);
    if (cudaMemsetAsync(c->d_counters, 0, sizeof(sw::PassCounters), c->stream) != cudaSuccess) {
        cudaGetLastError();
        if (c->owns_stream) cudaStreamDestroy(c->stream);
        if (c->owns_ws) cudaFree(c->ws);
        delete c;
        return SW_ERR_CUDA;
    }
    *out = c;
    return SW_OK;
}

}  // namespace

extern "C" {

const char *sw_version(void) { return "sw-b200 0.1 (sm_100a)"; }

size_t sw_workspace_bytes(uint32_t L, uint32_t q, uint32_t flags)
{
    if (L < 2 || L > 65536 || q < 2 || q > 255) return 0;
    return make_plan(L, q, flags).total;
}

int sw_create(sw_ctx **out, uint32_t L, uint32_t q, double K, uint64_t seed)
{
    return create_common(out, L, q, K, seed, SW_FLAG_DEFAULT, nullptr, 0, nullptr, false);
}

int sw_create_ex(sw_ctx **out, uint32_t L, uint32_t q, double K, uint64_t seed, uint32_t flags)
{
    return create_common(out, L, q, K, seed, flags, nullptr, 0, nullptr, false);
}

int sw_create_ws(sw_ctx **out, uint32_t L, uint32_t q, double K, uint64_t seed, uint32_t flags,
                 void *dev_ws, size_t ws_bytes, void *cuda_stream)
{
    return create_common(out, L, q, K, seed, flags, dev_ws, ws_bytes, cuda_stream, true);
}

void sw_destroy(sw_ctx *c)
{
    if (!c) return;
    DeviceGuard dg(c);
    cudaStreamSynchronize(c->stream);
    for (auto &ev : c->events) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
    for (auto &ev : c->event_pool) cudaEventDestroy(ev);
    if (c->d_sizes && c->owns_sizes) cudaFree(c->d_sizes);
    if (c->owns_ws) cudaFree(c->ws);
    if (c->owns_stream) cudaStreamDestroy(c->stream);
    delete c;
}

int sw_init(sw_ctx *c, int mode)
{
    if (!c) return SW_ERR_INVALID_ARG;
    DeviceGuard dg(c);
    if (mode == SW_INIT_ORDERED) {
        SW_CUDA(c, cudaMemsetAsync(c->d_spins, 0, c->N, c->stream));
    } else if (mode == SW_INIT_RANDOM) {
        const Params P = make_params(c, 0);
        c->launches += 1;
        sw::k_init_random<<<grid_for(c, c->N, 256), 256, 0, c->stream>>>(c->d_spins, P);
        SW_CUDA(c, cudaGetLastError());
    } else return fail(c, SW_ERR_INVALID_ARG, "sw_init: unknown mode");
    c->t = 0; c->have_spins = true; c->have_labels = false; c->labels_flat = false; c->sizes_t = ~0ull; c->counts_t = ~0ull;
    return SW_OK;
}

int sw_set_state(sw_ctx *c, const uint8_t *src, uint64_t t)
{
    if (!c || !src || t > 0xFFFFFFFFull) return fail(c, SW_ERR_INVALID_ARG, "sw_set_state: bad argument");
    DeviceGuard dg(c);
    SW_CUDA(c, cudaMemcpyAsync(c->d_spins, src, c->N, cudaMemcpyHostToDevice, c->stream));
    SW_CUDA(c, cudaMemsetAsync(c->d_flag, 0, 4, c->stream));
    const Params P = make_params(c, 0);
    c->launches += 1;
    sw::k_validate_spins<<<grid_for(c, c->N, 256), 256, 0, c->stream>>>(c->d_spins, P, c->d_flag);
    uint32_t bad = 0;
    SW_CUDA(c, cudaMemcpyAsync(&bad, c->d_flag, 4, cudaMemcpyDeviceToHost, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    c->have_labels = false; c->labels_flat = false; c->sizes_t = ~0ull; c->counts_t = ~0ull;
    if (bad) { c->have_spins = false; return fail(c, SW_ERR_INVALID_ARG, "sw_set_state: spin value >= q"); }
    c->t = t; c->have_spins = true;
    return SW_OK;
}

static bool packed_ok(const sw_ctx *c, uint32_t bits)
{
    return (bits == 1 || bits == 2 || bits == 4 || bits == 8) && c->q <= (1u << bits) && c->N % 16 == 0;
}

int sw_set_state_packed(sw_ctx *c, const void *src, uint32_t bits, uint64_t t)
{
    if (!c || !src || t > 0xFFFFFFFFull) return fail(c, SW_ERR_INVALID_ARG, "sw_set_state_packed: bad argument");
    if (!packed_ok(c, bits)) return fail(c, SW_ERR_INVALID_ARG, "sw_set_state_packed: bits must be 1, 2, 4 or 8 with q <= 2^bits, and L*L a multiple of 16");
    DeviceGuard dg(c);
    // the packed image is staged in the label array (the labels of the last sweep are forgotten by a new state anyway)
    uint8_t *staged = reinterpret_cast<uint8_t *>(c->d_labels);
    SW_CUDA(c, cudaMemcpyAsync(staged, src, (size_t)(c->N / 8 * bits), cudaMemcpyHostToDevice, c->stream));
    SW_CUDA(c, cudaMemsetAsync(c->d_flag, 0, 4, c->stream));
    const Params P = make_params(c, 0);
    c->launches += 1;
    sw::k_unpack_spins<<<grid_for(c, c->N / 16, 256), 256, 0, c->stream>>>(staged, c->d_spins, P, bits, c->d_flag);
    uint32_t bad = 0;
    SW_CUDA(c, cudaMemcpyAsync(&bad, c->d_flag, 4, cudaMemcpyDeviceToHost, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    c->have_labels = false; c->labels_flat = false; c->sizes_t = ~0ull; c->counts_t = ~0ull;
    if (bad) { c->have_spins = false; return fail(c, SW_ERR_INVALID_ARG, "sw_set_state_packed: spin value >= q"); }
    c->t = t; c->have_spins = true;
    return SW_OK;
}

int sw_get_spins_packed(sw_ctx *c, void *dst, uint32_t bits)
{
    if (!c || !dst) return fail(c, SW_ERR_INVALID_ARG, "sw_get_spins_packed: bad argument");
    if (!packed_ok(c, bits)) return fail(c, SW_ERR_INVALID_ARG, "sw_get_spins_packed: bits must be 1, 2, 4 or 8 with q <= 2^bits, and L*L a multiple of 16");
    if (!c->have_spins) return fail(c, SW_ERR_STATE, "no spins");
    DeviceGuard dg(c);
    // packed in chunks through the context's staging buffer, two halves in flight
    const uint64_t n_groups = c->N / 16, bytes_per_group = 2ull * bits;
    const uint64_t half = std::max<uint64_t>(1, (c->stage_bytes / 2) / bytes_per_group);      // groups per half
    uint64_t done = 0;
    for (int k = 0; done < n_groups; ++k) {
        const uint64_t m = std::min(half, n_groups - done);
        uint8_t *buf = c->d_stage + (k & 1) * (c->stage_bytes / 2);
        c->launches += 1;
        sw::k_pack_spins<<<grid_for(c, m, 256), 256, 0, c->stream>>>(c->d_spins, buf, done, m, bits);
        SW_CUDA(c, cudaMemcpyAsync((uint8_t *)dst + done * bytes_per_group, buf, (size_t)(m * bytes_per_group), cudaMemcpyDeviceToHost, c->stream));
        done += m;
    }
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    SW_CUDA(c, cudaGetLastError());
    return SW_OK;
}

int sw_sweep(sw_ctx *c, uint64_t n)
{
    if (!c) return SW_ERR_INVALID_ARG;
    if (!c->have_spins) return fail(c, SW_ERR_STATE, "sw_sweep: no spins (call sw_init or sw_set_state)");
    if (c->t + n > 0x100000000ull) return fail(c, SW_ERR_STATE, "sw_sweep: sweep counter would pass 2^32");
    DeviceGuard dg(c);
    if (c->cluster) {                    // small lattice: all the sweeps in one launch (chunks keep the 32-bit loop counter safe)
        for (uint64_t done = 0; done < n;) {
            const uint64_t m = std::min<uint64_t>(n - done, 1u << 16);   // (a launch of 65 536 sweeps runs for about two seconds)
            const int rc = sweep_cluster(c, m, 0, nullptr);
            if (rc != SW_OK) return rc;
            done += m;
        }
        SW_CUDA(c, cudaGetLastError());
        return SW_OK;
    }
    for (uint64_t k = 0; k < n; ++k) {
        const int rc = sweep_once(c, k + 1 == n);
        if (rc != SW_OK) return rc;
    }
    SW_CUDA(c, cudaGetLastError());
    return SW_OK;
}

int sw_measure(sw_ctx *c, uint64_t *energy_bonds, uint64_t *mag_counts, uint64_t *n_clusters, uint64_t *largest_cluster)
{
    if (!c) return SW_ERR_INVALID_ARG;
    if (!c->have_spins) return fail(c, SW_ERR_STATE, "sw_measure: no spins");
    DeviceGuard dg(c);
    const int rc = enqueue_observe(c, c->d_row, energy_bonds != nullptr, mag_counts != nullptr,
                                   n_clusters != nullptr || largest_cluster != nullptr, largest_cluster != nullptr);
    if (rc != SW_OK) return rc;
    std::vector<uint64_t> row(3 + c->q);
    SW_CUDA(c, cudaMemcpyAsync(row.data(), c->d_row, row.size() * 8, cudaMemcpyDeviceToHost, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    fix_row(c, row.data());
    if (energy_bonds) *energy_bonds = row[0];
    if (n_clusters) *n_clusters = c->have_labels ? row[1] : 0;
    if (largest_cluster) *largest_cluster = c->have_labels ? row[2] : 0;
    if (mag_counts) for (uint32_t s = 0; s < c->q; ++s) mag_counts[s] = row[3 + s];
    return SW_OK;
}

int sw_measure_clusters(sw_ctx *c, uint64_t *n_clusters, uint64_t *largest_cluster, uint64_t sum_sq[2])
{
    if (!c || !sum_sq) return SW_ERR_INVALID_ARG;
    if (!c->have_labels) return fail(c, SW_ERR_STATE, "sw_measure_clusters: no sweep since sw_init");
    DeviceGuard dg(c);
    unsigned long long *c2 = c->d_row + 3 + c->q;
    const int rc = enqueue_observe(c, c->d_row, false, false, true, true, c2);
    if (rc != SW_OK) return rc;
    std::vector<uint64_t> row(3 + c->q + 2);
    SW_CUDA(c, cudaMemcpyAsync(row.data(), c->d_row, row.size() * 8, cudaMemcpyDeviceToHost, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    fix_row(c, row.data());
    if (n_clusters) *n_clusters = row[1];
    if (largest_cluster) *largest_cluster = row[2];
    sum_sq[0] = row[3 + c->q]; sum_sq[1] = row[3 + c->q + 1];
    if (row[1] == 1 && c->N == (1ull << 32)) { sum_sq[0] = 0; sum_sq[1] = 1; }   // one cluster of 2^32 sites: its uint32 counter wrapped
    return SW_OK;
}

int sw_sweep_measure(sw_ctx *c, uint64_t n, uint64_t *out) { return sw_sweep_measure_ex(c, n, out, SW_OBS_ALL); }

int sw_sweep_measure_ex(sw_ctx *c, uint64_t n, uint64_t *out, uint32_t what)
{
    if (!c || (!out && n) || (what & ~(uint32_t)SW_OBS_ALL)) return SW_ERR_INVALID_ARG;
    if (!c->have_spins) return fail(c, SW_ERR_STATE, "sw_sweep_measure: no spins");
    if (c->t + n > 0x100000000ull) return fail(c, SW_ERR_STATE, "sw_sweep_measure: sweep counter would pass 2^32");
    if (n == 0) return SW_OK;
    DeviceGuard dg(c);
    const size_t stride = 3 + (size_t)c->q;
    const uint64_t chunk_max = c->rows_cap;              // the ring of rows is part of the context's workspace
    unsigned long long *d_rows = c->d_rows;
    int rc = SW_OK;
    for (uint64_t done = 0; done < n && rc == SW_OK;) {
        const uint64_t m = (n - done < chunk_max) ? n - done : chunk_max;
        if (c->cluster) rc = sweep_cluster(c, m, what, d_rows);
        else {
            cudaError_t e0 = cudaMemsetAsync(d_rows, 0, (size_t)m * stride * 8, c->stream);
            if (e0 != cudaSuccess) rc = cuda_fail(c, e0, "sw_sweep_measure memset");
            for (uint64_t k = 0; k < m && rc == SW_OK; ++k) {
                unsigned long long *row = d_rows + k * stride;
                rc = sweep_once(c, (what & (SW_OBS_CLUSTERS | SW_OBS_LARGEST)) != 0, (c->tiled && (what & SW_OBS_LARGEST)) ? row : nullptr);
                if (rc == SW_OK) rc = enqueue_observe(c, row, (what & SW_OBS_ENERGY) != 0, (what & SW_OBS_MAG) != 0,
                                                      (what & (SW_OBS_CLUSTERS | SW_OBS_LARGEST)) != 0, (what & SW_OBS_LARGEST) != 0, nullptr, true);
            }
        }
        if (rc == SW_OK) {
            cudaError_t e = cudaMemcpyAsync(out + done * stride, d_rows, (size_t)m * stride * 8, cudaMemcpyDeviceToHost, c->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
            if (e != cudaSuccess) rc = cuda_fail(c, e, "sw_sweep_measure copy");
        }
        if (rc == SW_OK) for (uint64_t k = 0; k < m; ++k) fix_row(c, out + (done + k) * stride);
        done += m;
    }
    return rc;
}

int sw_get_rows(sw_ctx *c, int what, uint32_t y0, uint32_t nrows, void *dst)
{
    if (!c || !dst || (uint64_t)y0 + nrows > c->L) return fail(c, SW_ERR_INVALID_ARG, "sw_get_rows: bad argument");
    if (nrows == 0) return SW_OK;
    DeviceGuard dg(c);
    const uint64_t first = (uint64_t)y0 * c->L, count = (uint64_t)nrows * c->L;
    if (what == 0) {
        if (!c->have_spins) return fail(c, SW_ERR_STATE, "no spins");
        SW_CUDA(c, cudaMemcpyAsync(dst, c->d_spins + first, count, cudaMemcpyDeviceToHost, c->stream));
    } else if (what == 1) {
        if (!c->have_labels) return fail(c, SW_ERR_STATE, "no labels: no sweep since sw_init");
        const int rc = ensure_flat(c);
        if (rc != SW_OK) return rc;
        SW_CUDA(c, cudaMemcpyAsync(dst, c->d_labels + first, count * 4, cudaMemcpyDeviceToHost, c->stream));
    } else if (what == 2) {
        if (!c->have_labels) return fail(c, SW_ERR_STATE, "no bonds: no sweep since sw_init");
        const uint64_t chunk = c->stage_bytes;           // staging buffer owned by the context
        uint8_t *tmp = c->d_stage;
        for (uint64_t done = 0; done < count;) {
            const uint64_t m = (count - done < chunk) ? count - done : chunk;
            c->launches += 1;
            sw::k_expand_bonds<<<grid_for(c, m, 256), 256, 0, c->stream>>>(c->d_bonds, tmp, first + done, m);
            cudaError_t e = cudaMemcpyAsync((uint8_t *)dst + done, tmp, m, cudaMemcpyDeviceToHost, c->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "sw_get_bonds copy");
            done += m;
        }
    } else return fail(c, SW_ERR_INVALID_ARG, "sw_get_rows: unknown array");
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    return SW_OK;
}

int sw_get_spins(sw_ctx *c, uint8_t *dst) { return c ? sw_get_rows(c, 0, 0, c->L, dst) : SW_ERR_INVALID_ARG; }
int sw_get_labels(sw_ctx *c, uint32_t *dst) { return c ? sw_get_rows(c, 1, 0, c->L, dst) : SW_ERR_INVALID_ARG; }
int sw_get_bonds(sw_ctx *c, uint8_t *dst) { return c ? sw_get_rows(c, 2, 0, c->L, dst) : SW_ERR_INVALID_ARG; }

int sw_get_threshold(sw_ctx *c, uint64_t *T)
{
    if (!c || !T) return SW_ERR_INVALID_ARG;
    *T = c->T;
    return SW_OK;
}

int sw_get_time(sw_ctx *c, uint64_t *t)
{
    if (!c || !t) return SW_ERR_INVALID_ARG;
    *t = c->t;
    return SW_OK;
}

int sw_synchronize(sw_ctx *c)
{
    if (!c) return SW_ERR_INVALID_ARG;
    DeviceGuard dg(c);
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    SW_CUDA(c, cudaGetLastError());
    return SW_OK;
}

int sw_get_stats(sw_ctx *c, sw_stats *out)
{
    if (!c || !out) return SW_ERR_INVALID_ARG;
    out->path = c->cluster ? 2u : c->tiled ? 1u : 0u;
    out->tile_w = out->tile_h = c->tiled ? sw::kTile : 0u;
    out->kernels_per_sweep = c->cluster ? 0u : c->tiled ? 3u : c->label_equiv ? (uint32_t)(3u + 2u * c->le_rounds_last) : (c->lazy ? 4u : 5u);
    out->kernel_launches = c->launches;
    out->device_bytes = c->ws_bytes + (c->owns_sizes ? c->N * 4 : 0);
    out->sweeps = c->sweeps;
    out->le_rounds_last = c->le_rounds_last;
    out->le_rounds_total = c->le_rounds_total;
    out->merge_links = out->merge_retries = out->merge_hops = out->chase_hops = 0;
    out->max_merge_depth = out->max_chase_depth = 0;
    if (c->count_passes) {
        DeviceGuard dg(c);
        sw::PassCounters pc;
        SW_CUDA(c, cudaMemcpyAsync(&pc, c->d_counters, sizeof(pc), cudaMemcpyDeviceToHost, c->stream));
        SW_CUDA(c, cudaStreamSynchronize(c->stream));
        out->merge_links = pc.merge_links; out->merge_retries = pc.merge_retries; out->merge_hops = pc.merge_hops;
        out->chase_hops = pc.chase_hops; out->max_merge_depth = pc.max_merge_depth; out->max_chase_depth = pc.max_chase_depth;
    }
    // algorithmic bytes the sweeps so far had to move (spins R + W, bond bits W, label passes)
    out->bytes_moved = (uint64_t)((double)c->sweeps * (double)c->N * (c->tiled ? (c->lazy ? 10.5 : 14.5) : 0.0));
    return SW_OK;
}

int sw_profile_begin(sw_ctx *c)
{
    if (!c) return SW_ERR_INVALID_ARG;
    for (auto &ev : c->events) { c->event_pool.push_back(ev.a); c->event_pool.push_back(ev.b); }
    c->events.clear();
    c->profiling = true;
    return SW_OK;
}

int sw_profile_end(sw_ctx *c, double ms_per_slot[SW_MAX_KERNEL_SLOTS], uint64_t launches_per_slot[SW_MAX_KERNEL_SLOTS])
{
    if (!c || !ms_per_slot || !launches_per_slot) return SW_ERR_INVALID_ARG;
    c->profiling = false;
    DeviceGuard dg(c);
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int s = 0; s < SW_MAX_KERNEL_SLOTS; ++s) { ms_per_slot[s] = 0.0; launches_per_slot[s] = 0; }
    c->series.clear();
    for (size_t i = 0; i < c->events.size();) {          // per sweep: first kernel's start to last kernel's end
        size_t j = i;
        while (j + 1 < c->events.size() && c->events[j + 1].sweep == c->events[i].sweep) ++j;
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, c->events[i].a, c->events[j].b) == cudaSuccess) c->series.push_back(ms);
        i = j + 1;
    }
    for (auto &ev : c->events) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, ev.a, ev.b) == cudaSuccess) { ms_per_slot[ev.slot] += ms; launches_per_slot[ev.slot] += 1; }
        c->event_pool.push_back(ev.a); c->event_pool.push_back(ev.b);
    }
    c->events.clear();
    return SW_OK;
}

int sw_profile_series(sw_ctx *c, double *ms_per_sweep, uint64_t cap, uint64_t *n)
{
    if (!c || !n || (!ms_per_sweep && cap)) return SW_ERR_INVALID_ARG;
    *n = c->series.size();
    for (uint64_t i = 0; i < cap && i < c->series.size(); ++i) ms_per_sweep[i] = c->series[i];
    return SW_OK;
}

const char *sw_kernel_name(sw_ctx *c, int slot)
{
    if (!c || slot < 0 || slot >= SW_MAX_KERNEL_SLOTS) return nullptr;
    if (c->cluster) return slot == SLOT_TILE ? "k_cluster_sweeps" : nullptr;
    const bool tiled_slot = slot <= SLOT_FLIP;
    if (tiled_slot != c->tiled) return nullptr;
    if (slot == SLOT_G_FLATTEN && c->lazy) return nullptr;
    if (c->label_equiv && slot == SLOT_G_UNION) return "k_le_scan";         // all rounds of a sweep accumulate in these two slots
    if (c->label_equiv && slot == SLOT_G_FLATTEN) return "k_le_analysis";
    return kSlotNames[slot];
}

const char *sw_last_error(const sw_ctx *c) { return c ? c->err.c_str() : "null context"; }

}  // extern "C"

// the super-lattice decomposition: same translation unit, its own context type
#include "sw_super.cuh"

// the embedded-cluster XY extension
#include "sw_xy.cuh"
