/*
 * sw.h -- C ABI of libsw.so: Swendsen-Wang multi-cluster sweeps of the 2D q-state
 * Potts model on one NVIDIA B200 (sm_100a).
 *
 * The method (Komura & Okabe, arXiv:1208.2080; line numbers refer to PAPER.md):
 *   H = -J sum_<ij> delta(S_i, S_j) on an L x L periodic square lattice   PAPER.md:33-38 (eq. 1 up to a constant)
 *   one sweep =  (1) activate each bond between EQUAL neighbours with p = 1 - exp(-K)
 *                (2) label the connected components of the active-bond graph
 *                (3) give every cluster a fresh uniform state in 0..q-1
 *   the label of a cluster is the smallest site index in it
 *
 * Determinism (BASELINE.json north_star; field layout frozen in DESIGN.md, reading R11):
 *   every draw is Philox4x32-10 with key = (seed lo, seed hi) and counter
 *   (idx lo, idx hi, sweep t, purpose); purpose 0 = INIT (idx = site), 1 = BOND
 *   (idx = site >> 1; words 2(site&1), 2(site&1)+1 = right, down bond), 2 = FLIP
 *   (idx = canonical root).  A bond is active iff draw < T = floor(p * 2^32).
 *   New state = floor(draw * q / 2^32).  The result of a sweep is therefore a pure
 *   function of (spins, L, q, K, seed, t) and does not depend on scheduling.
 *
 * Conventions
 *   site i = y*L + x (x fastest); right(i) = y*L + (x+1)%L; down(i) = ((y+1)%L)*L + x.
 *   spins: uint8, 0..q-1.  labels: uint32 canonical root (minimum site index of the cluster).
 *   bonds (sw_get_bonds): one byte per site, bit0 = right bond active, bit1 = down bond active.
 *   All `dst` / `src` / out pointers are HOST memory owned by the caller and sized as annotated;
 *   device memory is owned by the context (or by the caller of sw_create_ws, who lends it).
 *   Every call returns a status code; nothing throws or aborts.  Calls on one context must
 *   not be made concurrently from several threads.
 *   sw_sweep is asynchronous on the context's CUDA stream; every call that returns data to
 *   the host synchronises that stream first.
 */
#ifndef SW_H
#define SW_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sw_ctx sw_ctx;   /* opaque; freed only by sw_destroy */

enum {
    SW_OK = 0,
    SW_ERR_INVALID_ARG = 1,     /* NULL pointer, L/q/K out of range, spin >= q, ...        */
    SW_ERR_OOM = 2,             /* device or host allocation failed / workspace too small  */
    SW_ERR_CUDA = 3,            /* a CUDA runtime call failed (no device, launch error)    */
    SW_ERR_STATE = 4            /* call not valid in the current state (see each call)     */
};
enum { SW_INIT_ORDERED = 0, SW_INIT_RANDOM = 1 };

/* Creation flags (sw_create_ex / sw_create_ws). */
enum {
    SW_FLAG_DEFAULT       = 0,
    SW_FLAG_FORCE_GENERIC = 1,  /* use the any-L reference kernels even where the tiled path applies     */
    SW_FLAG_LAZY_LABELS   = 2,  /* do not materialise canonical labels every sweep; flatten on demand
                                   (sw_get_labels / sw_measure of cluster sizes).  Same results.        */
    SW_FLAG_LABEL_EQUIVALENCE = 4,/* comparison variant, any L: label step (2) with the "Label Equivalence" scheme
                                   the paper uses (scanning + analysis kernels iterated until the
                                   scanning changes nothing; the host reads a flag every round, so in this mode
                                   sw_sweep is SYNCHRONOUS).  Same results, much slower; sw_stats.le_rounds_*
                                   count the rounds (the paper: about 8.6).                                     */
    SW_FLAG_WS_CLUSTER_SIZES = 8, /* make the 4*L*L-byte scratch of sw_measure(largest_cluster) part of the
                                   workspace (sw_workspace_bytes grows by it).  Without the flag the library
                                   allocates that scratch itself, once, on the first call that needs it, and
                                   keeps it until sw_destroy (sw_stats.device_bytes counts it).  Everything
                                   else the library ever touches on the device lies inside the workspace.      */
    SW_FLAG_PASS_COUNTERS = 16,   /* count the passes actually taken (sw_stats.merge_*, chase_*): instantiations of
                                   the merge and flatten kernels with counters; off by default (a few per cent)  */
    SW_FLAG_NO_CLUSTER_PATH = 32  /* lattices of at most 16 tiles (L <= 256, L % 64 == 0) run all the sweeps of a
                                   call in ONE launch of a persistent kernel whose CTAs form one thread-block
                                   cluster (sw_stats.path == 2); this flag keeps them on the three-kernels-per-
                                   sweep path.  Same results.                                                   */
};

/* --- life cycle -------------------------------------------------------------------------------
 * sw_create: "q-state Potts model ... periodic boundary conditions", one context
 * per lattice.  2 <= L <= 65536 (L*L <= 2^32 so that a uint32 label can name every site), 2 <= q
 * <= 255, K = J/k_B T >= 0 or +inf; NaN or negative K -> SW_ERR_INVALID_ARG.  The library
 * allocates its own device memory on the current device and creates its own stream.            */
int sw_create(sw_ctx **out, uint32_t L, uint32_t q, double K, uint64_t seed);
int sw_create_ex(sw_ctx **out, uint32_t L, uint32_t q, double K, uint64_t seed, uint32_t flags);

/* Device memory and stream lent by the caller (PyTorch in the Python binding).  `dev_ws` must be
 * a device pointer aligned to 256 bytes with at least sw_workspace_bytes(L, q, flags) bytes and
 * must outlive the context; `cuda_stream` is a cudaStream_t (NULL = the legacy default stream).
 * The workspace holds everything: lattice arrays, the row ring of sw_sweep_measure, the staging
 * buffer of sw_get_bonds (see SW_FLAG_WS_CLUSTER_SIZES for the one optional exception).
 * Every call on a context runs on the device it was created on (the library switches to it and
 * back), so contexts on several devices can be driven from one thread.                          */
size_t sw_workspace_bytes(uint32_t L, uint32_t q, uint32_t flags);
int sw_create_ws(sw_ctx **out, uint32_t L, uint32_t q, double K, uint64_t seed, uint32_t flags,
                 void *dev_ws, size_t ws_bytes, void *cuda_stream);
/* Frees the context and the device memory the library allocated (a lent workspace stays the caller's); waits for the
 * context's stream first.  NULL is allowed.  (BASELINE.json north_star lists sw_destroy among the seven calls.)     */
void sw_destroy(sw_ctx *ctx);

/* --- state ------------------------------------------------------------------------------------
 * sw_init: ORDERED = all spins 0; RANDOM = spin_i = floor(Philox(INIT, i).w0 * q / 2^32).
 * Sets t = 0 and forgets the labels.  (S_i in 1..q in PAPER.md:35 is stored as 0..q-1.)         */
int sw_init(sw_ctx *ctx, int mode);
/* Load a spin configuration and the sweep counter: (spins, t) is the complete state of the
 * chain, so this is checkpoint/resume.  src: host uint8[L*L], every value < q else
 * SW_ERR_INVALID_ARG (checked on the device); t <= 2^32 - 1.                                     */
int sw_set_state(sw_ctx *ctx, const uint8_t *src, uint64_t t);

/* The same state in packed form: `bits` in {1, 2, 4, 8} bits per spin with q <= 2^bits; site i occupies bits
 * [bits (i % per), bits (i % per + 1)) of byte i / per, per = 8 / bits (little-endian inside the byte); L*L must be a
 * multiple of 16.  A q = 2 lattice of 2^32 sites is 512 MiB instead of 4 GiB: the form to move a checkpoint over PCIe.
 * src / dst: host, L*L*bits/8 bytes.  sw_set_state_packed validates every value (< q) like sw_set_state.            */
int sw_set_state_packed(sw_ctx *ctx, const void *src, uint32_t bits, uint64_t t);
int sw_get_spins_packed(sw_ctx *ctx, void *dst, uint32_t bits);

/* --- the hot path -----------------------------------------------------------------------------
 * sw_sweep: n full sweeps (PAPER.md:40 steps 1-3), asynchronous on the context stream.
 * SW_ERR_STATE before sw_init/sw_set_state, or if t + n would pass 2^32 (the sweep field of the
 * Philox counter is 32 bits).                                                                    */
int sw_sweep(sw_ctx *ctx, uint64_t n);

/* sw_measure: observables of the current state ("measurement of energy and
 * magnetization"; cluster statistics from BASELINE.json config 4).  Synchronises.
 *   energy_bonds    = #{nearest-neighbour pairs with equal spins}, each bond once, 0..2N
 *                     (E = -J*energy_bonds for H = -J sum delta; eq. 1 subtracts 2N)
 *   mag_counts[s]   = #{i : spin_i = s}, s = 0..q-1           (host uint64[q])
 *   n_clusters      = #{clusters} and largest_cluster = max cluster size of the bond
 *                     configuration drawn in the LAST sweep; both 0 if no sweep since sw_init.
 * Any out pointer may be NULL ("not wanted"); what is not wanted is not computed.               */
int sw_measure(sw_ctx *ctx, uint64_t *energy_bonds, uint64_t *mag_counts,
               uint64_t *n_clusters, uint64_t *largest_cluster);

/* Cluster statistics of the LAST sweep with the second moment of the size distribution: sum_sq[0] + 2^64 sum_sq[1] =
 * sum over clusters of |c|^2 (a device reduction over the cluster sizes).  It is the improved (cluster) estimator of the
 * magnetisation's second moment: q <sum_s n_s^2> - N^2 = (q - 1) <sum_c |c|^2>, the quantity behind the moment-ratio
 * check of PAPER.md:90.  n_clusters / largest_cluster may be NULL.  SW_ERR_STATE if no sweep since sw_init.          */
int sw_measure_clusters(sw_ctx *ctx, uint64_t *n_clusters, uint64_t *largest_cluster, uint64_t sum_sq[2]);

/* n x (one sweep, one measurement) without a host round trip per sweep; row k of `out`
 * (host uint64[n][3+q]) = energy_bonds, n_clusters, largest_cluster, mag_counts[0..q-1]
 * after sweep k.  Synchronises once at the end.                                                  */
int sw_sweep_measure(sw_ctx *ctx, uint64_t n, uint64_t *out);
/* The same with a choice of observables (BASELINE.json configs 3 and 4 want two of them each); columns that
 * are not wanted are 0.  SW_OBS_LARGEST implies the cluster count.                                           */
enum { SW_OBS_ENERGY = 1, SW_OBS_MAG = 2, SW_OBS_CLUSTERS = 4, SW_OBS_LARGEST = 8, SW_OBS_ALL = 15 };
int sw_sweep_measure_ex(sw_ctx *ctx, uint64_t n, uint64_t *out, uint32_t what);

/* --- read-back (all synchronise) ---------------------------------------------------------------*/
/* The spins S_i of PAPER.md:35 (stored 0..q-1), site i = y*L + x: the state of the chain after the last sweep (or as
 * set by sw_init / sw_set_state).  SW_ERR_STATE before any of those.                                                */
int sw_get_spins(sw_ctx *ctx, uint8_t *dst /* host [L*L] */);
/* canonical roots of the LAST sweep; SW_ERR_STATE if there was none since sw_init */
int sw_get_labels(sw_ctx *ctx, uint32_t *dst /* host [L*L] */);
/* bonds of the LAST sweep, one byte per site (bit0 right, bit1 down); SW_ERR_STATE as above      */
int sw_get_bonds(sw_ctx *ctx, uint8_t *dst /* host [L*L] */);
/* rows y0 .. y0+nrows-1 only of the same three arrays (spins PAPER.md:35, labels PAPER.md:42, bonds PAPER.md:40 step
 * 1), for sampling a lattice too large to copy whole (2^32 sites: SURVEY.md sec. 8 c-6); what: 0 = spins (uint8),
 * 1 = labels (uint32), 2 = bonds (uint8); dst: host, nrows*L elements; y0 + nrows <= L else SW_ERR_INVALID_ARG       */
int sw_get_rows(sw_ctx *ctx, int what, uint32_t y0, uint32_t nrows, void *dst);
int sw_get_threshold(sw_ctx *ctx, uint64_t *T);    /* floor((1-exp(-K)) * 2^32), 0..2^32          */
int sw_get_time(sw_ctx *ctx, uint64_t *t);         /* sweeps done since sw_init (or set_state's t) */
int sw_synchronize(sw_ctx *ctx);                   /* wait for the context stream                  */

/* --- introspection ------------------------------------------------------------------------------*/
typedef struct sw_stats {
    uint32_t path;              /* 0 = generic kernels, 1 = tiled path, 2 = tiled path as one persistent cluster kernel */
    uint32_t tile_w, tile_h;    /* tile shape of the tiled path                                     */
    uint32_t kernels_per_sweep; /* kernel launches one sweep issues (0 on path 2: one launch per call)    */
    uint64_t kernel_launches;   /* kernels launched by this context so far                          */
    uint64_t device_bytes;      /* device memory in use by this context                             */
    uint64_t sweeps;            /* sweeps issued so far                                             */
    uint64_t le_rounds_last;    /* SW_FLAG_LABEL_EQUIVALENCE: scanning + analysis rounds of the last sweep,   */
    uint64_t le_rounds_total;   /* ... and of all sweeps so far (the last round of a sweep changes nothing)   */
    /* passes actually taken by the labeling (SW_FLAG_PASS_COUNTERS, tiled path; else 0), summed over all sweeps:
     * the border merge (PAPER.md:66-68 one level down) is ONE pass whose cost is its find chains and lost races;
     * the flatten ("tracks back the label variable until [it] remains unchanged") is one chase per
     * tile-local root                                                                                          */
    uint64_t merge_links;       /* border links united (after the duplicate filter)                          */
    uint64_t merge_retries;     /* hooks that lost the race for a root and carried on                        */
    uint64_t merge_hops;        /* parent loads of all finds of the merge                                    */
    uint64_t chase_hops;        /* parent loads of all root chases of the flatten                            */
    uint32_t max_merge_depth;   /* longest single find of the merge, in hops                                 */
    uint32_t max_chase_depth;   /* longest single root chase of the flatten, in hops                         */
    uint64_t bytes_moved;       /* algorithmic bytes of all sweeps so far: 14.5 B/site/sweep on the tiled path
                                   (spins R+W 2, bond bits W+R 0.5, labels W, R, W 12),
                                   10.5 with SW_FLAG_LAZY_LABELS; 0 on the generic path                       */
} sw_stats;
int sw_get_stats(sw_ctx *ctx, sw_stats *out);
/* Time the kernels of the NEXT sweeps individually with CUDA events on the context stream:
 * after sw_profile_begin, each sw_sweep(n) records per-kernel events; sw_profile_end synchronises
 * and returns the accumulated milliseconds per kernel slot (see sw_kernel_name).                  */
#define SW_MAX_KERNEL_SLOTS 8
int sw_profile_begin(sw_ctx *ctx);
int sw_profile_end(sw_ctx *ctx, double ms_per_slot[SW_MAX_KERNEL_SLOTS], uint64_t launches_per_slot[SW_MAX_KERNEL_SLOTS]);
/* Per-sweep device time of the region closed by the last sw_profile_end (first kernel's start to last kernel's
 * end of each sweep, milliseconds): the time series SURVEY.md sec. 8(d) asks for.  *n = sweeps recorded; at most
 * `cap` values are written.                                                                                      */
int sw_profile_series(sw_ctx *ctx, double *ms_per_sweep, uint64_t cap, uint64_t *n);
const char *sw_kernel_name(sw_ctx *ctx, int slot); /* NULL if the slot is unused                   */
const char *sw_last_error(const sw_ctx *ctx);      /* text of the last failure on this context     */
const char *sw_version(void);

/* --- the super-lattice decomposition ---------------------------------------------------------
 * The L x L lattice cut into gx x gy equal sub-lattices ("each GPU has the information of spins ... of a sub-lattice",
 * PAPER.md:62), one per entry of `devices` (piece (px, py) = devices[py * gx + px]; NULL = the current device for
 * all; several pieces may share a device).  Labeling is two-stage: inside each piece, then between
 * pieces over the boundary sites only; label values are global site indices, the new state of a cluster comes from the
 * Philox key of its canonical root, so bonds, labels, spins and observables are IDENTICAL to those of sw_create with
 * the same (L, q, K, seed) -- the calls below mirror sw_init / sw_set_state / sw_sweep / sw_measure / sw_get_*, with
 * host arrays in the layout of the whole lattice (site i = y*L + x).
 * L % (64 gx) == 0 and L % (64 gy) == 0, gx*gy <= 64, 64 <= L <= 65536; devices that differ must have peer access
 * (NVLink): the bond kernel reads its neighbours' boundary spins and the inter-piece merge hooks roots with
 * system-scope atomicMin directly in the owner's memory, so the link must support native atomics
 * (cudaDevP2PAttrNativeAtomicSupported; PCIe-only peer access does not): otherwise SW_ERR_CUDA, and
 * sw_super_last_error(NULL) gives the reason of the calling thread's last failed creation.
 * Device memory is owned by the library.                                                                          */
typedef struct sw_super sw_super;
int  sw_create_super(sw_super **out, uint32_t L, uint32_t q, double K, uint64_t seed,
                     uint32_t gx, uint32_t gy, const int *devices /* [gx*gy] or NULL */);
void sw_super_destroy(sw_super *s);
int  sw_super_init(sw_super *s, int mode);
int  sw_super_set_state(sw_super *s, const uint8_t *src /* host [L*L] */, uint64_t t);
int  sw_super_sweep(sw_super *s, uint64_t n);                 /* asynchronous on the pieces' streams */
int  sw_super_measure(sw_super *s, uint64_t *energy_bonds, uint64_t *mag_counts /* [q] */,
                      uint64_t *n_clusters, uint64_t *largest_cluster);
int  sw_super_get_spins(sw_super *s, uint8_t *dst /* host [L*L] */);
int  sw_super_get_labels(sw_super *s, uint32_t *dst /* host [L*L], canonical roots = global site indices */);
int  sw_super_get_bonds(sw_super *s, uint8_t *dst /* host [L*L], bit0 right, bit1 down */);
int  sw_super_get_time(sw_super *s, uint64_t *t);
int  sw_super_synchronize(sw_super *s);
typedef struct sw_super_stats {
    uint32_t gx, gy, piece_w, piece_h;  /* the decomposition                                                      */
    uint32_t devices;                   /* distinct devices in use                                                */
    uint64_t sweeps, kernel_launches, device_bytes;
    uint64_t boundary_sites_per_piece;  /* 2 (W + H): all that stage 2 looks at ("4 N_x")             */
    uint64_t inter_links;               /* active bonds between pieces united by stage 2, all sweeps              */
    uint64_t inter_hops;                /* label loads of stage 2 + resolve (local or over NVLink)                */
    uint64_t inter_retries;             /* hooks that lost the race for a root                                    */
    uint64_t resolved_links;            /* links leaving a piece that the resolve pass re-pointed at the root     */
} sw_super_stats;
int  sw_super_get_stats(sw_super *s, sw_super_stats *out);
const char *sw_super_last_error(const sw_super *s);

/* One process per GPU (the launch the paper uses: one MPI rank per GPU).  Every rank creates a context that
 * OWNS one piece (on its current device) and learns where the other pieces are through CUDA IPC: each rank exports the
 * 64-byte handle of its piece, the ranks exchange them (torch.distributed all_gather in the Python binding) and import
 * the others'.  A sweep is three phases (0: stage 1 inside the piece, 1: stage 2 between pieces, 2: resolve + flatten +
 * flip); the caller calls sw_super_synchronize and a barrier of the process group after each phase -- that barrier is all
 * that is left of the paper's per-round flag exchange.  sw_super_init / _set_state / _get_* act on the
 * local piece (host arrays keep the layout of the whole lattice; only the local piece's part is read / written).
 * A measurement is three phases as well (0: zero, 1: count, 2: maxima and the local partial row [3+q]: all columns are
 * sums over the ranks except column 2, largest_cluster, which is a maximum).                                           */
#define SW_IPC_HANDLE_BYTES 64
int  sw_create_super_rank(sw_super **out, uint32_t L, uint32_t q, double K, uint64_t seed,
                          uint32_t gx, uint32_t gy, uint32_t my_piece);
int  sw_super_ipc_export(sw_super *s, void *handle_out /* host [SW_IPC_HANDLE_BYTES] */);
int  sw_super_ipc_import(sw_super *s, uint32_t piece, const void *handle /* host [SW_IPC_HANDLE_BYTES] */);
/* Tear-down of a rank context, first half: waits for the local stream and unmaps every imported piece.  CUDA IPC requires
 * that an exported allocation is freed only after every importer has closed it, so the ranks call this, THEN pass a barrier
 * of the process group, THEN call sw_super_destroy (which frees the local piece).  Afterwards the context accepts
 * sw_super_destroy only (phases and measurements return SW_ERR_STATE).                                                   */
int  sw_super_ipc_close_all(sw_super *s);
int  sw_super_phase(sw_super *s, int phase /* 0, 1, 2; phase 2 advances the sweep counter */);
int  sw_super_measure_phase(sw_super *s, int phase, uint32_t what /* SW_OBS_* */, uint64_t *part /* host [3+q], phase 2 */);

/* --- the extension the paper names: embedded-cluster sweeps of the 2D classical XY model -----------------
 * H = -J sum_<ij> s_i . s_j with unit vectors s_i; one sweep = the three steps of PAPER.md:40 on the Ising variables
 * embedded by a random direction r (Wolff): a_i = s_i . r; bond <ij> active iff a_i a_j > 0 and
 * draw < floor((1 - exp(-2 K a_i a_j)) 2^32); clusters labeled by their smallest site; a cluster is
 * reflected, s -> s - 2 (s . r) r, iff floor(FLIP draw of its root * 2 / 2^32) == 1.  Draws: the Potts layout (BOND,
 * FLIP, INIT) plus purpose 3 REFLECT (idx 0, sweep t, word 0): the angle of r is 2 pi (w0 + 1/2) / 2^32.
 * Spins are double[L*L][2] (x, y); all arithmetic is IEEE double with explicit roundings (X1-X6), any L >= 2.
 * sw_xy_init: ORDERED = all spins (1, 0); RANDOM = a point of (-1, 1)^2 from two INIT words (the other two if it lies
 * outside the unit disc), normalised.  energy_sum = sum over bonds of s_i . s_j (E = -J energy_sum); mag = sum of spins;
 * cluster statistics describe the bonds of the last sweep.  Device memory is owned by the library; all calls return a
 * status; sw_xy_sweep is asynchronous on the context's stream, the read-backs synchronise.                              */
typedef struct sw_xy sw_xy;
int  sw_xy_create(sw_xy **out, uint32_t L, double K, uint64_t seed);
void sw_xy_destroy(sw_xy *c);
int  sw_xy_init(sw_xy *c, int mode);
int  sw_xy_set_state(sw_xy *c, const double *spins /* host [L*L][2], finite */, uint64_t t);
int  sw_xy_sweep(sw_xy *c, uint64_t n);
int  sw_xy_measure(sw_xy *c, double *energy_sum, double mag[2], uint64_t *n_clusters, uint64_t *largest_cluster);
int  sw_xy_get_spins(sw_xy *c, double *dst /* host [L*L][2] */);
int  sw_xy_get_labels(sw_xy *c, uint32_t *dst /* host [L*L] */);
int  sw_xy_get_bonds(sw_xy *c, uint8_t *dst /* host [L*L], bit0 right, bit1 down */);
int  sw_xy_get_reflection(sw_xy *c, double r[2]);  /* the direction r of the last sweep */
int  sw_xy_get_time(sw_xy *c, uint64_t *t);
const char *sw_xy_last_error(const sw_xy *c);

/* --- cluster statistics without any device allocation ----------------------------------------------------------------
 * Who this is for.  sw_measure(largest_cluster) and sw_measure_clusters keep one uint32 counter per site, 4*L*L bytes,
 * which the library cudaMalloc's the first time it is needed (or takes from the workspace, SW_FLAG_WS_CLUSTER_SIZES).
 * Some programs cannot let a library do that: every byte of the GPU already belongs to the program's own memory pool, so
 * a cudaMalloc made behind its back fails or shrinks what the pool counted on; or the call sits inside a sweep loop that
 * cannot stop for the device-wide synchronisation an allocation brings with it; or the memory budget of the job was
 * fixed when the library was loaded and must not move afterwards.  sw_cluster_stats_static is the counting pass of
 * PAPER.md:42 / BASELINE.json config 4 (sites per cluster, keyed by the cluster's smallest site) for those callers: its
 * counters live in an array that is compiled into libsw.so (static __device__, SW_STATIC_MAX_SITES uint32 = 4 MiB on
 * every GPU that loads the library, held until the process exits), and the call itself allocates and frees nothing, on
 * the device or on the host.
 *
 *   dev_labels  DEVICE uint32[n_sites], on the current device: canonical labels, labels[i] = smallest site of i's
 *               cluster (what sw_get_labels returns), owned by the caller, only read
 *   n_sites     0 .. SW_STATIC_MAX_SITES (L <= 1024); anything larger -> SW_ERR_INVALID_ARG, nothing is launched and
 *               sw_static_last_error() says so: larger lattices have to go through sw_measure_clusters
 *   dev_out     DEVICE uint64[4], on the current device, owned by the caller, overwritten:
 *               [0] number of clusters, [1] size of the largest, [2] sum over clusters of size^2 (< 2^64 at this size),
 *               [3] number of sites whose label is not a canonical root of this lattice (>= n_sites, or
 *               labels[label] != label); such sites are left out of [0..2], so [3] != 0 means "bad input"
 *   cuda_stream cudaStream_t of the current device (NULL = the legacy default stream); three small kernels are enqueued
 *               on it and the call returns without waiting.  Read dev_out after synchronising that stream.
 *
 * Shared scratch.  There is ONE array per GPU and every call on that GPU uses it.  A call clears the part it needs
 * before counting, so nothing survives from the call before (whose counts stay in the array until then); but two calls
 * whose kernels can run at the same time on one GPU -- different streams, different host threads, different contexts
 * of this process -- count into the same words and both results are garbage.  Keep calls on one GPU in one stream, or
 * order them with events.
 * First call on a device.  The array's device address is looked up once per device (cudaGetSymbolAddress, with that
 * device current) by the first call made there, which may also make the runtime load the library's kernels.  Make that
 * first call during start-up, before any stream capture is begun.
 * Errors.  SW_ERR_INVALID_ARG (NULL, n_sites too large, a pointer that is not memory of the current device) or
 * SW_ERR_CUDA; sw_static_last_error() returns the reason of the calling thread's last failure ("" after a success).  */
#define SW_STATIC_MAX_SITES (1u << 20)
int sw_cluster_stats_static(const uint32_t *dev_labels, uint64_t n_sites, uint64_t *dev_out, void *cuda_stream);
uint64_t sw_static_max_sites(void);            /* SW_STATIC_MAX_SITES, for callers that bind at run time */
const char *sw_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
