// sw_common.cuh -- device-side building blocks shared by the kernels of libsw.so.
//
// Philox4x32-10 (Salmon et al., SC'11) with the ten round keys precomputed on the host,
// the draw layout of include/sw.h (reading R11), and the lock-free union-find
// primitives on a uint32 parent array (canonical root = minimum index).
//
// Product code: shares nothing with oracle/.
#pragma once

#include <cstdint>
#include <cuda_runtime.h>

namespace sw {

constexpr uint32_t kPurposeInit = 0u, kPurposeBond = 1u, kPurposeFlip = 2u;

// Kernel-parameter block: lives in the constant bank, so the round keys cost no registers.
struct Params {
    uint32_t rk0[10];     // k0 + r * 0x9E3779B9
    uint32_t rk1[10];     // k1 + r * 0xBB67AE85
    uint32_t L;           // linear size
    uint32_t q;           // number of Potts states
    uint32_t t;           // sweep counter (Philox counter word 2)
    uint32_t thr_m1;      // T - 1 (valid when thr_any != 0): bond active iff draw <= thr_m1
    uint32_t thr_any;     // 0 if T == 0 (no bond can be active), else 0xFFFFFFFF
    uint32_t log2L;       // log2(L) if L is a power of two, else 0xFFFFFFFF
    uint64_t N;           // L * L (up to 2^32)
    uint64_t divL_magic;  // ceil(2^40 / L): (d * magic) >> 40 == d / L for d < 2^24 (L <= 2^16)
    uint32_t pk_t[3];     // philox_sweep constants of sweep t (see there), and ...
    uint32_t pk_n[3];     // ... of sweep t + 1 (the flip kernel makes the next sweep's bond draws)
};

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const Params &P)
{
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        c0 = hi1 ^ c1 ^ P.rk0[r];
        c1 = lo1;
        c2 = hi0 ^ c3 ^ P.rk1[r];
        c3 = lo0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// Philox4x32-10 for the draws of a sweep: counter (idx, 0, t, purpose) with idx < 2^32.  Counter words 1 and 2 are the
// same for every thread, so the halves of rounds 0 and 1 that only depend on them are computed once per sweep on the
// host (sweep_keys in sw_api.cu): k[0] = lo(M1 t) ^ rk0[1], k[1] = hi(M0 A0) ^ rk1[1], k[2] = lo(M0 A0) with
// A0 = hi(M1 t) ^ rk0[0].  Bit for bit the same function as philox4x32_10(idx, 0, t, purpose): 37 instead of 40
// multiply / xor instructions per call.
__device__ __forceinline__ uint4 philox_sweep(uint32_t idx, uint32_t purpose, const uint32_t (&k)[3], const Params &P)
{
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    uint32_t c2 = __umulhi(M0, idx) ^ purpose ^ P.rk1[0], c3 = M0 * idx;             // round 0
    uint32_t c0 = __umulhi(M1, c2) ^ k[0], c1 = M1 * c2;                             // round 1
    c2 = c3 ^ k[1];
    c3 = k[2];
#pragma unroll
    for (int r = 2; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        c0 = hi1 ^ c1 ^ P.rk0[r];
        c1 = lo1;
        c2 = hi0 ^ c3 ^ P.rk1[r];
        c3 = lo0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// floor(w * q / 2^32): the draw -> state map (R9)
__device__ __forceinline__ uint32_t state_from_draw(uint32_t w, uint32_t q) { return __umulhi(w, q); }

__device__ __forceinline__ uint32_t flip_state(uint32_t root, const uint32_t (&pk_t)[3], const Params &P)
{
    return state_from_draw(philox_sweep(root, kPurposeFlip, pk_t, P).x, P.q);
}
__device__ __forceinline__ uint32_t flip_state(uint32_t root, const Params &P) { return flip_state(root, P.pk_t, P); }

// the per-sweep halves of Philox rounds 0 and 1 (see philox_sweep): on the host once per launch, or on the device
// by the persistent kernel that runs many sweeps in one launch
__host__ __device__ __forceinline__ void sweep_keys(const Params &P, uint32_t t, uint32_t (&k)[3])
{
    const uint64_t m1t = 0xCD9E8D57ull * t;
    const uint32_t a0 = (uint32_t)(m1t >> 32) ^ P.rk0[0], a1 = (uint32_t)m1t;
    const uint64_t m0a = 0xD2511F53ull * a0;
    k[0] = a1 ^ P.rk0[1];
    k[1] = (uint32_t)(m0a >> 32) ^ P.rk1[1];
    k[2] = (uint32_t)m0a;
}

// Data another CTA wrote earlier in the SAME launch (the persistent cluster kernel, sw_cluster.cuh; the neighbour
// pieces of the super-lattice) must not come through L1 or the non-coherent path: kCoherent loads go to L2.
template <bool kCoherent, class T>
__device__ __forceinline__ T ld_in(const T *p) { return kCoherent ? __ldcg(p) : *p; }

// ---- where a piece of the lattice lives ----------------------------------------------------------
// The kernels of the tiled path work on one rectangular piece of the lattice held in one set of arrays:
// the whole L x L lattice (one context, the default), or one sub-lattice of the super-lattice
// decomposition ("each GPU has the information of spins ... of a sub-lattice"; sw_super.cu).
// Label VALUES and Philox keys are always global site indices gy * Lg + gx (the label of a
// cluster is its smallest site); array ADDRESSES are local, ly * W + lx.  For the whole lattice the two
// coincide and the kernels are instantiated with kSuper = false (none of this is touched).
struct Dom {
    uint32_t W, H;          // sites per row / rows of this piece (multiples of 64)
    uint32_t Lg, log2Lg;    // global lattice size; log2 if a power of two, else 0xFFFFFFFF
    uint32_t ox, oy;        // global coordinates of the first site of the piece
    const uint8_t *right;   // spins of the piece on the right (its column 0 continues my rows; same H): "boundary layers"
    const uint8_t *down;    // spins of the piece below (its row 0 continues my columns; same W)
    uint32_t right_W;       // row stride of `right`
    uint32_t me;            // index of this piece in the super-lattice (owner id)
};

// label value -> local array offset
struct FlatAddr {
    __device__ __forceinline__ uint32_t operator()(uint32_t g) const { return g; }
};
struct DomAddr {
    uint32_t Lg, log2Lg, ox, oy, W, H;
    __device__ __forceinline__ DomAddr(const Dom &d) : Lg(d.Lg), log2Lg(d.log2Lg), ox(d.ox), oy(d.oy), W(d.W), H(d.H) {}
    __device__ __forceinline__ void split(uint32_t g, uint32_t &gx, uint32_t &gy) const
    {
        if (log2Lg != 0xFFFFFFFFu) { gy = g >> log2Lg; gx = g & (Lg - 1u); } else { gy = g / Lg; gx = g - gy * Lg; }
    }
    __device__ __forceinline__ bool mine(uint32_t g) const { uint32_t gx, gy; split(g, gx, gy); return gx - ox < W && gy - oy < H; }
    __device__ __forceinline__ uint32_t operator()(uint32_t g) const { uint32_t gx, gy; split(g, gx, gy); return (gy - oy) * W + (gx - ox); }
};

// ---- union-find on global memory -------------------------------------------------------------
// labels[] is a forest whose links always point to a smaller index.  Loads bypass L1 (other
// SMs update the array concurrently); a stale value is still an ancestor, so chases stay valid.
// `A` maps a label value to its array offset (FlatAddr: the identity).

template <class A = FlatAddr>
__device__ __forceinline__ uint32_t ld_label(const uint32_t *labels, uint32_t i, const A &addr = A())
{
    return __ldcg(labels + addr(i));
}

template <class A = FlatAddr>
__device__ __forceinline__ uint32_t find_root(const uint32_t *labels, uint32_t a, const A &addr = A())
{
    uint32_t p = ld_label(labels, a, addr);
    while (p != a) { a = p; p = ld_label(labels, a, addr); }
    return a;
}

// "Passes actually taken" (sw_get_stats): filled by the kStats instantiations of k_tile_merge and
// k_tile_flip when the context was created with SW_FLAG_PASS_COUNTERS; the default kernels carry no counting code.
struct PassCounters {
    unsigned long long merge_links;     // links the border merge united (after the duplicate filter)
    unsigned long long merge_retries;   // hooks that lost the race for a root and carried on from the parent they saw
    unsigned long long merge_hops;      // parent loads of all finds of the border merge
    unsigned long long chase_hops;      // parent loads of the root chases of the flatten (k_tile_flip)
    unsigned int max_merge_depth;       // longest single find of the border merge, in hops
    unsigned int max_chase_depth;       // longest single root chase of the flatten, in hops
};

// find with path halving: every second node on the way is re-pointed at its grandparent.  A link is
// only ever replaced by a link to an ancestor, so this is safe next to concurrent hooks (a hook that
// loses the race sees the old value come back from atomicMin and carries on from there).  The
// re-pointing is itself an atomicMin (a fire-and-forget RED): it can only lower a link, so it can
// never undo a canonical root that k_tile_flip of another tile has already written there.
// The same chase when the caller already holds p = labels[a] (possibly stale: still an ancestor).
// kStats: `hops` counts the parent loads.
template <bool kStats = false, class A = FlatAddr>
__device__ __forceinline__ uint32_t find_root_halving_from(uint32_t *labels, uint32_t a, uint32_t p, uint32_t *hops = nullptr, const A &addr = A())
{
    while (p != a) {
        const uint32_t gp = ld_label(labels, p, addr);
        if (kStats) *hops += 1;
        if (gp == p) return p;
        atomicMin(labels + addr(a), gp);
        a = gp;
        p = ld_label(labels, a, addr);
        if (kStats) *hops += 1;
    }
    return a;
}

template <bool kStats = false, class A = FlatAddr>
__device__ __forceinline__ uint32_t find_root_halving(uint32_t *labels, uint32_t a, uint32_t *hops = nullptr, const A &addr = A())
{
    const uint32_t p = ld_label(labels, a, addr);
    if (kStats) *hops += 1;
    return find_root_halving_from<kStats, A>(labels, a, p, hops, addr);
}

// Join the sets of a and b.  The larger root is hooked under the smaller with atomicMin; if the
// word we hit was no longer a root, the link it held is not lost: we carry on uniting its old
// target with b.  One pass over all bonds yields the complete partition (no outer iteration).
// kStats: st[0] += parent loads, st[1] = max(longest single find), st[2] += lost races.
template <bool kStats = false, class A = FlatAddr>
__device__ __forceinline__ void unite(uint32_t *labels, uint32_t a, uint32_t b, uint32_t *st = nullptr, const A &addr = A())
{
    uint32_t ha = 0, hb = 0;
    {   // the first hop of both chases is loaded together: the common case (both are roots) costs one round trip, not two
        const uint32_t pa = ld_label(labels, a, addr), pb = ld_label(labels, b, addr);
        if (kStats) { ha = 1; hb = 1; }
        a = find_root_halving_from<kStats, A>(labels, a, pa, &ha, addr);
        b = find_root_halving_from<kStats, A>(labels, b, pb, &hb, addr);
    }
    while (true) {
        if (kStats) { st[0] += ha + hb; st[1] = max(st[1], max(ha, hb)); ha = hb = 0; }
        if (a == b) return;
        if (a < b) { const uint32_t s = a; a = b; b = s; }
        const uint32_t old = atomicMin(labels + addr(a), b);
        if (old == a) return;
        if (kStats) st[2] += 1;
        a = find_root_halving<kStats, A>(labels, old, &ha, addr);
        b = find_root_halving<kStats, A>(labels, b, &hb, addr);
    }
}

// d / L for d < 64 * L <= 2^22
__device__ __forceinline__ uint32_t div_L(uint32_t d, const Params &P)
{
    return (P.log2L != 0xFFFFFFFFu) ? (d >> P.log2L) : (uint32_t)(((uint64_t)d * P.divL_magic) >> 40);
}

}  // namespace sw
