// sw_generic.cuh -- reference kernels that work for ANY lattice size 2 <= L <= 65536 (odd,
// tiny, not a multiple of the tile): one global union-find over all active bonds.  They are the
// slow-but-general path of libsw.so (and its internal cross-check for the tiled path); the hot
// path for L % 64 == 0 is in sw_tiled.cuh.
//
// Bond storage on the device (both paths): word w of `bonds` covers the 16 consecutive linear
// sites 16w .. 16w+15; bit j = right bond of site 16w+j, bit 16+j = its down bond.
#pragma once

#include "sw_common.cuh"

namespace sw {

// --- init / state -------------------------------------------------------------------------------

__global__ void k_init_random(uint8_t *__restrict__ spins, Params P)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) {
        const uint4 w = philox4x32_10((uint32_t)i, (uint32_t)(i >> 32), 0u, kPurposeInit, P);
        spins[i] = (uint8_t)state_from_draw(w.x, P.q);
    }
}

// flag[0] |= 1 if any spin >= q
__global__ void k_validate_spins(const uint8_t *__restrict__ spins, Params P, uint32_t *flag)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    bool bad = false;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride)
        bad |= spins[i] >= P.q;
    if (__any_sync(0xFFFFFFFFu, bad) && (threadIdx.x & 31) == 0) atomicOr(flag, 1u);
}

// --- packed spin states (sw_set_state_packed / sw_get_spins_packed): `bits` in {1, 2, 4, 8} per spin, site i in bits
// [bits (i % per), bits (i % per + 1)) of byte i / per, per = 8 / bits.  One thread per 16 sites (a uint4 of spins).
__global__ void k_unpack_spins(const uint8_t *__restrict__ packed, uint8_t *__restrict__ spins, Params P, uint32_t bits, uint32_t *flag)
{
    const uint64_t n_groups = P.N >> 4, stride = (uint64_t)gridDim.x * blockDim.x;   // N % 16 == 0 (checked by the caller)
    const uint32_t mask = (1u << bits) - 1u;
    bool bad = false;
    for (uint64_t g = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; g < n_groups; g += stride) {
        unsigned long long w = 0;                            // the 16 * bits <= 128 bits of this group; 8 bits per spin: two loads
        uint32_t out[4];
        if (bits == 8) {
            const uint4 v = *reinterpret_cast<const uint4 *>(packed + (g << 4));
            out[0] = v.x; out[1] = v.y; out[2] = v.z; out[3] = v.w;
        } else {
            if (bits == 1) w = *reinterpret_cast<const uint16_t *>(packed + (g << 1));
            else if (bits == 2) w = *reinterpret_cast<const uint32_t *>(packed + (g << 2));
            else w = *reinterpret_cast<const unsigned long long *>(packed + (g << 3));
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                uint32_t o = 0;
#pragma unroll
                for (int j = 0; j < 4; ++j) o |= (uint32_t)((w >> (bits * (4 * k + j))) & mask) << (8 * j);
                out[k] = o;
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int j = 0; j < 4; ++j) bad |= ((out[k] >> (8 * j)) & 0xFFu) >= P.q;
        *reinterpret_cast<uint4 *>(spins + (g << 4)) = make_uint4(out[0], out[1], out[2], out[3]);
    }
    if (__any_sync(0xFFFFFFFFu, bad) && (threadIdx.x & 31) == 0) atomicOr(flag, 1u);
}

__global__ void k_pack_spins(const uint8_t *__restrict__ spins, uint8_t *__restrict__ packed, uint64_t first_group, uint64_t n_groups, uint32_t bits)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n_groups; k += stride) {
        const uint64_t g = first_group + k;
        const uint4 v = *reinterpret_cast<const uint4 *>(spins + (g << 4));
        const uint32_t in[4] = {v.x, v.y, v.z, v.w};
        if (bits == 8) { *reinterpret_cast<uint4 *>(packed + (k << 4)) = v; continue; }
        unsigned long long w = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int j = 0; j < 4; ++j) w |= (unsigned long long)((in[a] >> (8 * j)) & 0xFFu) << (bits * (4 * a + j));
        if (bits == 1) *reinterpret_cast<uint16_t *>(packed + (k << 1)) = (uint16_t)w;
        else if (bits == 2) *reinterpret_cast<uint32_t *>(packed + (k << 2)) = (uint32_t)w;
        else *reinterpret_cast<unsigned long long *>(packed + (k << 3)) = w;
    }
}

// --- step (1): bonds, one thread per 16-site word -----------------------------------------------

__global__ void k_bonds_generic(const uint8_t *__restrict__ spins, uint32_t *__restrict__ bonds, Params P)
{
    const uint64_t n_words = (P.N + 15) >> 4;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t L = P.L;
    for (uint64_t w = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_words; w += stride) {
        uint32_t word = 0;
        for (uint32_t j = 0; j < 16; ++j) {
            const uint64_t i = (w << 4) + j;
            if (i >= P.N) break;
            const uint64_t y = i / L, x = i - y * L;
            const uint64_t ir = y * L + (x + 1 == L ? 0 : x + 1);
            const uint64_t id = (y + 1 == L ? 0 : y + 1) * L + x;
            const uint8_t s = spins[i];
            const bool er = s == spins[ir], ed = s == spins[id];
            if (er | ed) {
                const uint64_t pair = i >> 1;
                const uint4 d = philox4x32_10((uint32_t)pair, (uint32_t)(pair >> 32), P.t, kPurposeBond, P);
                const uint32_t dr = (i & 1) ? d.z : d.x;
                const uint32_t dd = (i & 1) ? d.w : d.y;
                if (er && P.thr_any && dr <= P.thr_m1) word |= 1u << j;
                if (ed && P.thr_any && dd <= P.thr_m1) word |= 1u << (16 + j);
            }
        }
        bonds[w] = word;
    }
}

// --- step (2): labels ---------------------------------------------------------------------------

__global__ void k_label_identity(uint32_t *__restrict__ labels, Params P)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride)
        labels[i] = (uint32_t)i;
}

__global__ void k_union_generic(const uint32_t *__restrict__ bonds, uint32_t *labels, Params P)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t L = P.L;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) {
        const uint32_t word = bonds[i >> 4];
        const uint32_t j = (uint32_t)(i & 15);
        const bool br = (word >> j) & 1u, bd = (word >> (16 + j)) & 1u;
        if (!(br | bd)) continue;
        const uint64_t y = i / L, x = i - y * L;
        if (br) unite(labels, (uint32_t)i, (uint32_t)(y * L + (x + 1 == L ? 0 : x + 1)));
        if (bd) unite(labels, (uint32_t)i, (uint32_t)((y + 1 == L ? 0 : y + 1) * L + x));
    }
}

// --- comparison variant: "Label Equivalence" of Kalentev et al., as the paper describes it -------
// SW_FLAG_LABEL_EQUIVALENCE.  Prior art, kept behind the same ABI to reproduce the one per-step figure the paper
// gives (about 8.6 scan + analysis rounds per sweep at 4096^2, q = 2, T_c) and to show what the tiled path buys.
//
// scanning: "compares the label of each site with that of the nearest-neighbor sites when the bond between [them] is
// active.  If the label of the nearest-neighbor site is smaller than the label of that site, the label variable with
// the label number, label[label], is updated to the smallest one."  All four neighbours are looked at (a site owns its
// right and down bond; the left and up bonds belong to the neighbours).  *changed is set if anything was lowered.
__global__ void k_le_scan(const uint32_t *__restrict__ bonds, uint32_t *labels, Params P, uint32_t *changed)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t L = P.L;
    bool any = false;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) {
        const uint64_t y = i / L, x = i - y * L;
        const uint64_t ir = y * L + (x + 1 == L ? 0 : x + 1), id = (y + 1 == L ? 0 : y + 1) * L + x;
        const uint64_t il = y * L + (x == 0 ? L - 1 : x - 1), iu = (y == 0 ? L - 1 : y - 1) * L + x;
        const uint32_t wi = bonds[i >> 4], wl = bonds[il >> 4], wu = bonds[iu >> 4];
        const uint32_t mine = ld_label(labels, (uint32_t)i);
        uint32_t m = mine;
        if ((wi >> (i & 15)) & 1u) m = min(m, ld_label(labels, (uint32_t)ir));
        if ((wi >> (16 + (i & 15))) & 1u) m = min(m, ld_label(labels, (uint32_t)id));
        if ((wl >> (il & 15)) & 1u) m = min(m, ld_label(labels, (uint32_t)il));
        if ((wu >> (16 + (iu & 15))) & 1u) m = min(m, ld_label(labels, (uint32_t)iu));
        if (m < mine) { atomicMin(labels + mine, m); any = true; }
    }
    if (__any_sync(0xFFFFFFFFu, any) && (threadIdx.x & 31) == 0) atomicOr(changed, 1u);
}

// analysis: "each thread tracks back the label variable until the label variable, label, remains unchanged."
__global__ void k_le_analysis(uint32_t *labels, Params P)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) {
        uint32_t l = ld_label(labels, (uint32_t)i), r = ld_label(labels, l);
        while (r != l) { l = r; r = ld_label(labels, l); }
        labels[i] = l;
    }
}

// labels[i] <- root(i).  In-place is safe: whatever another thread reads is an ancestor.
__global__ void k_flatten_generic(uint32_t *labels, Params P)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride) {
        const uint32_t l = ld_label(labels, (uint32_t)i);
        if (l == (uint32_t)i) continue;
        const uint32_t r = find_root(labels, l);
        if (r != l) labels[i] = r;
    }
}

// --- step (3): flip; works on a flattened OR an unflattened forest ------------------------------

__global__ void k_flip_generic(const uint32_t *__restrict__ labels, uint8_t *__restrict__ spins, Params P)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += stride)
        spins[i] = (uint8_t)flip_state(find_root(labels, (uint32_t)i), P);
}

// --- expand the packed bond words to one byte per site (sw_get_bonds) ---------------------------

__global__ void k_expand_bonds(const uint32_t *__restrict__ bonds, uint8_t *__restrict__ out,
                               uint64_t first_site, uint64_t n_sites)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n_sites; k += stride) {
        const uint64_t i = first_site + k;
        const uint32_t word = bonds[i >> 4];
        const uint32_t j = (uint32_t)(i & 15);
        out[k] = (uint8_t)(((word >> j) & 1u) | (((word >> (16 + j)) & 1u) << 1));
    }
}

}  // namespace sw
