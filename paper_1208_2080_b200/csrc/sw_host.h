// sw_host.h -- host-side helpers shared by the translation units of libsw.so (sw_api.cu, sw_super.cu, sw_xy.cu).
#pragma once

#include <cmath>
#include <cstdint>

#include "sw_common.cuh"

namespace swh {

// north_star: T = floor(p * 2^32), p = 1 - exp(-K), computed once on the host (R10)
inline bool host_threshold(double K, uint64_t *T)
{
    if (std::isnan(K) || K < 0.0) return false;
    if (std::isinf(K)) { *T = 1ull << 32; return true; }
    const double scaled = std::floor(std::ldexp(-std::expm1(-K), 32));
    *T = scaled <= 0.0 ? 0ull : (scaled >= 4294967296.0 ? (1ull << 32) : (uint64_t)scaled);
    return true;
}

inline uint32_t log2_exact(uint32_t v)
{
    for (uint32_t b = 0; b < 32; ++b) if ((1u << b) == v) return b;
    return 0xFFFFFFFFu;
}

// kernel parameter block for sweep t of an L x L lattice (N = number of sites the launch covers)
inline sw::Params make_params(uint32_t L, uint32_t q, uint64_t N, uint64_t seed, uint64_t T, uint64_t t)
{
    sw::Params P{};
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        P.rk0[r] = k0; P.rk1[r] = k1;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    P.L = L; P.q = q; P.t = (uint32_t)t; P.N = N;
    P.thr_any = T ? 0xFFFFFFFFu : 0u;
    P.thr_m1 = T ? (uint32_t)(T - 1) : 0u;
    P.log2L = log2_exact(L);
    P.divL_magic = ((1ull << 40) + L - 1) / L;
    sw::sweep_keys(P, P.t, P.pk_t);
    sw::sweep_keys(P, P.t + 1u, P.pk_n);
    return P;
}

constexpr size_t kAlign = 256;
inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

}  // namespace swh
