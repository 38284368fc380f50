// Philox4x32-10 counter-based generator for the device path.
//
// The flip step of Algorithm 2 ("flip sigma_i with probability F_p";
// L160 describes one cuRAND generator per thread) is made stateless here: one call
// is keyed on (seed; spin id, absolute sweep, replica>>2, domain) and yields the
// uint32 words of four consecutive replicas (reading Q11).  This is the
// CUDA path's own implementation of the published Philox4x32-10 algorithm (Salmon et
// al., SC'11); it shares nothing with oracle/.
#pragma once
#include <cstdint>

namespace ising {

constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;
constexpr uint32_t kDomainFlip = 0u;
constexpr uint32_t kDomainInit = 1u;
constexpr uint32_t kDomainFlipN = 2u;   // Algorithm 1's exact-N flip step: counter word 0 = draw index

// The ten round keys depend on the seed only, so the host computes them once per call
// and the kernels receive them by value (they end up in uniform registers / constants).
struct PhiloxKeys {
    uint32_t k0[10];
    uint32_t k1[10];
};

inline PhiloxKeys philox_make_keys(uint64_t seed) {
    PhiloxKeys k;
    uint32_t a = (uint32_t)(seed & 0xFFFFFFFFull), b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        k.k0[r] = a;
        k.k1[r] = b;
        a += kPhiloxW0;
        b += kPhiloxW1;
    }
    return k;
}

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const PhiloxKeys& k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(kPhiloxM0, c0), lo0 = kPhiloxM0 * c0;
        const uint32_t hi1 = __umulhi(kPhiloxM1, c2), lo1 = kPhiloxM1 * c2;
        c0 = hi1 ^ c1 ^ k.k0[r];
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k.k1[r];
        c3 = lo0;
    }
    return make_uint4(c0, c1, c2, c3);
}

}  // namespace ising
