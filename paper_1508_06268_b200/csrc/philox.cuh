// philox.cuh -- Philox4x32-10 for the device (S2; Salmon et al., SC'11).
// One call: 128-bit counter + 64-bit key -> four 32-bit words; ten rounds, key bumped by the Weyl
// constants between rounds.  Written for the IMAD.WIDE pipe: one 32x32->64 multiply per product.
#pragma once
#include <cstdint>

namespace rfim {

constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;

// counter word 3 (S2)
enum : uint32_t { kDomColour0 = 0, kDomColour1 = 1, kDomExchange = 2, kDomInitSpins = 3, kDomField = 4 };

struct Words4 { uint32_t w0, w1, w2, w3; };

__host__ __device__ __forceinline__ Words4 philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1,
                                                         uint32_t c2, uint32_t c3) {
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += kPhiloxW0;
        k1 += kPhiloxW1;
    }
    Words4 r;
    r.w0 = c0; r.w1 = c1; r.w2 = c2; r.w3 = c3;
    return r;
}

__host__ __device__ __forceinline__ uint32_t pick_word(const Words4& w, uint32_t k) {
    return k == 0 ? w.w0 : (k == 1 ? w.w1 : (k == 2 ? w.w2 : w.w3));
}

}  // namespace rfim
