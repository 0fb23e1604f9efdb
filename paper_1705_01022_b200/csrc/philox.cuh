// Philox4x32-10 for the sweep kernels (counter-based RNG; the paper is silent on the generator,
// DESIGN.md R19 fixes it).  Written for the device: one IMAD.WIDE.U32 per 32x32->64 product, the ten
// round keys are precomputed on the host once per handle and live in the kernel-parameter constant
// bank, so the key schedule costs no instructions.
#pragma once
#include <cstdint>

namespace octb {

struct PhiloxRoundKeys {
    uint32_t k0[10];
    uint32_t k1[10];
};

// Stream tags, counter = (c0, c1, tag<<30 | set<<28 | dom, t)   (R19)
constexpr uint32_t kTagCell = 0u, kTagBlock = 1u, kTagGlobal = 2u;

__host__ inline PhiloxRoundKeys make_round_keys(uint64_t seed)
{
    PhiloxRoundKeys rk;
    uint32_t a = static_cast<uint32_t>(seed), b = static_cast<uint32_t>(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        rk.k0[r] = a;
        rk.k1[r] = b;
        a += 0x9E3779B9u;   // golden-ratio Weyl increments of the Philox key schedule
        b += 0xBB67AE85u;
    }
    return rk;
}

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              const PhiloxRoundKeys& rk, uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = static_cast<uint64_t>(0xD2511F53u) * c0;
        const uint64_t p1 = static_cast<uint64_t>(0xCD9E8D57u) * c2;
        const uint32_t n0 = static_cast<uint32_t>(p1 >> 32) ^ c1 ^ rk.k0[r];
        const uint32_t n2 = static_cast<uint32_t>(p0 >> 32) ^ c3 ^ rk.k1[r];
        c1 = static_cast<uint32_t>(p1);
        c3 = static_cast<uint32_t>(p0);
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

}  // namespace octb
