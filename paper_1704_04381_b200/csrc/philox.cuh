// philox.cuh -- Philox4x32-10 on the device (Salmon et al., SC'11).
// Counter-based: one 128-bit block is a pure function of (counter, key); nothing is stored.
#pragma once
#include <cstdint>

namespace rosen {

struct PhiloxKeys {   // the 10 round keys of the Weyl schedule, computed once per call on the host: as members of the kernel
    uint32_t k0[10], k1[10];   // parameter struct they are constant-bank operands of the round's XOR (no per-round key arithmetic)
};

inline PhiloxKeys philox_round_keys(uint64_t seed)
{
    PhiloxKeys K;
    for (int r = 0; r < 10; ++r) {
        K.k0[r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u;
        K.k1[r] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
    }
    return K;
}

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxKeys& K, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ K.k0[r];
        const uint32_t n2 = hi0 ^ c3 ^ K.k1[r];
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t key0, uint32_t key1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t k0 = key0 + (uint32_t)r * 0x9E3779B9u;   // folded to constants + uniform adds
        const uint32_t k1 = key1 + (uint32_t)r * 0xBB67AE85u;
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

}  // namespace rosen
