// Philox4x32-10 counter-based generator (Salmon et al., SC'11) for device and
// host code of the CUDA path, plus the keyed permutation used by the network
// generator.  Counter layout of every draw: (a_lo, a_hi | stream << 24, b_lo,
// b_hi), key = seed.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace dbk {

__host__ __device__ __forceinline__ uint32_t mulhi32(uint32_t a, uint32_t b) {
#ifdef __CUDA_ARCH__
    return __umulhi(a, b);
#else
    return (uint32_t)(((uint64_t)a * (uint64_t)b) >> 32);
#endif
}

__host__ __device__ __forceinline__ uint4 philox4x32_10(uint4 ctr, uint32_t k0, uint32_t k1) {
    constexpr uint32_t kMulA = 0xD2511F53u, kMulB = 0xCD9E8D57u;
    constexpr uint32_t kWeylA = 0x9E3779B9u, kWeylB = 0xBB67AE85u;
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t hiA = mulhi32(kMulA, ctr.x), loA = kMulA * ctr.x;
        const uint32_t hiB = mulhi32(kMulB, ctr.z), loB = kMulB * ctr.z;
        ctr = make_uint4(hiB ^ ctr.y ^ k0, loB, hiA ^ ctr.w ^ k1, loA);
        k0 += kWeylA;
        k1 += kWeylB;
    }
    return ctr;
}

// Same function with the ten round keys taken from a table (kernel parameters: they become
// constant-bank operands of the xor, and the key schedule costs nothing per draw).
__device__ __forceinline__ uint4 philox4x32_10_rk(uint4 ctr, const uint32_t (&rk)[20]) {
    constexpr uint32_t kMulA = 0xD2511F53u, kMulB = 0xCD9E8D57u;
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t hiA = __umulhi(kMulA, ctr.x), loA = kMulA * ctr.x;
        const uint32_t hiB = __umulhi(kMulB, ctr.z), loB = kMulB * ctr.z;
        ctr = make_uint4(hiB ^ ctr.y ^ rk[2 * round], loB, hiA ^ ctr.w ^ rk[2 * round + 1], loA);
    }
    return ctr;
}

__host__ __device__ __forceinline__ uint4 keyed_draw(uint32_t seed_lo, uint32_t seed_hi, uint32_t stream,
                                                     uint64_t a, uint64_t b) {
    return philox4x32_10(make_uint4((uint32_t)a, (uint32_t)(a >> 32) | (stream << 24),
                                    (uint32_t)b, (uint32_t)(b >> 32)), seed_lo, seed_hi);
}

__host__ __device__ __forceinline__ uint32_t avalanche32(uint32_t h) {   // MurmurHash3 finaliser
    h ^= h >> 16; h *= 0x85EBCA6Bu;
    h ^= h >> 13; h *= 0xC2B2AE35u;
    h ^= h >> 16;
    return h;
}

// Keyed permutation of [0, M): 8-round alternating Feistel network over
// max(2, ceil(log2 M)) bits, cycle-walked back into range.
__host__ __device__ __forceinline__ uint32_t feistel_perm(uint32_t x, uint32_t M, const uint4 key) {
    if (M <= 1u) return 0u;
    int bits = 2;
    while (bits < 32 && (1ull << bits) < (unsigned long long)M) ++bits;
    const int hi_bits = bits >> 1, lo_bits = bits - hi_bits;
    const uint32_t hi_mask = (1u << hi_bits) - 1u, lo_mask = (1u << lo_bits) - 1u;
    const uint32_t rk[4] = {key.x, key.y, key.z, key.w};
    do {
        uint32_t left = x >> lo_bits, right = x & lo_mask;
        // rounds alternate the widths: even rounds produce hi_bits, odd rounds lo_bits
#pragma unroll
        for (int r = 0; r < 8; r += 2) {
            const uint32_t wob = (uint32_t)(r >> 2) * 0x9E3779B9u;
            const uint32_t f0 = avalanche32(right + rk[r & 3] + wob) & hi_mask;
            const uint32_t mid = left ^ f0;                       // hi_bits wide, new right
            const uint32_t f1 = avalanche32(mid + rk[(r + 1) & 3] + wob) & lo_mask;
            const uint32_t nxt = right ^ f1;                      // lo_bits wide
            left = mid; right = nxt;                              // after two rounds widths are (hi, lo) again
        }
        x = (left << lo_bits) | right;
    } while (x >= M);
    return x;
}

}  // namespace dbk
