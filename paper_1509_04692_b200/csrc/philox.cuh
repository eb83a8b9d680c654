// Philox4x32-10 counter-based RNG for the CUDA path (R3, R4).
// Replaces the paper's Saru hash keyed on (particle index, time step, seed, rank).
// Independent restatement: shares no code with oracle/.
#pragma once
#include <cstdint>

namespace hpmc {

constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;

constexpr uint32_t kTagShift = 1u;  // grid shift of a sweep
constexpr uint32_t kTagPerm = 2u;   // colour permutation of a sweep
constexpr uint32_t kTagTrial = 3u;  // one trial move

struct U4 {
    uint32_t x, y, z, w;
};

__host__ __device__ __forceinline__ uint32_t mulhi32(uint32_t a, uint32_t b)
{
#ifdef __CUDA_ARCH__
    return __umulhi(a, b);
#else
    return (uint32_t)(((uint64_t)a * (uint64_t)b) >> 32);
#endif
}

__host__ __device__ __forceinline__ U4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                     uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = mulhi32(kPhiloxM0, c0), lo0 = kPhiloxM0 * c0;
        const uint32_t hi1 = mulhi32(kPhiloxM1, c2), lo1 = kPhiloxM1 * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += kPhiloxW0;
        k1 += kPhiloxW1;
    }
    return U4{c0, c1, c2, c3};
}

// The same block function with the round keys rk[2 r] = k0 + r W0, rk[2 r + 1] = k1 + r W1 precomputed (GridParams::philox_rk)
__device__ __forceinline__ U4 philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const uint32_t (&rk)[20])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        // one 32 x 32 -> 64 bit product per multiplier (IMAD.WIDE) instead of a high and a low multiply
        const uint64_t p0 = (uint64_t)kPhiloxM0 * (uint64_t)c0, p1 = (uint64_t)kPhiloxM1 * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        c0 = hi1 ^ c1 ^ rk[2 * r];
        c1 = lo1;
        c2 = hi0 ^ c3 ^ rk[2 * r + 1];
        c3 = lo0;
    }
    return U4{c0, c1, c2, c3};
}

// R4: exact in fp32 (a 24-bit integer times a power of two)
__host__ __device__ __forceinline__ float u01(uint32_t r) { return (float)(r >> 8) * (1.0f / 16777216.0f); }
__host__ __device__ __forceinline__ float usym(uint32_t r)
{
    return (float)((int32_t)(r >> 8) - 8388608) * (1.0f / 8388608.0f);
}

}  // namespace hpmc
