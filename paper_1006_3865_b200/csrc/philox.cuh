// philox.cuh — counter-based Philox4x32-10 (Salmon et al., SC'11) for the device path.
// S8c.2: multipliers 0xD2511F53 (on ctr[0]) and 0xCD9E8D57 (on ctr[2]); key increments
// 0x9E3779B9 / 0xBB67AE85; ten rounds.  No RNG state ever lives in HBM (BASELINE north_star).
#pragma once
#ifdef __CUDACC_RTC__          // run-time compilation (planes_jit.cu): no host headers
typedef unsigned char uint8_t;
typedef signed char int8_t;
typedef unsigned short uint16_t;
typedef unsigned int uint32_t;
typedef unsigned long long uint64_t;
typedef unsigned long size_t;
#else
#include <cstdint>
#endif

namespace ising {

constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;

// Stream tags carried in ctr[1] (S8c.3).
constexpr uint32_t kTagSweep = 0u;
constexpr uint32_t kTagInit = 1u;
constexpr uint32_t kTagPlanes = 3u;   // RNG mapping "planes": head planes of a 32-site block, call n adds 256*n
constexpr uint32_t kTagTail = 4u;     // RNG mapping "planes": per-site tail bits
constexpr int kHeadBits = 12;         // leading bits of r taken from bit-planes (DESIGN.md §3 R6)
constexpr int kTailBits = 32 - kHeadBits;

struct u32x4 { uint32_t x, y, z, w; };

// One call = 20 IMAD.WIDE.U32 + 20 LOP3 on sm_100a (key schedule folds to immediates or
// uniform registers when the key is warp-uniform).
__device__ __forceinline__ u32x4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t lo0 = kPhiloxM0 * c0;
        const uint32_t hi0 = __umulhi(kPhiloxM0, c0);
        const uint32_t lo1 = kPhiloxM1 * c2;
        const uint32_t hi1 = __umulhi(kPhiloxM1, c2);
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += kPhiloxW0;
        k1 += kPhiloxW1;
    }
    return u32x4{c0, c1, c2, c3};
}

}  // namespace ising
