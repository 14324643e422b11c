// planes_common.cuh — device helpers shared by the multi-spin (bit-plane) tile kernels
// (tile_planes.cu: 2D, tile3d_planes.cu: 3D).  DESIGN.md §6.1.
#pragma once
#include <cstdint>

#include "philox.cuh"

namespace ising {

template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(r) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return r;
}
// LOP3 immediates: value of f(a,b,c) at bit (a<<2 | b<<1 | c), a = 0xF0, b = 0xCC, c = 0xAA.
constexpr int kLutChain = (~0xF0 & 0xAA) | (~(0xF0 ^ 0xAA) & 0xCC);    // (~p & u) | (~(p ^ u) & bw): p=a, bw=b, u=c
constexpr int kLutNe = 0xF0 | (0xCC ^ 0xAA);                            // ne | (p ^ u): ne=a, p=b, u=c

// Own-tile data is read once and written back by the same lane: plain (coherent) loads that
// do not allocate in L1.  Halo data belongs to tiles of the other coarse colour, which this
// launch never writes, so it may use the read-only path (__ldg).
__device__ __forceinline__ uint4 ldg128(const void* p) {
    uint4 v;
    asm volatile("ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t ldg32(const void* p) {
    uint32_t v;
    asm volatile("ld.global.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void stg128(void* p, uint4 v) {
    asm volatile("st.global.v4.u32 [%4], {%0,%1,%2,%3};" ::"r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(p) : "memory");
}

// 4 bytes of 0/1 -> 4 bits in the top nibble: b0 -> bit 28, ..., b3 -> bit 31 (no carries collide).
__device__ __forceinline__ uint32_t pack_step(uint32_t acc, uint32_t w) {
    return __funnelshift_l(w * 0x10204080u, acc, 4);     // (acc << 4) | nibble
}
// 16 bytes (pairs 0..15) appended below acc: acc = (acc << 16) | bits, bit k = byte k.
__device__ __forceinline__ uint32_t pack16(uint32_t acc, const uint4& v) {
    acc = pack_step(acc, v.w);
    acc = pack_step(acc, v.z);
    acc = pack_step(acc, v.y);
    return pack_step(acc, v.x);
}

// int8 write-back table: 8 bits -> 8 bytes of 0/1.  A compile-time constant array in global memory (2 KB, stays in
// L1 / L2); lookups go through the read-only path, so no kernel builds a copy or needs a barrier.
struct ByteLut {
    uint2 e[256];
    constexpr ByteLut() : e() {
        for (int i = 0; i < 256; ++i) {
            unsigned lo = 0, hi = 0;
            for (int b = 0; b < 4; ++b) {
                lo |= (unsigned)((i >> b) & 1) << (8 * b);
                hi |= (unsigned)((i >> (4 + b)) & 1) << (8 * b);
            }
            e[i].x = lo; e[i].y = hi;
        }
    }
};
__device__ const ByteLut kByteLutGlobal = ByteLut();

// ceil(2^32 / d) on the host; q / d on the device = umulhi(q, magic) corrected by at most one either way.
inline uint32_t fastdiv_magic(uint32_t d) { return d <= 1 ? 0xffffffffu : (uint32_t)((0x100000000ull + d - 1) / d); }
__device__ __forceinline__ uint32_t fastdiv(uint32_t q, uint32_t d, uint32_t magic) {
    uint32_t r = __umulhi(q, magic);
    if (r * d > q) --r;
    if ((r + 1) * d <= q) ++r;
    return r;
}

}  // namespace ising
