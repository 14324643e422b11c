// planes_common.cuh — device helpers shared by the multi-spin (bit-plane) tile kernels
// (tile_planes.cu: 2D, tile3d_planes.cu: 3D).  DESIGN.md §6.1.
#pragma once
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

// Own-tile data is read once and written back by the same lane: plain (coherent) loads that do not allocate in
// L1.  Halo data belongs to tiles of the other coarse colour, which this launch never writes — but with
// programmatic dependent launch this grid may be resident while the previous colour's grid is still writing those very
// words, and ld.global.nc requires data that is read-only for the whole lifetime of the kernel: so the halos, too, are read
// with coherent loads after griddepcontrol.wait (ldh128 / ldh64 / ldh32), never through the read-only path;
// and they are cached in L2 only (.cg), so that a persistent kernel (k_flow_planes) can never meet a stale copy in L1.
// L2 policy for the tile bodies: when the records exceed L2 they are touched once per pass, so they are
// streamed (evict-first) and the small edge copies the next launch needs stay resident (+5 % at L = 16384);
// when the records fit L2 the normal policy keeps them there (streaming costs 7-10 % at L <= 8192).
__device__ __forceinline__ uint64_t body_policy(bool stream) {
    uint64_t first, normal;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(first));
    asm("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(normal));
    return stream ? first : normal;
}
__device__ __forceinline__ uint4 ldg128(const void* p, uint64_t pol) {
    uint4 v;
    asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t ldg32(const void* p) {
    uint32_t v;
    asm volatile("ld.global.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint4 ldh128(const void* p) {
    uint4 v;
    asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint2 ldh64(const void* p) {
    uint2 v;
    asm volatile("ld.global.cg.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t ldh32(const void* p) {
    uint32_t v;
    asm volatile("ld.global.cg.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t ldh8(const void* p) {
    uint32_t v;
    asm volatile("ld.global.cg.u8 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint4 lds128(uint32_t saddr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(saddr));
    return v;
}
__device__ __forceinline__ uint32_t lds32(uint32_t saddr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr));
    return v;
}
__device__ __forceinline__ uint2 lds64(uint32_t saddr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(saddr));
    return v;
}
__device__ __forceinline__ void stg128(void* p, uint4 v) {
    asm volatile("st.global.v4.u32 [%4], {%0,%1,%2,%3};" ::"r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(p) : "memory");
}
__device__ __forceinline__ void stg128(void* p, uint4 v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v4.u32 [%4], {%0,%1,%2,%3}, %5;" ::"r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(p), "l"(pol) : "memory");
}

// int8 pieces.  A piece = 16 bytes of 0/1 = the 16 sites k = 0..15 of one half-word.  Site k lives at byte
// piece_byte(k): sites 0..7 in words 0,1, sites 8..15 in words 2,3, inside a word pair even sites in the first
// word, odd sites in the second.  That order makes packing two multiplies per 8 sites:
//   c = w_even + 2 * w_odd has the site pair (2i, 2i+1) in bits (8i, 8i+1);  c * 0x01041040 moves them to bits
//   24+2i, 25+2i (all other partial products land below bit 24 or overflow, none collide), i.e. 8 sites in the top byte.
__host__ __device__ constexpr int piece_byte(int k) { return 8 * (k >> 3) + 4 * (k & 1) + ((k & 7) >> 1); }

__device__ __forceinline__ uint32_t pack_step(uint32_t acc, uint32_t w_even, uint32_t w_odd) {
    return __funnelshift_l((w_even + 2u * w_odd) * 0x01041040u, acc, 8);     // (acc << 8) | 8 site bits
}
// 16 bytes appended below acc: acc = (acc << 16) | bits, bit k = site k.
__device__ __forceinline__ uint32_t pack16(uint32_t acc, const uint4& v) {
    acc = pack_step(acc, v.z, v.w);
    return pack_step(acc, v.x, v.y);
}

// int8 write-back table: 8 bits -> 8 bytes of 0/1.  A compile-time constant array in global memory (2 KB, stays in
// L1 / L2); lookups go through the read-only path, so no kernel builds a copy or needs a barrier.
struct ByteLut {
    uint2 e[256];
    __host__ __device__ constexpr ByteLut() : e() {
        for (int i = 0; i < 256; ++i) {
            unsigned lo = 0, hi = 0;
            for (int b = 0; b < 4; ++b) {                    // piece_byte order: even sites, then odd sites
                lo |= (unsigned)((i >> (2 * b)) & 1) << (8 * b);
                hi |= (unsigned)((i >> (2 * b + 1)) & 1) << (8 * b);
            }
            e[i].x = lo; e[i].y = hi;
        }
    }
};
__device__ const ByteLut kByteLutGlobal = ByteLut();

// ceil(2^32 / d) on the host; q / d on the device = umulhi(q, magic) corrected by at most one either way.
#ifndef __CUDACC_RTC__
inline uint32_t fastdiv_magic(uint32_t d) { return d <= 1 ? 0xffffffffu : (uint32_t)((0x100000000ull + d - 1) / d); }
#endif
__device__ __forceinline__ uint32_t fastdiv(uint32_t q, uint32_t d, uint32_t magic) {
    uint32_t r = __umulhi(q, magic);
    if (r * d > q) --r;
    if ((r + 1) * d <= q) ++r;
    return r;
}

}  // namespace ising
