// tile_planes.cu — the 2D double-checkerboard tile kernel in multi-spin (bit-plane) form,
// RNG mapping "planes" (DESIGN.md §3 R6, §5, §6).  Steps a1, a3-a7 of SURVEY §8(a).
//
// Arithmetic form.  A 32-bit word holds the 32 same-colour sites of one RNG block: 16 pairs
// p_x x 2 rows, bit j = (y & 1) * 16 + (p_x & 15).  For a half-sweep of colour c the four
// neighbours of all 32 sites are four words of the other colour (same block; same block with
// its halves swapped; the blocks above/below; the block shifted by one pair), so
//   disagreement masks, a 4-input bit adder, and
//   flip = [n_dis >= 2] | [n_dis >= 1] & R1 | R2,    R_m = [r < thr[m]] per site
// cost ~10 LOP3 per 32 sites.  R_m comes from the 12 head planes of the block (3 Philox calls)
// by a bit-serial borrow chain against the head bits of thr[m] (uniform operands), LSB plane
// first; a site whose head equals the head of a threshold it needs (probability 2^-12) draws its
// 20 tail bits from the per-site call.  Everything runs in registers: a warp owns 64 tile rows
// (one 64x64 tile or two 32x32 tiles), lane = block row, vertical neighbours come by shuffle,
// the k inner sweeps never touch memory.
//
// HBM layouts (tile records; PG below):
//   int8  record = T*T body + 64 edge bytes, 0/1 per spin.  Body is piece-major: the 16 bytes
//         (row 2Y+rp, colour cc, pairs 16gx..16gx+15) sit at ((rp*2+cc)*NW+gx)*LPT*16 + Y*16, so lane Y
//         loads its 4*NW pieces with fully coalesced 128-bit accesses and no shared-memory staging.
//   bits  record = T*T/8 body + 64 edge bytes: word (cc, Y, gx) at ((cc*NW+gx)*LPT + Y)*4.
//   edge  = bit-packed copies of the tile's own first / last block row and first / last column, written by
//         the tile, so that every halo is one 16-byte run of ready-made words in the neighbour's record.
#include <algorithm>
#include <cooperative_groups.h>

#include "kernels.h"
#include "tile_planes_device.cuh"
#include "grid_planes_device.cuh"
#include "flow_planes_device.cuh"

namespace ising {

namespace {

// a8: plain checkerboard of a 64x64 lattice (tile = L = 64, BASELINE config 1).  One warp holds a whole
// replica in registers and runs all n passes of the call in one launch; E and M after every pass (a10) come
// from popcounts: M = 2*#up - N, E = -(2N - 2*#unsatisfied bonds), every bond seen once from its colour-0 end.
template <bool BITS, bool HASJ>
__global__ void __launch_bounds__(32) k_plain64_planes(PlaneArgs A, int n, long long* __restrict__ E, long long* __restrict__ M) {
    constexpr int T = 64;
    using G = PG<T>;
    const uint2* lut = kByteLutGlobal.e;
    const int Y = threadIdx.x, r = blockIdx.x;
    TileRegs<T> t;
    load_tile<T, BITS>(A, r, 0, 0, Y, 0, t);
    uint4 Jw[2][G::NW];
#pragma unroll
    for (int cc = 0; cc < 2; ++cc)
#pragma unroll
        for (int gx = 0; gx < G::NW; ++gx)
            Jw[cc][gx] = HASJ ? __ldg(A.jrec + (cc * G::NW + gx) * G::LPT + Y) : make_uint4(0u, 0u, 0u, 0u);
    const uint64_t seed = A.seeds[r];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    const uint32_t g0 = (uint32_t)Y * G::NW, p0 = 2u * (uint32_t)Y * (T / 2);
    for (int pass = 0; pass < n; ++pass) {
        for (int j = 0; j < A.k; ++j) {
            const uint64_t tt = A.t_first + (uint64_t)pass * (uint64_t)A.k + (uint64_t)j;
            half_sweep<T, HASJ, true>(A, t, Jw, 0, Y, g0, p0, 2 * tt, k0, k1);
            half_sweep<T, HASJ, true>(A, t, Jw, 1, Y, g0, p0, 2 * tt + 1, k0, k1);
        }
        if (E || M) {
            int up = 0, unsat = 0;
            count_row<T, true>(t, Jw, Y, up, unsat);
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                up += __shfl_xor_sync(0xffffffffu, up, d);
                unsat += __shfl_xor_sync(0xffffffffu, unsat, d);
            }
            if (Y == 0) {
                if (M) M[(size_t)pass * A.R + r] = 2ll * up - (long long)(T * T);
                if (E) E[(size_t)pass * A.R + r] = 2ll * unsat - 2ll * (T * T);
            }
        }
    }
    store_tile<T, BITS>(A, r, 0, 0, Y, 0, t, lut);
}

// a10 directly on the tile records (no conversion to the canonical array): one launch per coarse colour C adds
// the colour-C tiles' share to E[r], M[r] (zeroed by the caller): warp shuffle reduction over the lanes of a tile,
// then the (up to 8) tiles of the CTA meet in shared memory and one thread adds them per replica: all CTAs add to the
// same two words, and at L = 16384 the 65536 same-address atomics of a tile-level add cost more than reading the tiles.
template <int T, bool BITS, bool HASJ>
__global__ void __launch_bounds__(kPlaneThreads) k_observables_planes(PlaneArgs A, long long* __restrict__ E, long long* __restrict__ M) {
    using G = PG<T>;
    constexpr int NT = kPlaneThreads / 32 * G::TPW;        // tiles per CTA
    __shared__ int s_r[NT], s_up[NT], s_unsat[NT];
    const int lane = threadIdx.x & 31;
    const uint32_t job = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int sub = lane / G::LPT, Y = lane % G::LPT;
    int r = -1, up = 0, unsat = 0;
    if (job < A.njobs) {                                   // warp-uniform
        int tx, ty;
        job_tile<T>(A, job, sub, r, tx, ty);
        TileRegs<T> t;
        load_tile<T, BITS>(A, r, tx, ty, Y, sub * G::LPT, t);
        uint4 Jw[2][G::NW];
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int gx = 0; gx < G::NW; ++gx)
                Jw[cc][gx] = HASJ ? __ldg(A.jrec + ((size_t)ty * A.B + tx) * (2 * G::NW * G::LPT) + (cc * G::NW + gx) * G::LPT + Y)
                                  : make_uint4(0u, 0u, 0u, 0u);
        count_row<T, false>(t, Jw, Y, up, unsat);
#pragma unroll
        for (int d = G::LPT / 2; d > 0; d >>= 1) {           // reduce over the lanes of one tile
            up += __shfl_xor_sync(0xffffffffu, up, d);
            unsat += __shfl_xor_sync(0xffffffffu, unsat, d);
        }
    }
    if (Y == 0) {
        const int i = (threadIdx.x >> 5) * G::TPW + sub;
        s_r[i] = r; s_up[i] = up; s_unsat[i] = unsat;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int cr = -1;
        long long m = 0, e = 0;
        for (int i = 0; i <= NT; ++i) {
            const int ri = i < NT ? s_r[i] : -1;
            if (ri != cr) {                                 // tiles of a CTA are consecutive jobs: runs of equal r
                if (cr >= 0) {
                    if (M) atomicAdd(reinterpret_cast<unsigned long long*>(M + cr), (unsigned long long)m);
                    if (E) atomicAdd(reinterpret_cast<unsigned long long*>(E + cr), (unsigned long long)e);
                }
                cr = ri; m = 0; e = 0;
            }
            if (ri >= 0) {
                m += 2ll * s_up[i] - (long long)(T * T);
                e += 2ll * s_unsat[i] - 2ll * (T * T);
            }
        }
    }
}

// ---- layout converters (a11): canonical int8 +-1 <-> bit records; not on the timed path ----
// One thread per site; MODE 2: canonical -> bit records, 3: bit records -> canonical.  Bit fields are set by atomicOr
// into zeroed storage.  (The int8 records have their own converters below.)
template <int MODE>
__global__ void k_convert_planes(int8_t* __restrict__ canon, uint8_t* __restrict__ tiles, int L, int T, int R) {
    static_assert(MODE == 2 || MODE == 3, "bit records only");
    const uint64_t N = (uint64_t)L * L;
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= N * (uint64_t)R) return;
    const int r = (int)(gid / N);
    const uint64_t i = gid - (uint64_t)r * N;
    const int x = (int)(i % L), y = (int)(i / L);
    const int B = L / T, NW = T / 32, LPT = T / 2;
    const int tx = x / T, ty = y / T, lx = x - tx * T, ly = y - ty * T;
    const int cc = (lx + ly) & 1, px = lx >> 1, gx = px >> 4, kk = px & 15, rp = ly & 1, Y = ly >> 1;
    const size_t tile = ((size_t)r * B + ty) * B + tx;
    const size_t body_bytes = (size_t)(T * T / 8);
    uint8_t* rec = tiles + tile * (body_bytes + 64);
    uint32_t* w = reinterpret_cast<uint32_t*>(rec) + ((cc * NW + gx) * LPT + Y);
    const int j = rp * 16 + kk;
    if (MODE == 3) { canon[gid] = ((*w >> j) & 1u) ? 1 : -1; return; }
    if (canon[gid] <= 0) return;
    atomicOr(w, 1u << j);
    uint32_t* e = reinterpret_cast<uint32_t*>(rec + body_bytes);          // boundary copies (zeroed first), see PG
    if (Y == 0) atomicOr(e + 0 + cc * NW + gx, 1u << j);                  // TOP: words of block row 0
    if (Y == LPT - 1) atomicOr(e + 8 + cc * NW + gx, 1u << j);            // BOT: words of block row LPT-1
    if (lx == 0) atomicOr(e + 4 + rp, 1u << Y);                           // COL: L0, L1
    if (lx == T - 1) atomicOr(e + 6 + rp, 1u << Y);                       //      R0, R1
}

// ---- fast converters for the int8 records (the layout behind ising_set_spins / ising_copy_spins on the headline
// path).  Lane = block row Y of a tile (T = 64: a warp per tile; T = 32: two tiles per warp): it owns the rows 2Y and
// 2Y+1, i.e. one 16-byte piece per (rp, cc, gx).  Canonical side: 32-byte runs of a row (whole sectors); record side:
// the 32 (16) lanes of a tile touch consecutive pieces.  A 32-byte run of row ly holds the 16 sites of both colours
// of one RNG block row: site k of colour cc at byte 2k + a, a = (cc + ly) & 1, and piece_byte() wants words
// {k even of 0..7, k odd of 0..7, k even of 8..15, k odd of 8..15}: two byte permutations per word.
template <int T>
__global__ void __launch_bounds__(256) k_canon_to_planes_i8(const int8_t* __restrict__ canon, uint8_t* __restrict__ tiles,
                                                            int L, int B, uint32_t ntiles) {
    using G = PG<T>;
    const int lane = threadIdx.x & 31;
    const uint32_t warp = (uint32_t)((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    const uint32_t tile = warp * G::TPW + (uint32_t)(lane / G::LPT);
    const int Y = lane % G::LPT;
    const bool live = tile < ntiles;
    const uint32_t tc = live ? tile : 0;
    const uint32_t per_rep = (uint32_t)B * B;
    const uint32_t r = tc / per_rep, t2 = tc - r * per_rep;
    const int ty = (int)(t2 / B), tx = (int)(t2 - (uint32_t)ty * B);
    uint8_t* rec = tiles + (size_t)tc * G::REC_I8;
    uint32_t words[2 * G::NW];                         // this lane's bit words [cc * NW + gx]: TOP for Y = 0, BOT for Y = LPT-1
#pragma unroll
    for (int i = 0; i < 2 * G::NW; ++i) words[i] = 0;
    uint32_t col[4];                                    // L0, L1, R0, R1 ballots
#pragma unroll
    for (int rp = 1; rp >= 0; --rp) {                   // row 2Y+1 first: pack16 shifts the earlier half up
        const int8_t* rowp = canon + (size_t)r * L * L + (size_t)(ty * T + 2 * Y + rp) * L + (size_t)tx * T;
        bool left = false, right = false;
#pragma unroll
        for (int gx = 0; gx < G::NW; ++gx) {
            uint4 a = make_uint4(0, 0, 0, 0), b = a;
            if (live) {
                a = __ldg(reinterpret_cast<const uint4*>(rowp + 32 * gx));
                b = __ldg(reinterpret_cast<const uint4*>(rowp + 32 * gx + 16));
            }
            uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
            for (int i = 0; i < 8; ++i) w[i] = ~(w[i] >> 1) & 0x01010101u;         // +1 (0x01) -> 1, -1 (0xff) -> 0
            if (gx == 0) left = (w[0] & 1u) != 0;
            if (gx == G::NW - 1) right = (w[7] >> 24) != 0;
            uint4 pe, po;                                // even bytes (a = 0) and odd bytes (a = 1) of the run
            {
                const uint32_t e01 = __byte_perm(w[0], w[1], 0x6240), e23 = __byte_perm(w[2], w[3], 0x6240);
                const uint32_t e45 = __byte_perm(w[4], w[5], 0x6240), e67 = __byte_perm(w[6], w[7], 0x6240);
                pe = make_uint4(__byte_perm(e01, e23, 0x5410), __byte_perm(e01, e23, 0x7632), __byte_perm(e45, e67, 0x5410), __byte_perm(e45, e67, 0x7632));
                const uint32_t o01 = __byte_perm(w[0], w[1], 0x7351), o23 = __byte_perm(w[2], w[3], 0x7351);
                const uint32_t o45 = __byte_perm(w[4], w[5], 0x7351), o67 = __byte_perm(w[6], w[7], 0x7351);
                po = make_uint4(__byte_perm(o01, o23, 0x5410), __byte_perm(o01, o23, 0x7632), __byte_perm(o45, o67, 0x5410), __byte_perm(o45, o67, 0x7632));
            }
            // a = (cc + ly) & 1 and ly = 2Y + rp: the even bytes are colour rp, the odd bytes colour 1 - rp
#pragma unroll
            for (int odd = 0; odd < 2; ++odd) {
                const int cc = odd ? 1 - rp : rp;
                const uint4 piece = odd ? po : pe;
                if (live) *reinterpret_cast<uint4*>(rec + ((((rp * 2 + cc) * G::NW + gx) * G::LPT) + Y) * 16) = piece;
                words[cc * G::NW + gx] = pack16(words[cc * G::NW + gx], piece);
            }
        }
        col[0 + rp] = __ballot_sync(0xffffffffu, left);
        col[2 + rp] = __ballot_sync(0xffffffffu, right);
    }
    if (!live) return;
    const int sh = (lane / G::LPT) * G::LPT;                                       // T = 32: this tile's half of the ballot
    const uint32_t mask = G::LPT == 32 ? 0xffffffffu : ((1u << G::LPT) - 1u);
    uint32_t* e = reinterpret_cast<uint32_t*>(rec + G::BODY);
    if (Y == 0) {
        uint32_t top[4] = {0, 0, 0, 0};
#pragma unroll
        for (int i = 0; i < 2 * G::NW; ++i) top[i] = words[i];
        *reinterpret_cast<uint4*>(e + 0) = make_uint4(top[0], top[1], top[2], top[3]);
        *reinterpret_cast<uint4*>(e + 4) = make_uint4((col[0] >> sh) & mask, (col[1] >> sh) & mask, (col[2] >> sh) & mask, (col[3] >> sh) & mask);
        *reinterpret_cast<uint4*>(e + 12) = make_uint4(0, 0, 0, 0);
    }
    if (Y == G::LPT - 1) {
        uint32_t bot[4] = {0, 0, 0, 0};
#pragma unroll
        for (int i = 0; i < 2 * G::NW; ++i) bot[i] = words[i];
        *reinterpret_cast<uint4*>(e + 8) = make_uint4(bot[0], bot[1], bot[2], bot[3]);
    }
}

// Records -> canonical rows.  A lane owns a block row (two tile rows), so a direct store would scatter every 16-byte store
// instruction over 32 different rows (round 1: 3.4 TB/s, LG throttle 19.5 per issue); the tile is therefore staged in shared
// memory (per warp, 128-byte blocks of 8 swizzled 16-byte chunks: conflict-free both ways) and written out as whole rows.
template <int T>
__global__ void __launch_bounds__(256) k_planes_i8_to_canon(int8_t* __restrict__ canon, const uint8_t* __restrict__ tiles,
                                                            int L, int B, uint32_t ntiles) {
    using G = PG<T>;
    __shared__ __align__(16) uint8_t stage_all[8][4096];
    const int lane = threadIdx.x & 31;
    const uint32_t warp = (uint32_t)((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    const uint32_t tile = warp * G::TPW + (uint32_t)(lane / G::LPT);
    const int Y = lane % G::LPT;
    if (tile >= ntiles) return;                              // whole warps only: ntiles is even
    uint8_t* stage = stage_all[threadIdx.x >> 5];
    const uint8_t* rec = tiles + (size_t)tile * G::REC_I8;
    // where chunk c (16 bytes) of row 2Y + rp of this lane's tile goes
    const int blk = T == 64 ? Y : lane >> 1;
    auto slot = [&](int rp, int c) { return blk * 128 + ((((T == 64 ? rp * 4 : (lane & 1) * 4 + rp * 2) + c) ^ (blk & 7)) << 4); };
#pragma unroll
    for (int rp = 0; rp < 2; ++rp) {
#pragma unroll
        for (int gx = 0; gx < G::NW; ++gx) {
            // even bytes of the run = colour rp, odd bytes = colour 1 - rp
            const uint4 pe = __ldg(reinterpret_cast<const uint4*>(rec + ((((rp * 2 + rp) * G::NW + gx) * G::LPT) + Y) * 16));
            const uint4 po = __ldg(reinterpret_cast<const uint4*>(rec + ((((rp * 2 + 1 - rp) * G::NW + gx) * G::LPT) + Y) * 16));
            uint32_t w[8];
            // word m of the run = sites k = 2m (piece word 0/2, byte m & 3) and 2m+1 (piece word 1/3) of both colours:
            // bytes {pe[k=2m], po[k=2m], pe[k=2m+1], po[k=2m+1]}
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                const uint32_t ee = half ? pe.z : pe.x, eo = half ? pe.w : pe.y;      // colour "even byte": k even, k odd
                const uint32_t oe = half ? po.z : po.x, oo = half ? po.w : po.y;
                const uint32_t lo_e = __byte_perm(ee, oe, 0x5140), hi_e = __byte_perm(ee, oe, 0x7362);   // (ee.b0, oe.b0, ee.b1, oe.b1), (.b2, .b3)
                const uint32_t lo_o = __byte_perm(eo, oo, 0x5140), hi_o = __byte_perm(eo, oo, 0x7362);
                w[4 * half + 0] = __byte_perm(lo_e, lo_o, 0x5410);        // k = 0 (both colours), k = 1 (both colours)
                w[4 * half + 1] = __byte_perm(lo_e, lo_o, 0x7632);        // k = 2, 3
                w[4 * half + 2] = __byte_perm(hi_e, hi_o, 0x5410);        // k = 4, 5
                w[4 * half + 3] = __byte_perm(hi_e, hi_o, 0x7632);        // k = 6, 7
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) w[i] = ((w[i] ^ 0x01010101u) * 255u) | w[i];   // 1 -> 0x01, 0 -> 0xff
            *reinterpret_cast<uint4*>(stage + slot(rp, 2 * gx)) = make_uint4(w[0], w[1], w[2], w[3]);
            *reinterpret_cast<uint4*>(stage + slot(rp, 2 * gx + 1)) = make_uint4(w[4], w[5], w[6], w[7]);
        }
    }
    __syncwarp();
    // out: instruction i writes bytes [512 i, 512 i + 512) of the warp's tiles in row-major order, 16 bytes per lane
    const uint32_t per_rep = (uint32_t)B * B;
#pragma unroll
    for (int i = 0; i < G::TPW * T * T / 512; ++i) {
        const int s = (512 * i) / (T * T), o = (512 * i) % (T * T) + 16 * lane;
        const int row = o / T, c = (o % T) >> 4, y = row >> 1, rp = row & 1;
        const int lsrc = s * G::LPT + y, bsrc = T == 64 ? y : lsrc >> 1;
        const int src = bsrc * 128 + ((((T == 64 ? rp * 4 : (lsrc & 1) * 4 + rp * 2) + c) ^ (bsrc & 7)) << 4);
        const uint32_t tl = warp * G::TPW + (uint32_t)s;
        const uint32_t r = tl / per_rep, t2 = tl - r * per_rep;
        const int ty = (int)(t2 / B), tx = (int)(t2 - (uint32_t)ty * B);
        int8_t* dst = canon + (size_t)r * L * L + (size_t)(ty * T + row) * L + (size_t)tx * T + 16 * c;
        *reinterpret_cast<uint4*>(dst) = *reinterpret_cast<const uint4*>(stage + src);
    }
}

// Couplings, canonical J[d][i] (bond i -> i + e_d) -> coupling records (zeroed first).  One thread per site:
// it owns the four bonds seen from that site, in the order of the neighbour words of update_block.
__global__ void k_convert_couplings(const int8_t* __restrict__ J, uint32_t* __restrict__ jrec, int L, int T) {
    const uint64_t N = (uint64_t)L * L;
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int x = (int)(i % L), y = (int)(i / L);
    const int B = L / T, NW = T / 32, LPT = T / 2;
    const int tx = x / T, ty = y / T, lx = x - tx * T, ly = y - ty * T;
    const int cc = (lx + ly) & 1, px = lx >> 1, gx = px >> 4, kk = px & 15, rp = ly & 1, Y = ly >> 1;
    const uint64_t iL = (uint64_t)(x == 0 ? L - 1 : x - 1) + (uint64_t)L * y;         // site to the left
    const uint64_t iU = (uint64_t)x + (uint64_t)L * (y == 0 ? L - 1 : y - 1);         // site above (y - 1)
    const bool right = J[i] < 0, left = J[iL] < 0, down = J[N + i] < 0, up = J[N + iU] < 0;
    const bool v1 = rp == 0 ? down : up;          // V1 = the other row of the block
    const bool v2 = rp == 0 ? up : down;          // V2 = the row outside the block
    const bool h1 = (x & 1) == 0 ? right : left;  // H1 = the other site of the aligned pair (2p_x, 2p_x + 1)
    const bool h2 = (x & 1) == 0 ? left : right;
    uint32_t* w = jrec + (((size_t)ty * B + tx) * (2 * NW * LPT) + (cc * NW + gx) * LPT + Y) * 4;
    const uint32_t bit = 1u << (rp * 16 + kk);
    if (v1) atomicOr(w + 0, bit);
    if (v2) atomicOr(w + 1, bit);
    if (h1) atomicOr(w + 2, bit);
    if (h2) atomicOr(w + 3, bit);
}

// tiles per lane (k_tile_planes NS): two for tile 32 where the tile rows allow it, so that a warp job is 4096 sites at either
// tile edge; ISING_SLOTS overrides (testing / tuning aid)
static int plane_slots(int T, int B) {
    static const int forced = getenv("ISING_SLOTS") ? atoi(getenv("ISING_SLOTS")) : 0;
    int ns = forced ? forced : (T == 32 ? 2 : 1);
    if (ns != 1 && ns != 2) ns = 1;
    if ((B / 2) % ns) ns = 1;
    return ns;
}

template <int T, bool BITS, int NS>
int launch_colour_planes(PlaneArgs A, bool use_jit, bool* used_jit) {
    const int warps = kPlaneThreads / 32;
    A.njobs /= (uint32_t)NS;
    const uint32_t grid = (A.njobs + warps - 1) / warps;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(warps * 32); cfg.dynamicSmemBytes = 0; cfg.stream = hooks().stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    static const int pdl = getenv("ISING_NO_PDL") ? 0 : 1;
    attr[0].val.programmaticStreamSerializationAllowed = pdl;
    cfg.attrs = attr; cfg.numAttrs = 1;
    // specialised on the threshold head bits (planes_jit.cu) when asked for and available, else run-time operands
    cudaKernel_t spec = (use_jit && !A.force) ? planes_jit_kernel(T, BITS, A.jrec != nullptr, A.hp, A.B, A.R, NS) : nullptr;
    if (spec) {
        void* args[] = {&A};
        ISING_CUDA_OK(cudaLaunchKernelExC(&cfg, (const void*)spec, args));
    } else if (A.jrec) {
        ISING_CUDA_OK((cudaLaunchKernelEx(&cfg, k_tile_planes<T, BITS, true, kNoSpec, NS>, A)));
    } else {
        ISING_CUDA_OK((cudaLaunchKernelEx(&cfg, k_tile_planes<T, BITS, false, kNoSpec, NS>, A)));
    }
    if (used_jit) *used_jit = spec != nullptr;
    count_launch();
    return 0;
}

template <int T, bool BITS>
int launch_colour_planes(const PlaneArgs& A, bool use_jit, bool* used_jit) {
    return plane_slots(T, A.B) == 2 ? launch_colour_planes<T, BITS, 2>(A, use_jit, used_jit) : launch_colour_planes<T, BITS, 1>(A, use_jit, used_jit);
}

}  // namespace

bool tile_planes_supported(const ising_ctx* h, int T) {
    if (h->dim != 2 || h->J_per_replica) return false;     // coupling records are shared by the replicas
    if (T != 32 && T != 64) return false;
    if (h->L % T) return false;
    const int B = h->L / T;
    return B >= 2 && (B % 2 == 0);
}

size_t coupling_record_bytes(const ising_ctx* h) { return (size_t)h->N / 2 * 4; }   // 4 bond bits per site

int launch_convert_couplings(ising_ctx* h, int T, void* d_jrec) {
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemsetAsync(d_jrec, 0, coupling_record_bytes(h), st));
    k_convert_couplings<<<(unsigned)((h->N + 255) / 256), 256, 0, st>>>(h->d_J, (uint32_t*)d_jrec, h->L, T);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

size_t tile_planes_bytes(const ising_ctx* h, int T, bool bits) {
    const size_t B = (size_t)(h->L / T);
    return (size_t)h->R * B * B * (size_t)((bits ? T * T / 8 : T * T) + 64);
}

int launch_canon_to_planes(ising_ctx* h, int T, bool bits, const int8_t* d_canon, void* d_tiles) {
    const uint64_t total = h->N * (uint64_t)h->R;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    cudaStream_t st = hooks().stream;
    if (!bits) {                                  // fast path: a warp per tile, whole sectors on both sides
        const uint32_t ntiles = (uint32_t)h->R * (uint32_t)(h->L / T) * (uint32_t)(h->L / T);
        const uint32_t warps = (ntiles + (64 / T) - 1) / (64 / T);
        const unsigned grid = (warps + 7) / 8;
        if (T == 64) k_canon_to_planes_i8<64><<<grid, 256, 0, st>>>(d_canon, (uint8_t*)d_tiles, h->L, h->L / T, ntiles);
        else k_canon_to_planes_i8<32><<<grid, 256, 0, st>>>(d_canon, (uint8_t*)d_tiles, h->L, h->L / T, ntiles);
        count_launch();
        ISING_CUDA_OK(cudaGetLastError());
        return 0;
    }
    ISING_CUDA_OK(cudaMemsetAsync(d_tiles, 0, tile_planes_bytes(h, T, bits), st));
    k_convert_planes<2><<<blocks, 256, 0, st>>>(const_cast<int8_t*>(d_canon), (uint8_t*)d_tiles, h->L, T, h->R);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_planes_to_canon(ising_ctx* h, int T, bool bits, const void* d_tiles, int8_t* d_canon) {
    const uint64_t total = h->N * (uint64_t)h->R;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    cudaStream_t st = hooks().stream;
    if (!bits) {
        const uint32_t ntiles = (uint32_t)h->R * (uint32_t)(h->L / T) * (uint32_t)(h->L / T);
        const uint32_t warps = (ntiles + (64 / T) - 1) / (64 / T);
        const unsigned grid = (warps + 7) / 8;
        if (T == 64) k_planes_i8_to_canon<64><<<grid, 256, 0, st>>>(d_canon, (const uint8_t*)d_tiles, h->L, h->L / T, ntiles);
        else k_planes_i8_to_canon<32><<<grid, 256, 0, st>>>(d_canon, (const uint8_t*)d_tiles, h->L, h->L / T, ntiles);
        count_launch();
        ISING_CUDA_OK(cudaGetLastError());
        return 0;
    }
    k_convert_planes<3><<<blocks, 256, 0, st>>>(d_canon, (uint8_t*)const_cast<void*>(d_tiles), h->L, T, h->R);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

constexpr size_t kL2StreamBytes = 96u << 20;    // records larger than this do not stay in the 126 MB L2 between passes

bool plain64_supported(const ising_ctx* h, int T) { return h->dim == 2 && h->L == 64 && T == 64 && !h->J_per_replica; }

static void fill_accept(PlaneArgs& A, const Accept& acc) {
    for (int q = 0; q < kHeadBits; ++q) {
        A.u1[q] = ((acc.thr[0] >> (31 - q)) & 1u) ? 0xffffffffu : 0u;
        A.u2[q] = ((acc.thr[1] >> (31 - q)) & 1u) ? 0xffffffffu : 0u;
    }
    A.force = acc.thr_is_2p32[0] ? 0xffffffffu : 0u;       // thr[m] = 2^32 happens only at beta = 0, for every m at once
    A.hp = ((acc.thr[0] >> kTailBits) << kHeadBits) | (acc.thr[1] >> kTailBits);
    A.t1_tail = acc.thr[0] & ((1u << kTailBits) - 1u);
    A.t2_tail = acc.thr[1] & ((1u << kTailBits) - 1u);
}

// a8: all n passes of a 64x64 plain-checkerboard run in one launch, one warp per replica; d_E / d_M (n*R each) optional.
int launch_plain64(ising_ctx* h, const Accept& acc, bool bits, int n, int k, uint64_t t_first, long long* d_E, long long* d_M) {
    PlaneArgs A;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = 64; A.B = 1; A.R = h->R; A.k = k; A.t_first = t_first; A.C = 0; A.njobs = (uint32_t)h->R;
    A.magic_rep = A.magic_hb = 0;
    A.stream = 0;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    fill_accept(A, acc);
    cudaStream_t st = hooks().stream;
    if (bits) {
        if (A.jrec) k_plain64_planes<true, true><<<h->R, 32, 0, st>>>(A, n, d_E, d_M);
        else k_plain64_planes<true, false><<<h->R, 32, 0, st>>>(A, n, d_E, d_M);
    } else {
        if (A.jrec) k_plain64_planes<false, true><<<h->R, 32, 0, st>>>(A, n, d_E, d_M);
        else k_plain64_planes<false, false><<<h->R, 32, 0, st>>>(A, n, d_E, d_M);
    }
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// a10 on tile records: E[r], M[r] (R values each, either may be null) of the state held in plane records.
int launch_observables_planes(ising_ctx* h, int T, bool bits, long long* d_E, long long* d_M) {
    cudaStream_t st = hooks().stream;
    if (d_E) ISING_CUDA_OK(cudaMemsetAsync(d_E, 0, sizeof(long long) * h->R, st));
    if (d_M) ISING_CUDA_OK(cudaMemsetAsync(d_M, 0, sizeof(long long) * h->R, st));
    PlaneArgs A = {};
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = h->L; A.B = h->L / T; A.R = h->R; A.k = 0; A.t_first = 0;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    const uint32_t tiles_per_colour = (uint32_t)((size_t)h->R * A.B * A.B / 2);
    A.njobs = tiles_per_colour / (uint32_t)(64 / T);
    A.magic_rep = fastdiv_magic((uint32_t)A.B * (uint32_t)A.B / 2u);
    A.magic_hb = fastdiv_magic((uint32_t)A.B / 2u);
    const int warps = kPlaneThreads / 32;
    const uint32_t grid = (A.njobs + warps - 1) / warps;
    for (int C = 0; C < 2; ++C) {
        A.C = C;
#define ISING_OBS(TT, BB)                                                                                   \
        do {                                                                                                \
            if (A.jrec) k_observables_planes<TT, BB, true><<<grid, warps * 32, 0, st>>>(A, d_E, d_M);      \
            else k_observables_planes<TT, BB, false><<<grid, warps * 32, 0, st>>>(A, d_E, d_M);            \
        } while (0)
        if (T == 64) { if (bits) ISING_OBS(64, true); else ISING_OBS(64, false); }
        else { if (bits) ISING_OBS(32, true); else ISING_OBS(32, false); }
#undef ISING_OBS
        count_launch();
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// a1: one outer pass = colour-0 launch, colour-1 launch, k inner sweeps each.
int launch_tile_planes_pass(ising_ctx* h, const Accept& acc, int T, bool bits, int k, uint64_t t_first, bool use_jit) {
    PlaneArgs A;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = h->L; A.B = h->L / T; A.R = h->R; A.k = k; A.t_first = t_first;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    A.stream = tile_planes_bytes(h, T, bits) > kL2StreamBytes ? 1u : 0u;
    const uint32_t tiles_per_colour = (uint32_t)((size_t)h->R * A.B * A.B / 2);
    A.njobs = tiles_per_colour / (uint32_t)(64 / T);
    A.magic_rep = fastdiv_magic((uint32_t)A.B * (uint32_t)A.B / 2u);
    A.magic_hb = fastdiv_magic((uint32_t)A.B / 2u);
    fill_accept(A, acc);
    for (int C = 0; C < 2; ++C) {
        A.C = C;
        bool used = false;
        const int rc = T == 64 ? (bits ? launch_colour_planes<64, true>(A, use_jit, &used) : launch_colour_planes<64, false>(A, use_jit, &used))
                               : (bits ? launch_colour_planes<32, true>(A, use_jit, &used) : launch_colour_planes<32, false>(A, use_jit, &used));
        if (rc) return rc;
        h->last_jit = used ? 1 : 0;
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// ---- coarse tiles smaller than a register tile (the paper's own T = 4, 8, 16): the double checkerboard of
// coarse tiles Tc = 2, 4, 8, 16 (and of the powers of two above 64, where a mask is all or nothing) on the register tiling
// T in {32, 64}.  A phase (coarse colour Cc, inner sweep, fine
// colour c) is a half-sweep of the whole lattice in which only the sites of the colour-Cc coarse tiles may flip: the
// flip word is masked.  Bit j = 16 rp + kk of a block word is the site x = 32 gx + 2 kk + a, y = 2 Yg + rp, so the parity
// of x / Tc is a fixed bit pattern and that of y / Tc depends on the block row only.
__device__ __forceinline__ uint32_t coarse_mask(int Tc, uint32_t Yg, uint32_t gxg, int Cc) {
    if (Tc == 0) return 0xffffffffu;
    const uint32_t typ = ((2u * Yg) / (uint32_t)Tc) & 1u;
    if (Tc >= 32) {                                        // the 32 columns of the block lie in one coarse tile: all or nothing
        const uint32_t txp = ((32u * gxg) / (uint32_t)Tc) & 1u;
        return ((txp ^ typ ^ (uint32_t)Cc) & 1u) ? 0u : 0xffffffffu;
    }
    const uint32_t even_x = Tc == 16 ? 0x00ff00ffu : Tc == 8 ? 0x0f0f0f0fu : Tc == 4 ? 0x33333333u : 0x55555555u;
    return ((typ ^ (uint32_t)Cc) & 1u) ? ~even_x : even_x;
}

// gxg0: global block column of the lane's word gx = 0
template <int T, bool HASJ>
__device__ __forceinline__ void half_sweep_masked(const PlaneArgs& A, TileRegs<T>& t, const uint4 (&Jw)[2][PG<T>::NW], int c, int Y,
                                                  uint32_t g0, uint32_t p0, uint64_t H, uint32_t k0, uint32_t k1, int Tc, uint32_t Yg,
                                                  uint32_t gxg0, int Cc) {
    uint32_t old[PG<T>::NW];
#pragma unroll
    for (int gx = 0; gx < PG<T>::NW; ++gx) old[gx] = t.S[c][gx];
    half_sweep<T, HASJ, false, kNoSpec>(A, t, Jw, c, Y, g0, p0, H, k0, k1);
#pragma unroll
    for (int gx = 0; gx < PG<T>::NW; ++gx) {
        const uint32_t mask = coarse_mask(Tc, Yg, gxg0 + (uint32_t)gx, Cc);
        t.S[c][gx] = (t.S[c][gx] & mask) | (old[gx] & ~mask);
    }
}

// store_tile for a half-sweep that changed only fine colour c: that colour's pieces and the boundary copies (a plain-
// checkerboard half-sweep then writes half the lattice, 1.5 N bytes of traffic instead of 2 N).
template <int T, bool BITS>
__device__ __forceinline__ void store_tile_colour(const PlaneArgs& A, int r, int tx, int ty, int Y, int sub, const TileRegs<T>& t,
                                                  const uint2* lut, int c) {
    using G = PG<T>;
    constexpr uint32_t REC = BITS ? G::REC_BITS : G::REC_I8;
    constexpr uint32_t BODY = REC - G::EDGE;
    uint8_t* rec = A.tiles + (uint64_t)(((uint32_t)r * (uint32_t)A.B + (uint32_t)ty) * (uint32_t)A.B + (uint32_t)tx) * REC;
    const uint64_t pol = body_policy(A.stream != 0);
#pragma unroll
    for (int gx = 0; gx < G::NW; ++gx) {
        const uint32_t w = c ? t.S[1][gx] : t.S[0][gx];
        if (BITS) {
            *reinterpret_cast<uint32_t*>(rec + ((c * G::NW + gx) * G::LPT + Y) * 4) = w;
        } else {
#pragma unroll
            for (int rp = 0; rp < 2; ++rp) {
                const uint2 a = __ldg(lut + ((w >> (16 * rp)) & 0xffu));
                const uint2 b = __ldg(lut + ((w >> (16 * rp + 8)) & 0xffu));
                stg128(rec + ((((rp * 2 + c) * G::NW + gx) * G::LPT) + Y) * 16, make_uint4(a.x, a.y, b.x, b.y), pol);
            }
        }
    }
    const uint32_t sh = (uint32_t)sub * G::LPT, m = G::LPT == 32 ? 0xffffffffu : ((1u << G::LPT) - 1u);
    const uint32_t L0 = (__ballot_sync(0xffffffffu, t.S[0][0] & 1u) >> sh) & m;
    const uint32_t L1 = (__ballot_sync(0xffffffffu, (t.S[1][0] >> 16) & 1u) >> sh) & m;
    const uint32_t R0 = (__ballot_sync(0xffffffffu, (t.S[1][G::NW - 1] >> 15) & 1u) >> sh) & m;
    const uint32_t R1 = (__ballot_sync(0xffffffffu, t.S[0][G::NW - 1] >> 31) >> sh) & m;
    if (Y == 0 || Y == G::LPT - 1) {
        const uint4 w = G::NW == 2 ? make_uint4(t.S[0][0], t.S[0][1], t.S[1][0], t.S[1][1]) : make_uint4(t.S[0][0], t.S[1][0], 0u, 0u);
        uint8_t* e = rec + BODY + (Y == 0 ? G::E_TOP : G::E_BOT);
        stg128(e, w);
        stg128(e + 16, Y == 0 ? make_uint4(L0, L1, R0, R1) : make_uint4(0u, 0u, 0u, 0u));
    }
}

// ---- a8 for large lattices: the plain checkerboard (tile == L) with a launch per half-sweep.  Every tile of the
// register tiling T takes part: load (neighbours' boundary copies of the other fine colour are not being changed by
// this launch), one half-sweep of fine colour c, store.  The scheme the paper starts from: the whole lattice
// crosses HBM twice per sweep, which is what the double checkerboard's k inner sweeps per load avoid.
template <int T, bool BITS, bool HASJ>
__global__ void __launch_bounds__(kPlaneThreads) k_tile_planes_plain(PlaneArgs A, int c, uint64_t tt, int Tc, int Cc) {
    using G = PG<T>;
    const uint2* lut = kByteLutGlobal.e;
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int lane = threadIdx.x & 31;
    const uint32_t job = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (job >= A.njobs) return;
    const int sub = lane / G::LPT, Y = lane % G::LPT;
    const uint32_t B = (uint32_t)A.B, q = job * G::TPW + (uint32_t)sub;        // all tiles, replica-major, row-major
    const int r = (int)(q / (B * B));
    const uint32_t qq = q - (uint32_t)r * B * B;
    const int ty = (int)(qq / B), tx = (int)(qq - (uint32_t)ty * B);
    TileRegs<T> t;
    load_tile<T, BITS>(A, r, tx, ty, Y, sub * G::LPT, t);
    uint4 Jw[2][G::NW];
#pragma unroll
    for (int cc = 0; cc < 2; ++cc)
#pragma unroll
        for (int gx = 0; gx < G::NW; ++gx)
            Jw[cc][gx] = HASJ ? __ldg(A.jrec + ((size_t)ty * B + tx) * (2 * G::NW * G::LPT) + (cc * G::NW + gx) * G::LPT + Y)
                              : make_uint4(0u, 0u, 0u, 0u);
    const uint64_t seed = A.seeds[r];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    const uint32_t Yg = (uint32_t)(ty * G::LPT + Y);
    const uint32_t g0 = Yg * (B * G::NW) + (uint32_t)(tx * G::NW);
    const uint32_t p0 = 2u * Yg * (B * (uint32_t)(T / 2)) + 16u * (uint32_t)(tx * G::NW);
    half_sweep_masked<T, HASJ>(A, t, Jw, c, Y, g0, p0, 2 * tt + (uint64_t)c, k0, k1, Tc, Yg, (uint32_t)(tx * G::NW), Cc);
    store_tile_colour<T, BITS>(A, r, tx, ty, Y, sub, t, lut, c);
}

// n passes of k plain-checkerboard sweeps: 2 n k launches; with coarse tiles Tc (0: none) n passes of the double
// checkerboard of Tc-tiles: 4 n k launches.
int launch_tile_planes_plain(ising_ctx* h, const Accept& acc, int T, bool bits, int n, int k, uint64_t t_first, int Tc) {
    PlaneArgs A;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = h->L; A.B = h->L / T; A.R = h->R; A.k = k; A.t_first = t_first; A.C = 0;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    A.stream = tile_planes_bytes(h, T, bits) > kL2StreamBytes ? 1u : 0u;
    A.njobs = (uint32_t)((size_t)h->R * A.B * A.B / (size_t)(64 / T));
    A.magic_rep = A.magic_hb = 0;
    fill_accept(A, acc);
    const int warps = kPlaneThreads / 32;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((A.njobs + warps - 1) / warps); cfg.blockDim = dim3(warps * 32); cfg.dynamicSmemBytes = 0; cfg.stream = hooks().stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    static const int pdl = getenv("ISING_NO_PDL") ? 0 : 1;
    attr[0].val.programmaticStreamSerializationAllowed = pdl;
    cfg.attrs = attr; cfg.numAttrs = 1;
    for (int pass = 0; pass < n; ++pass)
        for (int Cc = 0; Cc < (Tc ? 2 : 1); ++Cc)
            for (int j = 0; j < k; ++j)
                for (int c = 0; c < 2; ++c) {
                    const uint64_t tt = t_first + (uint64_t)pass * (uint64_t)k + (uint64_t)j;
#define ISING_PLAIN(TT, BB)                                                                                                  \
                    do {                                                                                                     \
                        if (A.jrec) ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile_planes_plain<TT, BB, true>, A, c, tt, Tc, Cc));    \
                        else ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile_planes_plain<TT, BB, false>, A, c, tt, Tc, Cc));          \
                    } while (0)
                    if (T == 64) { if (bits) ISING_PLAIN(64, true); else ISING_PLAIN(64, false); }
                    else { if (bits) ISING_PLAIN(32, true); else ISING_PLAIN(32, false); }
#undef ISING_PLAIN
                    count_launch();
                }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// ---- whole lattice on chip ("a persistent whole-lattice-on-chip kernel for small L") ----------------
// For L <= 512 a pass of the tile kernel is two launches whose duration is launch latency + one L2 round trip, not
// work.  Here one thread-block cluster per replica keeps every tile in registers for the whole call: warp w of the
// cluster owns the jobs w, w + W, ... of each coarse colour (a job = 64 / T tiles, lane = block row, exactly as in
// k_tile_planes), a tile publishes its boundary words (TOP / COL / BOT of PG) in the shared memory of its CTA after
// every phase, its neighbours — of the other colour, so idle in that phase — read them through distributed shared
// memory at the start of theirs, and the two coarse-colour phases of a pass are separated by cluster barriers
// instead of kernel boundaries.  HBM is touched twice: records in at the start, records out at the end.
constexpr int kResWarps = 4;       // warps per CTA: one per SM sub-partition
constexpr int kResMaxJobs = 1;     // jobs per warp and colour: with more, 16 SMs are slower than per-pass launches on 148 (measured at L = 1024)
constexpr int kResMaxCluster = 16;

struct ResArgs {
    PlaneArgs P;
    int n;                         // outer passes
    uint32_t jobs_per_colour;      // per replica
    long long* E;                  // optional series (a10 after every pass): E[pass * R + r], M[pass * R + r]
    long long* M;
    int plain;                     // 1: the plain checkerboard of the whole lattice (tile == L, a8): every tile takes part in
                                   // every half-sweep, a barrier after each; T is then only how the lattice is cut into registers
    int coarse;                    // with plain: coarse tile edge Tc in {2, 4, 8, 16} of a masked double checkerboard, or 0
};

template <int T, bool BITS, bool HASJ>
__global__ void __launch_bounds__(kResWarps * 32) k_resident_planes(ResArgs R) {
    using G = PG<T>;
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    const uint32_t CL = cluster.num_blocks(), rank = cluster.block_rank();
    const PlaneArgs& A = R.P;
    const int r = (int)(blockIdx.x / CL);                              // one cluster per replica
    const int lane = threadIdx.x & 31, wic = threadIdx.x >> 5;
    const uint32_t wg = rank * kResWarps + (uint32_t)wic, W = CL * kResWarps;
    const int sub = lane / G::LPT, Y = lane % G::LPT;
    const uint32_t B = (uint32_t)A.B, hb = B >> 1, JC = R.jobs_per_colour;
    const uint2* lut = kByteLutGlobal.e;
    __shared__ __align__(16) uint32_t edges[2][kResMaxJobs][kResWarps][G::TPW][12];
    __shared__ int acc[2][2];          // rank 0 only: {#up, #unsatisfied bonds} of the replica, for even / odd passes
    if (threadIdx.x < 4) (&acc[0][0])[threadIdx.x] = 0;
    int* const acc0 = cluster.map_shared_rank(&acc[0][0], 0);
    const bool series = R.E != nullptr || R.M != nullptr;
    const long long nsites = (long long)A.L * A.L;
    auto write_series = [&](int pass) {                                // by one thread of the cluster, a barrier after the atomics
        if (rank == 0 && threadIdx.x == 0) {
            int* a = &acc[pass & 1][0];
            if (R.M) R.M[(size_t)pass * A.R + r] = 2ll * a[0] - nsites;
            if (R.E) R.E[(size_t)pass * A.R + r] = 2ll * a[1] - 2ll * nsites;
            a[0] = 0; a[1] = 0;
        }
    };

    auto tile_of = [&](int C, uint32_t job, int& tx, int& ty) {
        const uint32_t qq = job * G::TPW + (uint32_t)sub;
        ty = (int)(qq / hb);
        tx = (int)(2u * (qq - (uint32_t)ty * hb)) + ((ty + C) & 1);
    };
    auto edge_of = [&](uint32_t tx, uint32_t ty) -> const uint32_t* {   // published words of tile (tx, ty), anywhere in the cluster
        const uint32_t C = (tx + ty) & 1u, qq = ty * hb + (tx >> 1);
        const uint32_t job = qq / G::TPW, sb = qq % G::TPW, w = job % W, m = job / W;
        return cluster.map_shared_rank(&edges[C][m][w % kResWarps][sb][0], w / kResWarps);
    };
    auto publish = [&](int C, int m, const TileRegs<T>& t) {
        const uint32_t sh = (uint32_t)sub * G::LPT, msk = G::LPT == 32 ? 0xffffffffu : ((1u << G::LPT) - 1u);
        const uint32_t L0 = (__ballot_sync(0xffffffffu, t.S[0][0] & 1u) >> sh) & msk;
        const uint32_t L1 = (__ballot_sync(0xffffffffu, (t.S[1][0] >> 16) & 1u) >> sh) & msk;
        const uint32_t R0 = (__ballot_sync(0xffffffffu, (t.S[1][G::NW - 1] >> 15) & 1u) >> sh) & msk;
        const uint32_t R1 = (__ballot_sync(0xffffffffu, t.S[0][G::NW - 1] >> 31) >> sh) & msk;
        uint32_t* e = &edges[C][m][wic][sub][0];
        const uint4 w = G::NW == 2 ? make_uint4(t.S[0][0], t.S[0][1], t.S[1][0], t.S[1][1]) : make_uint4(t.S[0][0], t.S[1][0], 0u, 0u);
        if (Y == 0) {
            *reinterpret_cast<uint4*>(e + G::E_TOP / 4) = w;
            *reinterpret_cast<uint4*>(e + G::E_COL / 4) = make_uint4(L0, L1, R0, R1);
        }
        if (Y == G::LPT - 1) *reinterpret_cast<uint4*>(e + G::E_BOT / 4) = w;
    };
    struct Nb { const uint32_t *up, *dn, *lf, *rt; };                  // the four neighbours' published words (fixed for the run)
    auto neighbours = [&](int tx, int ty) {
        const uint32_t utx = (uint32_t)tx, uty = (uint32_t)ty;
        const uint32_t tyU = uty == 0 ? B - 1 : uty - 1, tyD = uty == B - 1 ? 0 : uty + 1;
        const uint32_t txL = utx == 0 ? B - 1 : utx - 1, txR = utx == B - 1 ? 0 : utx + 1;
        return Nb{edge_of(utx, tyU), edge_of(utx, tyD), edge_of(txL, uty), edge_of(txR, uty)};
    };
    auto refresh = [&](const Nb& nb, TileRegs<T>& t) {                 // halos from the neighbours' published words
        uint4 hv = make_uint4(0u, 0u, 0u, 0u);
        if (Y == 0) hv = *reinterpret_cast<const uint4*>(nb.up + G::E_BOT / 4);
        else if (Y == G::LPT - 1) hv = *reinterpret_cast<const uint4*>(nb.dn + G::E_TOP / 4);
        t.vrow[0][0] = hv.x;
        if (G::NW == 2) { t.vrow[0][1] = hv.y; t.vrow[1][0] = hv.z; t.vrow[1][1] = hv.w; }
        else t.vrow[1][0] = hv.y;
        const uint2 cl = *reinterpret_cast<const uint2*>(nb.lf + G::E_COL / 4 + 2);   // {R0, R1}
        const uint2 cr = *reinterpret_cast<const uint2*>(nb.rt + G::E_COL / 4);       // {L0, L1}
        t.hL0 = (cl.x >> Y) & 1u; t.hL1 = (cl.y >> Y) & 1u;
        t.hR0 = (cr.x >> Y) & 1u; t.hR1 = (cr.y >> Y) & 1u;
    };

    TileRegs<T> t[2][kResMaxJobs];
    int txs[2][kResMaxJobs], tys[2][kResMaxJobs];
    Nb nbs[2][kResMaxJobs];
    uint4 Jws[2][kResMaxJobs][2][G::NW];                               // coupling words of the tiles (a9), zero for J = +1
#pragma unroll
    for (int C = 0; C < 2; ++C)
#pragma unroll
        for (int m = 0; m < kResMaxJobs; ++m) {
            const uint32_t job = wg + (uint32_t)m * W;
            if (job < JC) {
                tile_of(C, job, txs[C][m], tys[C][m]);
                nbs[C][m] = neighbours(txs[C][m], tys[C][m]);
#pragma unroll
                for (int cc = 0; cc < 2; ++cc)
#pragma unroll
                    for (int gx = 0; gx < G::NW; ++gx)
                        Jws[C][m][cc][gx] = HASJ ? __ldg(A.jrec + ((size_t)tys[C][m] * B + txs[C][m]) * (2 * G::NW * G::LPT) + (cc * G::NW + gx) * G::LPT + Y)
                                                 : make_uint4(0u, 0u, 0u, 0u);
                load_tile<T, BITS>(A, r, txs[C][m], tys[C][m], Y, sub * G::LPT, t[C][m]);
                publish(C, m, t[C][m]);
            }
        }
    cluster.sync();

    const uint64_t seed = A.seeds[r];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int pass = 0; pass < R.n && R.plain; ++pass) {                 // a8: fine colour 0 of every tile, barrier, fine colour 1, barrier
      for (int Cc = 0; Cc < (R.coarse ? 2 : 1); ++Cc)                   // (masked double checkerboard: both coarse colours in turn)
        for (int j = 0; j < A.k; ++j) {
            const uint64_t tt = A.t_first + (uint64_t)pass * (uint64_t)A.k + (uint64_t)j;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                if (series && Cc == 0 && j == 0 && c == 1 && pass > 0) write_series(pass - 1);
#pragma unroll
                for (int C = 0; C < 2; ++C)
#pragma unroll
                    for (int m = 0; m < kResMaxJobs; ++m) {
                        const uint32_t job = wg + (uint32_t)m * W;
                        if (job < JC) {
                            const int tx = txs[C][m], ty = tys[C][m];
                            refresh(nbs[C][m], t[C][m]);
                            const uint32_t Yg = (uint32_t)(ty * G::LPT + Y);
                            const uint32_t g0 = Yg * (B * G::NW) + (uint32_t)(tx * G::NW);
                            const uint32_t p0 = 2u * Yg * (B * (uint32_t)(T / 2)) + 16u * (uint32_t)(tx * G::NW);
                            half_sweep_masked<T, HASJ>(A, t[C][m], Jws[C][m], c, Y, g0, p0, 2 * tt + (uint64_t)c, k0, k1, R.coarse, Yg, (uint32_t)(tx * G::NW), Cc);
                            publish(C, m, t[C][m]);
                        }
                    }
                cluster.sync();
            }
        }
        if (series) {
            int up = 0, unsat = 0;
#pragma unroll
            for (int C = 0; C < 2; ++C)
#pragma unroll
                for (int m = 0; m < kResMaxJobs; ++m) {
                    const uint32_t job = wg + (uint32_t)m * W;
                    if (job < JC) {
                        refresh(nbs[C][m], t[C][m]);
                        count_row<T, false>(t[C][m], Jws[C][m], Y, up, unsat);
                    }
                }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                up += __shfl_xor_sync(0xffffffffu, up, d);
                unsat += __shfl_xor_sync(0xffffffffu, unsat, d);
            }
            if (lane == 0) {
                atomicAdd(acc0 + 2 * (pass & 1), up);
                atomicAdd(acc0 + 2 * (pass & 1) + 1, unsat);
            }
        }
    }
    for (int pass = 0; pass < R.n && !R.plain; ++pass) {
#pragma unroll
        for (int C = 0; C < 2; ++C) {
            // the previous pass's sums were added after its last barrier and are complete since the barrier just passed
            if (series && C == 1 && pass > 0) write_series(pass - 1);
#pragma unroll
            for (int m = 0; m < kResMaxJobs; ++m) {
                const uint32_t job = wg + (uint32_t)m * W;
                if (job < JC) {
                    const int tx = txs[C][m], ty = tys[C][m];
                    refresh(nbs[C][m], t[C][m]);
                    const uint32_t Yg = (uint32_t)(ty * G::LPT + Y);
                    const uint32_t g0 = Yg * (B * G::NW) + (uint32_t)(tx * G::NW);
                    const uint32_t p0 = 2u * Yg * (B * (uint32_t)(T / 2)) + 16u * (uint32_t)(tx * G::NW);
                    for (int j = 0; j < A.k; ++j) {
                        const uint64_t tt = A.t_first + (uint64_t)pass * (uint64_t)A.k + (uint64_t)j;
                        half_sweep<T, HASJ, false, kNoSpec>(A, t[C][m], Jws[C][m], 0, Y, g0, p0, 2 * tt, k0, k1);
                        half_sweep<T, HASJ, false, kNoSpec>(A, t[C][m], Jws[C][m], 1, Y, g0, p0, 2 * tt + 1, k0, k1);
                    }
                    publish(C, m, t[C][m]);
                }
            }
            cluster.sync();
        }
        if (series) {
            // a10 on the registers: every bond has one end of fine colour 0; the colour-0 tiles' halos are one phase
            // old, the colour-1 tiles' are current.  Sums go to rank 0 (alternating slots, so that the thread that
            // writes pass p out, one barrier later, never meets the atomics of pass p + 1).
            int up = 0, unsat = 0;
#pragma unroll
            for (int C = 0; C < 2; ++C)
#pragma unroll
                for (int m = 0; m < kResMaxJobs; ++m) {
                    const uint32_t job = wg + (uint32_t)m * W;
                    if (job < JC) {
                        if (C == 0) refresh(nbs[C][m], t[C][m]);
                        count_row<T, false>(t[C][m], Jws[C][m], Y, up, unsat);
                    }
                }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                up += __shfl_xor_sync(0xffffffffu, up, d);
                unsat += __shfl_xor_sync(0xffffffffu, unsat, d);
            }
            if (lane == 0) {
                atomicAdd(acc0 + 2 * (pass & 1), up);
                atomicAdd(acc0 + 2 * (pass & 1) + 1, unsat);
            }
        }
    }
    if (series && R.n > 0) {
        cluster.sync();
        write_series(R.n - 1);
    }
#pragma unroll
    for (int C = 0; C < 2; ++C)
#pragma unroll
        for (int m = 0; m < kResMaxJobs; ++m) {
            const uint32_t job = wg + (uint32_t)m * W;
            if (job < JC) store_tile<T, BITS>(A, r, txs[C][m], tys[C][m], Y, sub, t[C][m], lut);
        }
    cluster.sync();            // no CTA leaves while its shared memory may still be read or added to
}

bool resident_planes_supported(const ising_ctx* h, int T) {
    if (!tile_planes_supported(h, T)) return false;
    const uint32_t B = (uint32_t)(h->L / T);
    return B * B / 2u / (uint32_t)(64 / T) <= (uint32_t)(kResMaxCluster * kResWarps * kResMaxJobs);
}

template <int T, bool BITS, bool HASJ>
static int launch_resident(const ResArgs& R, int replicas) {
    const uint32_t want = (R.jobs_per_colour + kResWarps - 1) / kResWarps;
    unsigned cl = 1;
    while (cl < want && cl < (unsigned)kResMaxCluster) cl *= 2;
    if (cl > 8) ISING_CUDA_OK(cudaFuncSetAttribute(k_resident_planes<T, BITS, HASJ>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cl * (unsigned)replicas); cfg.blockDim = dim3(kResWarps * 32); cfg.dynamicSmemBytes = 0; cfg.stream = hooks().stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cl; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_resident_planes<T, BITS, HASJ>, R));
    count_launch();
    return 0;
}

// n passes in one launch; the records must hold the state (ensure_store) and are current again afterwards.
int launch_resident_planes(ising_ctx* h, const Accept& acc, int T, bool bits, int n, int k, uint64_t t_first,
                           long long* d_E, long long* d_M, bool plain, int Tc) {
    ResArgs R;
    R.E = d_E; R.M = d_M;
    R.plain = plain ? 1 : 0;
    R.coarse = plain ? Tc : 0;
    PlaneArgs& A = R.P;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = h->L; A.B = h->L / T; A.R = h->R; A.k = k; A.t_first = t_first; A.C = 0;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;        // shared by the replicas
    A.stream = 0;
    A.njobs = 0; A.magic_rep = A.magic_hb = 0;
    fill_accept(A, acc);
    R.n = n;
    R.jobs_per_colour = (uint32_t)A.B * (uint32_t)A.B / 2u / (uint32_t)(64 / T);
    int rc;
    if (A.jrec) rc = T == 64 ? (bits ? launch_resident<64, true, true>(R, h->R) : launch_resident<64, false, true>(R, h->R))
                             : (bits ? launch_resident<32, true, true>(R, h->R) : launch_resident<32, false, true>(R, h->R));
    else rc = T == 64 ? (bits ? launch_resident<64, true, false>(R, h->R) : launch_resident<64, false, false>(R, h->R))
                      : (bits ? launch_resident<32, true, false>(R, h->R) : launch_resident<32, false, false>(R, h->R));
    if (rc) return rc;
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// E[p][r] = 2 #unsat - 2N, M[p][r] = 2 #up - N from the slot copies of the accumulators
__global__ void k_grid_series_finish(const long long* __restrict__ acc, long long* __restrict__ E, long long* __restrict__ Mo,
                                     uint32_t count, long long nsites) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;          // pass * R + r
    if (i >= count) return;
    long long up = 0, unsat = 0;
    for (int s = 0; s < kGridAccSlots; ++s) { up += acc[((size_t)i * kGridAccSlots + s) * 2]; unsat += acc[((size_t)i * kGridAccSlots + s) * 2 + 1]; }
    if (Mo) Mo[i] = 2 * up - nsites;
    if (E) E[i] = 2 * unsat - 2 * nsites;
}

namespace {
constexpr uint32_t kGridMaxJobsPerWarp = 16;

template <int T, bool BITS, bool HASJ>
int launch_grid_one(GridArgs& R, bool use_jit, bool* fits, bool* used_jit, bool allow_pc) {
    int dev = 0, sms = 0;
    ISING_CUDA_OK(cudaGetDevice(&dev));
    ISING_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    // producer / consumer form (one consumer + three producer warps per job pair): where a warp would be alone on its scheduler
    // anyway, i.e. at most four jobs of a colour per SM (L = 1024, and L = 2048 at tile 64: measured);
    // ISING_GRID_PC = 0 / 1 overrides (tuning aid); not when the caller insists on the run-time specialised kernel
    static const int pc_mode = getenv("ISING_GRID_PC") ? atoi(getenv("ISING_GRID_PC")) : -1;
    const uint64_t total_hs = (uint64_t)R.n * 4u * (uint64_t)R.P.k;
    if (allow_pc && (pc_mode == 1 || (pc_mode < 0 && R.jobs_total <= (uint32_t)sms * 4u)) && total_hs < 0x7fffffffull) {
        const void* fn = (const void*)k_grid_planes<T, BITS, HASJ, kNoSpec, true>;
        const size_t smem = (2u * (2u * PG<T>::NW + 7u) * 32u + kPcRing * 2u * PG<T>::NW * 32u + kPcRing + 1u) * sizeof(uint32_t);
        int occ = 0;
        static const int pc_warps = getenv("ISING_GRID_PC_WARPS") ? atoi(getenv("ISING_GRID_PC_WARPS")) : 4;      // consumer + producers: 4 (default) or 8 (no faster)
        const int pc_threads = pc_warps == 4 ? 128 : 256;
        ISING_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, pc_threads, smem));
        if (R.jobs_total <= (uint32_t)sms * (uint32_t)occ) {
            R.jobs_per_warp = 1;
            R.magic_k = fastdiv_magic((uint32_t)R.P.k);
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(R.jobs_total); cfg.blockDim = dim3(pc_threads); cfg.dynamicSmemBytes = smem; cfg.stream = hooks().stream;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeCooperative;
            attr[0].val.cooperative = 1;
            cfg.attrs = attr; cfg.numAttrs = 1;
            void* args[] = {&R};
            ISING_CUDA_OK(cudaLaunchKernelExC(&cfg, fn, args));
            count_launch();
            *fits = true;
            *used_jit = false;
            return 0;
        }
    }
    // Specialised on the threshold head bits (planes_jit.cu) when asked for and available; that build also takes the CTA
    // shape the lattice wants: ONE CTA per SM with ceil(warps / SMs) warps (rounding them up to a multiple of four loses SMs: -2 % at L = 4096, tile 64), so that every
    // SM and every scheduler carries the same number of jobs (as launch_grid3d_one, measured there).
    *fits = false; *used_jit = false;
    static const uint32_t warp_cap = getenv("ISING_GRID_WARPS") ? (uint32_t)atoi(getenv("ISING_GRID_WARPS")) : 0u;   // testing aid: several jobs per warp on small lattices
    static const uint32_t wsm_cap = getenv("ISING_G2_WSM") ? (uint32_t)atoi(getenv("ISING_G2_WSM")) : 28u;        // 28 warps: 72 registers each
    static const int park_mode = getenv("ISING_G2_PARK") ? atoi(getenv("ISING_G2_PARK")) : -1;                  // testing aid: 0 = never park the constants
    bool shaped = use_jit && !R.P.force;
    // The pre-compiled kernel (fixed shape) loses to the per-pass kernels beyond two jobs of a colour per warp (BASELINE.md
    // 5.1, round 2); the shaped run-time build keeps winning (L = 8192, tile 64, k = 1 / 4 / 16: 2895 / 3303 / 3455 against
    // 2313 / 3019 / 3334 flips/ns), but a call must be long enough to pay for loading and storing the lattice once (n k >= 8
    // beyond two jobs per warp), and with 8 or 16 jobs per warp (L = 16384: all of the shared memory of the GPU holds spins)
    // its 28 warps per SM lose to the 40 of the per-pass kernels where those are not HBM-bound.  Measured at L = 16384, on
    // chip against the best other path, flips/ns: tile 64 int8 k = 1 / 2 / 4 / 16: 2896 / 3109 / 3232 / 3404 against 2486 /
    // 2962 / 3233 / 3491, bits k = 1 / 4: 3026 / 3369 against 2942 / 3315; tile 32 int8 k = 1 / 2 / 4: 2380 / 2815 / 3044
    // against 2100 / 2858 / 3185, bits k = 1: 2480 against 2836; tile 32 as strips (below), int8 k = 1 / 2 / 3 / 4: 2645 / 2983 /
    // 3107 / 3175 against 2100 / 2867 / 3083 / 3194, bits k = 1 / 2: 2685 / 3033 against 2842 / 3186.  Hence: up to k = 3; at tile 32
    // int8 records only.
    const uint32_t max_m = kGridMaxJobsPerWarp;
    constexpr size_t kSmemMax = 227 * 1024;
    for (uint32_t M = 1; M <= max_m; ++M) {
        const uint32_t warps_needed = (R.jobs_total + M - 1) / M;
        if (warp_cap && warps_needed > warp_cap && M < kGridMaxJobsPerWarp) continue;
        if (M > 2 && !warp_cap) {
            if ((uint64_t)R.n * (uint64_t)R.P.k < 8u) break;
            static const bool any = getenv("ISING_GRID_ANY") != nullptr;                   // tuning aid: on chip whatever k and layout
            if (M > 4 && !(R.P.k <= 3 && (T == 64 || !BITS)) && !any) break;               // measured at L = 16384, above
        }
        const uint32_t w_sm = (warps_needed + (uint32_t)sms - 1) / (uint32_t)sms;
        int wpb = 0;
        bool park = true;
        const void* fn = nullptr;
        const size_t lane_bytes = 32u * sizeof(uint32_t);
        if (shaped) {
            if (w_sm > wsm_cap) continue;                         // more jobs per warp
            wpb = (int)w_sm;
            park = park_mode != 0 && (size_t)wpb * 2u * M * (2u * PG<T>::NW + 7u) * lane_bytes <= kSmemMax;
            if (!park && (size_t)wpb * 2u * M * (2u * PG<T>::NW) * lane_bytes > kSmemMax) break;      // the lattice does not fit on chip
            // several jobs per warp: as a strip of adjacent tiles of one tile row where M divides the jobs of a row (ISING_G2_STRIP in
            // grid_planes_device.cuh: left / right neighbours from the warp's own shared memory); ISING_G2_STRIP=0: testing aid
            static const bool strip_ok = !(getenv("ISING_G2_STRIP") && atoi(getenv("ISING_G2_STRIP")) == 0);
            const uint32_t jobs_per_row = (uint32_t)R.P.B / 2u / (uint32_t)(64 / T);
            // tile 32 only: at tile 64 (twice the state per lane, half the exchanges per site) the extra code spills and loses 4 %
            // (and a job of two 32 x 32 tiles must not straddle tile rows: the B / 2 tiles of a colour in a row must be an even number)
            const int strip = (strip_ok && T == 32 && M >= 2 && ((uint32_t)R.P.B / 2u) % (uint32_t)(64 / T) == 0 && jobs_per_row % M == 0) ? (int)M : 0;
            fn = (const void*)grid_jit_kernel(T, BITS, HASJ, R.P.hp, R.P.B, R.P.R, wpb * 32, 1, park, R.acc != nullptr, strip);
            if (!fn) { shaped = false; M = 0; continue; }         // no run-time compiler: again with the pre-compiled kernel
            *used_jit = true;
        } else {
            if (M > 2 && !warp_cap) break;
            fn = (const void*)k_grid_planes<T, BITS, HASJ>;
            // few jobs: one warp per CTA, so that the CTAs (and the schedulers they land on) spread over all SMs
            wpb = warps_needed <= (uint32_t)sms * 4u ? 1 : (warps_needed <= (uint32_t)sms * 8u ? 2 : 4);
        }
        const size_t smem = (size_t)wpb * 2u * M * (2u * PG<T>::NW + (park ? 7u : 0u)) * lane_bytes;     // words (+ constants) of every job
        if (smem > kSmemMax) break;
        ISING_CUDA_OK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax));
        int occ = 0;
        ISING_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, wpb * 32, smem));
        const uint32_t grid = (warps_needed + wpb - 1) / wpb;
        if (grid > (uint32_t)sms * (uint32_t)occ) continue;      // not co-resident: more jobs per warp
        R.jobs_per_warp = M;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(wpb * 32); cfg.dynamicSmemBytes = smem; cfg.stream = hooks().stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeCooperative;
        attr[0].val.cooperative = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        void* args[] = {&R};
        ISING_CUDA_OK(cudaLaunchKernelExC(&cfg, fn, args));
        count_launch();
        *fits = true;
        return 0;
    }
    return 0;
}
}  // namespace

size_t grid_planes_xedge_bytes(const ising_ctx* h, int T) { return (size_t)h->R * (size_t)(h->L / T) * (size_t)(h->L / T) * 128; }
size_t grid_planes_acc_bytes(const ising_ctx* h, int n) { return (size_t)n * (size_t)h->R * kGridAccSlots * 2 * sizeof(long long); }

// n passes in one cooperative launch; returns 1 if the lattice does not fit the register files of the GPU (nothing launched).
// d_xedge: grid_planes_xedge_bytes; d_acc: grid_planes_acc_bytes(n) if a series is wanted, else nullptr.
int launch_grid_planes(ising_ctx* h, const Accept& acc, int T, bool bits, int n, int k, uint64_t t_first, void* d_xedge, void* d_acc,
                       long long* d_E, long long* d_M, bool use_jit, bool allow_pc) {
    GridArgs R;
    PlaneArgs& A = R.P;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = h->L; A.B = h->L / T; A.R = h->R; A.k = k; A.t_first = t_first; A.C = 0;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    A.stream = 0;
    A.njobs = 0;
    A.magic_rep = fastdiv_magic((uint32_t)A.B * (uint32_t)A.B / 2u);
    A.magic_hb = fastdiv_magic((uint32_t)A.B / 2u);
    fill_accept(A, acc);
    R.n = n;
    R.jobs_per_warp = 1;
    R.magic_k = 0;
    R.tiles_per_colour = (uint32_t)A.B * (uint32_t)A.B / 2u;
    R.jobs_total = (uint32_t)h->R * R.tiles_per_colour / (uint32_t)(64 / T);
    R.xedge = (unsigned long long*)d_xedge;
    const bool series = (d_E || d_M) && n > 0;
    R.acc = series ? (long long*)d_acc : nullptr;
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemsetAsync(d_xedge, 0, grid_planes_xedge_bytes(h, T), st));     // version 0 = nothing published
    if (series) ISING_CUDA_OK(cudaMemsetAsync(d_acc, 0, grid_planes_acc_bytes(h, n), st));
    bool fits = false, used = false;
    int rc;
    if (A.jrec) rc = T == 64 ? (bits ? launch_grid_one<64, true, true>(R, use_jit, &fits, &used, allow_pc) : launch_grid_one<64, false, true>(R, use_jit, &fits, &used, allow_pc))
                             : (bits ? launch_grid_one<32, true, true>(R, use_jit, &fits, &used, allow_pc) : launch_grid_one<32, false, true>(R, use_jit, &fits, &used, allow_pc));
    else rc = T == 64 ? (bits ? launch_grid_one<64, true, false>(R, use_jit, &fits, &used, allow_pc) : launch_grid_one<64, false, false>(R, use_jit, &fits, &used, allow_pc))
                      : (bits ? launch_grid_one<32, true, false>(R, use_jit, &fits, &used, allow_pc) : launch_grid_one<32, false, false>(R, use_jit, &fits, &used, allow_pc));
    if (rc) return rc;
    if (!fits) return 1;
    h->last_jit = used ? 1 : 0;
    if (series) {
        const uint32_t count = (uint32_t)n * (uint32_t)h->R;
        k_grid_series_finish<<<(count + 255) / 256, 256, 0, st>>>((const long long*)d_acc, d_E, d_M, count, (long long)h->N);
        count_launch();
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

bool grid_planes_supported(const ising_ctx* h, int T) {
    if (!tile_planes_supported(h, T)) return false;
    // the version counter is 32 bits wide: 2 n + 1 versions per call (n < 2^31) always fit; whether the state fits the shared
    // memory of the resident warps is decided at launch (launch_grid_planes returns 1 if it does not)
    const uint64_t jobs = (uint64_t)h->R * (uint64_t)(h->L / T) * (uint64_t)(h->L / T) / 2u / (uint64_t)(64 / T);
    return jobs <= 148u * 32u * kGridMaxJobsPerWarp;
}

// ---- k_grid_plain: the plain checkerboard (a8, tile == L) and the double checkerboard of coarse tiles other than the
// register tiles (the paper's own T = 2 ... 16; 128, ...) on chip on all SMs, beyond the cluster-resident kernel.
// With a launch per half-sweep the whole lattice crosses HBM twice per half-sweep and small lattices pay a launch
// latency per half-sweep (L = 1024: 125 flips/ns).  Here, as in k_grid_planes, one cooperative launch keeps every register
// tile in shared memory for the whole call; but EVERY tile takes part in every phase (a phase = one half-sweep of fine
// colour c of the whole lattice, masked to the coarse colour Cc where there are coarse tiles), so a tile's neighbours are
// being updated while it is.  A tile therefore keeps TWO exchange records, used in turn: phase p reads the neighbours'
// version p + 1 from record (p + 1) & 1 and writes its own version p + 2 into record p & 1, which held version p — read
// by the neighbours in their phase p - 1, which they had finished before they published the version p + 1 this tile has
// just waited for.  No grid barrier.
template <int T, bool BITS, bool HASJ>
__global__ void __launch_bounds__(896, 1) k_grid_plain(GridArgs R, int Tc, int split) {
    using G = PG<T>;
    constexpr int NWORDS = 2 * G::NW;                         // words per lane and job: S[cc][gx]
    constexpr int NSLOT = NWORDS + 7;                         // ... + the job's constants (decoded once): self, nU, nD, nL, nR, tx | ty << 16, r
    extern __shared__ uint32_t grid_plain_smem[];             // per warp: [colour][job][word][lane]
    const PlaneArgs& A = R.P;
    const int lane = threadIdx.x & 31, wic = threadIdx.x >> 5;
    // split (small lattices): a warp owns jobs of ONE colour of register tiles (the parity of its index), so that twice as many
    // warps share a phase; else warp w owns the jobs w, w + W, ... of both
    const uint32_t wg_all = blockIdx.x * (blockDim.x >> 5) + (uint32_t)wic, W_all = gridDim.x * (blockDim.x >> 5);
    const uint32_t wg = split ? wg_all >> 1 : wg_all, W = split ? W_all >> 1 : W_all;
    const int C0 = split ? (int)(wg_all & 1u) : 0, C1 = split ? C0 + 1 : 2;
    const int sub = lane / G::LPT, Y = lane % G::LPT;
    const uint32_t B = (uint32_t)A.B, Mw = R.jobs_per_warp;
    uint32_t* const ws = grid_plain_smem + (size_t)wic * (2u * Mw * NSLOT * 32u) + lane;
    const uint2* lut = kByteLutGlobal.e;

    struct Job { int r, tx, ty; uint32_t self, nU, nD, nL, nR; };
    auto decode = [&](uint32_t job, int C) {
        int ri, txi, tyi;
        job_tile<T>(A, job, sub, ri, txi, tyi, C);
        const uint32_t r = (uint32_t)ri, tx = (uint32_t)txi, ty = (uint32_t)tyi;
        const uint32_t base = r * B * B, row = base + ty * B;
        const uint32_t tyU = ty == 0 ? B - 1 : ty - 1, tyD = ty == B - 1 ? 0 : ty + 1;
        const uint32_t txL = tx == 0 ? B - 1 : tx - 1, txR = tx == B - 1 ? 0 : tx + 1;
        return Job{(int)r, (int)tx, (int)ty, row + tx, base + tyU * B + tx, base + tyD * B + tx, row + txL, row + txR};
    };
    // record of tile i for version v: 16 u64 = TOP[4] | {L0, L1, R0, R1} | BOT[4] | pad, u64 = version << 32 | word
    auto rec = [&](uint32_t i, uint32_t v) { return R.xedge + ((size_t)i * 2u + (v & 1u)) * 16u; };
    auto publish = [&](const TileRegs<T>& tt, const Job& jb, uint32_t ver) {
        const uint32_t sh = (uint32_t)sub * G::LPT, msk = G::LPT == 32 ? 0xffffffffu : ((1u << G::LPT) - 1u);
        const uint32_t L0 = (__ballot_sync(0xffffffffu, tt.S[0][0] & 1u) >> sh) & msk;
        const uint32_t L1 = (__ballot_sync(0xffffffffu, (tt.S[1][0] >> 16) & 1u) >> sh) & msk;
        const uint32_t R0 = (__ballot_sync(0xffffffffu, (tt.S[1][G::NW - 1] >> 15) & 1u) >> sh) & msk;
        const uint32_t R1 = (__ballot_sync(0xffffffffu, tt.S[0][G::NW - 1] >> 31) >> sh) & msk;
        const unsigned long long v = (unsigned long long)ver << 32;
        unsigned long long* e = rec(jb.self, ver);
        if (Y == 0 || Y == G::LPT - 1) {
            unsigned long long* rw = e + (Y == 0 ? 0 : 8);          // TOP : BOT
            if (G::NW == 2) {
                st_xedge2(rw, v | tt.S[0][0], v | tt.S[0][1]);
                st_xedge2(rw + 2, v | tt.S[1][0], v | tt.S[1][1]);
            } else {
                st_xedge2(rw, v | tt.S[0][0], v | tt.S[1][0]);
            }
        }
        if (Y == 0) {
            st_xedge2(e + 4, v | L0, v | L1);
            st_xedge2(e + 6, v | R0, v | R1);
        }
    };
    auto refresh = [&](TileRegs<T>& tt, const Job& jb, uint32_t want) {
        const unsigned long long* rowp = rec(Y == 0 ? jb.nU : jb.nD, want) + (Y == 0 ? 8 : 0);     // BOT of the tile above : TOP of the tile below
        const unsigned long long* lf = rec(jb.nL, want) + 6;                                       // {R0, R1}
        const unsigned long long* rt = rec(jb.nR, want) + 4;                                       // {L0, L1}
        const bool need_row = Y == 0 || Y == G::LPT - 1;
        for (;;) {
            ulonglong2 r0 = make_ulonglong2(0, 0), r1 = r0;
            const ulonglong2 a = ld_xedge2(lf), b = ld_xedge2(rt);
            bool ok = (uint32_t)(a.x >> 32) == want && (uint32_t)(a.y >> 32) == want && (uint32_t)(b.x >> 32) == want && (uint32_t)(b.y >> 32) == want;
            if (need_row) {
                r0 = ld_xedge2(rowp);
                ok = ok && (uint32_t)(r0.x >> 32) == want && (uint32_t)(r0.y >> 32) == want;
                if (G::NW == 2) {
                    r1 = ld_xedge2(rowp + 2);
                    ok = ok && (uint32_t)(r1.x >> 32) == want && (uint32_t)(r1.y >> 32) == want;
                }
            }
            if (__all_sync(0xffffffffu, ok)) {
                tt.vrow[0][0] = (uint32_t)r0.x;
                if (G::NW == 2) { tt.vrow[0][1] = (uint32_t)r0.y; tt.vrow[1][0] = (uint32_t)r1.x; tt.vrow[1][1] = (uint32_t)r1.y; }
                else tt.vrow[1][0] = (uint32_t)r0.y;
                tt.hL0 = ((uint32_t)a.x >> Y) & 1u; tt.hL1 = ((uint32_t)a.y >> Y) & 1u;
                tt.hR0 = ((uint32_t)b.x >> Y) & 1u; tt.hR1 = ((uint32_t)b.y >> Y) & 1u;
                return;
            }
        }
    };
    auto slot = [&](int C, uint32_t m) { return ws + (size_t)((uint32_t)C * Mw + m) * (NSLOT * 32u); };
    auto sm_job = [&](int C, uint32_t m) {                             // the constants parked by the prologue
        const uint32_t* p = slot(C, m) + NWORDS * 32;
        const uint32_t xy = p[5 * 32];
        return Job{(int)p[6 * 32], (int)(xy & 0xffffu), (int)(xy >> 16), p[0], p[1 * 32], p[2 * 32], p[3 * 32], p[4 * 32]};
    };
    auto sm_put_job = [&](const Job& jb, int C, uint32_t m) {
        uint32_t* p = slot(C, m) + NWORDS * 32;
        p[0] = jb.self; p[1 * 32] = jb.nU; p[2 * 32] = jb.nD; p[3 * 32] = jb.nL; p[4 * 32] = jb.nR;
        p[5 * 32] = (uint32_t)jb.tx | ((uint32_t)jb.ty << 16); p[6 * 32] = (uint32_t)jb.r;
    };
    auto sm_load = [&](TileRegs<T>& tt, int C, uint32_t m) {
        const uint32_t* p = slot(C, m);
#pragma unroll
        for (int i = 0; i < NWORDS; ++i) tt.S[i / G::NW][i % G::NW] = p[i * 32];
    };
    auto sm_store = [&](const TileRegs<T>& tt, int C, uint32_t m) {
        uint32_t* p = slot(C, m);
#pragma unroll
        for (int i = 0; i < NWORDS; ++i) p[i * 32] = tt.S[i / G::NW][i % G::NW];
    };

    // records -> shared memory; every tile publishes its boundary as version 1 (what phase 0 waits for)
    for (int C = C0; C < C1; ++C)
        for (uint32_t m = 0; m < Mw; ++m) {
            const uint32_t job = wg + m * W;
            if (job >= R.jobs_total) break;                               // warp-uniform
            const Job jb = decode(job, C);
            TileRegs<T> tt;
            load_tile<T, BITS>(A, jb.r, jb.tx, jb.ty, Y, sub * G::LPT, tt);
            sm_store(tt, C, m);
            sm_put_job(jb, C, m);
            publish(tt, jb, 1u);
        }
    uint32_t ph = 0;                                                      // phases done: waits for version ph + 1, publishes ph + 2
    for (int pass = 0; pass < R.n; ++pass)
        for (int Cc = 0; Cc < (Tc ? 2 : 1); ++Cc)                         // (coarse tiles: both coarse colours in turn)
            for (int j = 0; j < A.k; ++j) {
                const uint64_t t64 = A.t_first + (uint64_t)pass * (uint64_t)A.k + (uint64_t)j;
                for (int c = 0; c < 2; ++c, ++ph)
                    for (int C = C0; C < C1; ++C)
#pragma unroll 1
                        for (uint32_t m = 0; m < Mw; ++m) {
                            const uint32_t job = wg + m * W;
                            if (job >= R.jobs_total) break;
                            const Job jb = sm_job(C, m);
                            TileRegs<T> tt;
                            sm_load(tt, C, m);
                            uint4 Jw[2][G::NW];
#pragma unroll
                            for (int cc = 0; cc < 2; ++cc)
#pragma unroll
                                for (int gx = 0; gx < G::NW; ++gx)
                                    Jw[cc][gx] = HASJ ? __ldg(A.jrec + ((size_t)jb.ty * B + jb.tx) * (2 * G::NW * G::LPT) + (cc * G::NW + gx) * G::LPT + Y)
                                                      : make_uint4(0u, 0u, 0u, 0u);
                            refresh(tt, jb, ph + 1u);
                            const uint64_t seed = A.seeds[jb.r];
                            const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
                            const uint32_t Yg = (uint32_t)(jb.ty * G::LPT + Y);
                            const uint32_t g0 = Yg * (B * G::NW) + (uint32_t)(jb.tx * G::NW);
                            const uint32_t p0 = 2u * Yg * (B * (uint32_t)(T / 2)) + 16u * (uint32_t)(jb.tx * G::NW);
                            half_sweep_masked<T, HASJ>(A, tt, Jw, c, Y, g0, p0, 2 * t64 + (uint64_t)c, k0, k1, Tc, Yg, (uint32_t)(jb.tx * G::NW), Cc);
                            publish(tt, jb, ph + 2u);
                            sm_store(tt, C, m);
                        }
            }
    for (int C = C0; C < C1; ++C)
        for (uint32_t m = 0; m < Mw; ++m) {
            const uint32_t job = wg + m * W;
            if (job >= R.jobs_total) break;
            const Job jb = sm_job(C, m);
            TileRegs<T> tt;
            sm_load(tt, C, m);
            store_tile<T, BITS>(A, jb.r, jb.tx, jb.ty, Y, sub, tt, lut);
        }
}

size_t grid_plain_xedge_bytes(const ising_ctx* h, int T) { return 2 * grid_planes_xedge_bytes(h, T); }

// n passes (of k sweeps each) of the plain checkerboard (Tc = 0) or of the double checkerboard of coarse tiles Tc in one
// cooperative launch; returns 1 (nothing launched) if the lattice does not fit the shared memory of the GPU or the launch
// is refused.  d_xedge: grid_plain_xedge_bytes.
int launch_grid_plain(ising_ctx* h, const Accept& acc, int T, bool bits, int n, int k, uint64_t t_first, int Tc, void* d_xedge) {
    GridArgs R;
    PlaneArgs& A = R.P;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = h->L; A.B = h->L / T; A.R = h->R; A.k = k; A.t_first = t_first; A.C = 0;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    A.stream = 0;
    A.njobs = 0;
    A.magic_rep = fastdiv_magic((uint32_t)A.B * (uint32_t)A.B / 2u);
    A.magic_hb = fastdiv_magic((uint32_t)A.B / 2u);
    fill_accept(A, acc);
    R.n = n;
    R.magic_k = 0;
    R.tiles_per_colour = (uint32_t)A.B * (uint32_t)A.B / 2u;
    R.jobs_total = (uint32_t)h->R * R.tiles_per_colour / (uint32_t)(64 / T);
    R.xedge = (unsigned long long*)d_xedge;
    R.acc = nullptr;
    // versions are 32 bits wide: two per phase
    if ((uint64_t)n * (uint64_t)(Tc ? 2 : 1) * (uint64_t)k * 2u + 2u >= 0xffffffffull) return 1;
    int dev = 0, sms = 0;
    ISING_CUDA_OK(cudaGetDevice(&dev));
    ISING_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const void* fn = T == 64 ? (bits ? (A.jrec ? (const void*)k_grid_plain<64, true, true> : (const void*)k_grid_plain<64, true, false>)
                                     : (A.jrec ? (const void*)k_grid_plain<64, false, true> : (const void*)k_grid_plain<64, false, false>))
                             : (bits ? (A.jrec ? (const void*)k_grid_plain<32, true, true> : (const void*)k_grid_plain<32, true, false>)
                                     : (A.jrec ? (const void*)k_grid_plain<32, false, true> : (const void*)k_grid_plain<32, false, false>));
    constexpr size_t kSmemMax = 227 * 1024;
    ISING_CUDA_OK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax));
    static const uint32_t warp_cap = getenv("ISING_GRID_WARPS") ? (uint32_t)atoi(getenv("ISING_GRID_WARPS")) : 0u;   // testing aid, as in launch_grid_one
    const uint32_t nwords = 2u * (uint32_t)(T / 32) + 7u;      // spin words + the job's parked constants
    // one job per warp and phase where the GPU holds a warp for every register-tile job of either colour
    int split = (!warp_cap && 2u * R.jobs_total <= (uint32_t)sms * 28u) ? 1 : 0;
    for (uint32_t M = 1; M <= kGridMaxJobsPerWarp; ++M) {
        if (split && M > 1) split = 0, M = 1;
        const uint32_t warps_needed = (split ? 2u : 1u) * ((R.jobs_total + M - 1) / M);
        if (warp_cap && warps_needed > warp_cap && M < kGridMaxJobsPerWarp) continue;
        const uint32_t w_sm = (warps_needed + (uint32_t)sms - 1) / (uint32_t)sms;
        if (w_sm > 28u) continue;                                 // more jobs per warp
        const int wpb = (int)((w_sm + 1u) & ~1u);                 // even: with split, the two colours alternate over the warp index
        const size_t smem = (size_t)wpb * 2u * M * nwords * 32u * sizeof(uint32_t);
        if (smem > kSmemMax) break;                               // the lattice does not fit on chip
        int occ = 0;
        ISING_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, wpb * 32, smem));
        const uint32_t grid = (warps_needed + wpb - 1) / wpb;
        if (grid > (uint32_t)sms * (uint32_t)occ) continue;
        R.jobs_per_warp = M;
        cudaStream_t st = hooks().stream;
        ISING_CUDA_OK(cudaMemsetAsync(d_xedge, 0, grid_plain_xedge_bytes(h, T), st));      // version 0 = nothing published
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(wpb * 32); cfg.dynamicSmemBytes = smem; cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeCooperative;
        attr[0].val.cooperative = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        void* args[] = {&R, &Tc, &split};
        if (cudaLaunchKernelExC(&cfg, fn, args) != cudaSuccess) { cudaGetLastError(); return 1; }      // refused (shared or partitioned GPU)
        count_launch();
        return 0;
    }
    return 1;
}

// ---- k_flow_planes (flow_planes_device.cuh): all n passes of an HBM-resident lattice in one persistent launch ----
namespace {
template <int T, bool BITS, int NS>
int launch_flow_one(FlowArgs& F, bool use_jit, bool* used_jit, int stage_mode) {
    const PlaneArgs& A = F.P;
    int dev = 0, sms = 0;
    ISING_CUDA_OK(cudaGetDevice(&dev));
    ISING_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int threads = kPlaneThreads;       // measured on config 3: 128 x 10 CTAs per SM 2485 / 2100 flips/ns (tile 64 / 32); 256 x 5 2463 / 2092; 320 x 4 2450 / 2088; 640 x 2 2416 / 2057; 1024 x 1 2340 / 1788
    const uint32_t warps = threads / 32;
    // TMA staging of the next job's bodies: only where a tile's previous write-back is certainly older than anything this
    // grid still has in flight (a phase of more than 2 x the resident warps), and never with coupling records (kept simple)
    const uint32_t resident_max = (uint32_t)sms * 16u * warps;
    bool staged = stage_mode == 1 || (stage_mode == 0 && false);
    if (F.jobs_per_phase <= 2u * resident_max || A.jrec) staged = false;
    const size_t smem = staged ? (size_t)warps * (64 / T) * NS * (BITS ? T * T / 8 : T * T) : 0;
    cudaKernel_t spec = (use_jit && !A.force) ? flow_jit_kernel(T, BITS, A.jrec != nullptr, A.hp, A.B, A.R, NS, staged) : nullptr;
    const void* fn = spec ? (const void*)spec
                   : staged ? (const void*)k_flow_planes_staged<T, BITS, false, kNoSpec, NS>
                   : (A.jrec ? (const void*)k_flow_planes<T, BITS, true, kNoSpec, NS> : (const void*)k_flow_planes<T, BITS, false, kNoSpec, NS>);
    int occ = 0;
    ISING_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, threads, smem));
    if (occ < 1) { set_error("k_flow_planes does not fit an SM"); return ISING_ECUDA; }
    uint32_t grid = (uint32_t)sms * (uint32_t)occ;
    grid = std::min<uint32_t>(grid, (F.jobs_per_phase + warps - 1) / warps);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = smem; cfg.stream = hooks().stream;
    void* args[] = {&F};
    ISING_CUDA_OK(cudaLaunchKernelExC(&cfg, fn, args));
    count_launch();
    *used_jit = spec != nullptr;
    return 0;
}
}  // namespace

size_t flow_planes_scratch_bytes(const ising_ctx* h, int T) { return 256 + (size_t)h->R * (size_t)(h->L / T) * (size_t)(h->L / T) * sizeof(uint32_t); }

bool flow_planes_supported(const ising_ctx* h, int T, int n) {
    if (!tile_planes_supported(h, T)) return false;
    // tickets are 32 bits wide: 2 n phases x jobs per phase (at most R * tiles / 2) must stay below 2^32
    const uint64_t jobs = (uint64_t)h->R * (uint64_t)(h->L / T) * (uint64_t)(h->L / T) / 2u;
    return n >= 2 && 2ull * (uint64_t)n * jobs < 0xffffffffull;
}

// n passes in one persistent launch.  d_scratch: flow_planes_scratch_bytes (ticket counter + one progress word per tile).
int launch_flow_planes(ising_ctx* h, const Accept& acc, int T, bool bits, int n, int k, uint64_t t_first, void* d_scratch, bool use_jit) {
    static const int stage_mode = getenv("ISING_FLOW_STAGE") ? atoi(getenv("ISING_FLOW_STAGE")) : 0;     // 1: TMA staging of the next job (profiles/r02: measured, not faster), default off
    FlowArgs F;
    PlaneArgs& A = F.P;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = h->L; A.B = h->L / T; A.R = h->R; A.k = k; A.t_first = t_first; A.C = 0;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    A.stream = tile_planes_bytes(h, T, bits) > kL2StreamBytes ? 1u : 0u;
    A.magic_rep = fastdiv_magic((uint32_t)A.B * (uint32_t)A.B / 2u);
    A.magic_hb = fastdiv_magic((uint32_t)A.B / 2u);
    fill_accept(A, acc);
    const int ns = plane_slots(T, A.B);
    const uint32_t tiles_per_colour = (uint32_t)((size_t)h->R * A.B * A.B / 2);
    const uint32_t per_job = (uint32_t)(64 / T) * (uint32_t)ns;
    A.njobs = tiles_per_colour / per_job;
    F.jobs_per_phase = A.njobs;
    F.n_phases = 2u * (uint32_t)n;
    F.phase_shift = (2u * (uint32_t)(A.B / 2) + per_job - 1) / per_job;      // two tile rows of jobs
    if (F.phase_shift >= F.jobs_per_phase) F.phase_shift = 0;
    F.magic_jp = fastdiv_magic(F.jobs_per_phase);
    F.total = F.n_phases * F.jobs_per_phase;
    F.ticket = (unsigned int*)d_scratch;
    F.prog = (uint32_t*)((char*)d_scratch + 256);
    ISING_CUDA_OK(cudaMemsetAsync(d_scratch, 0, flow_planes_scratch_bytes(h, T), hooks().stream));
    bool used = false;
    int rc;
    if (ns == 2) rc = T == 64 ? (bits ? launch_flow_one<64, true, 2>(F, use_jit, &used, stage_mode) : launch_flow_one<64, false, 2>(F, use_jit, &used, stage_mode))
                              : (bits ? launch_flow_one<32, true, 2>(F, use_jit, &used, stage_mode) : launch_flow_one<32, false, 2>(F, use_jit, &used, stage_mode));
    else rc = T == 64 ? (bits ? launch_flow_one<64, true, 1>(F, use_jit, &used, stage_mode) : launch_flow_one<64, false, 1>(F, use_jit, &used, stage_mode))
                      : (bits ? launch_flow_one<32, true, 1>(F, use_jit, &used, stage_mode) : launch_flow_one<32, false, 1>(F, use_jit, &used, stage_mode));
    if (rc) return rc;
    h->last_jit = used ? 1 : 0;
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

}  // namespace ising
