// heis.cu — classical Heisenberg (O(3)) double-checkerboard Metropolis, include/heisenberg.h (SURVEY.md
// §8(f) item 4; readings H1-H8 of DESIGN.md §3.7).  Single precision, every operation stated: the device code
// below uses the round-to-nearest intrinsics (__fmaf_rn, __fmul_rn, __fadd_rn, __fsub_rn, __fsqrt_rn), which the
// compiler neither contracts nor re-associates, so the trajectory is a pure function of (seed, schedule).
//
// Storage: three float planes s[c][i] (c = x, y, z) in index order.  Two kernel families:
//   k_heis_tile<DIM, T>   one CTA per tile of the launch's coarse colour: tile + halo faces staged in shared memory
//                         (128-bit loads of the rows), k inner sweeps of both fine colours on chip, interior written
//                         back with 128-bit stores (steps a3, a5-a7 of the Ising path, same schedule);
//   k_heis_generic        one launch per half-sweep on the live array (any valid tile, T = L included).
#include <algorithm>
#include <cmath>
#include <new>

#include "kernels.h"
#include "philox.cuh"
#include "../../include/heisenberg.h"

struct heis_ctx {
    int dim = 2;
    int L = 0;
    uint64_t N = 0;
    uint64_t seed = 0;
    uint64_t t = 0;
    float* d_s = nullptr;       // 3*N floats
    double* d_obs = nullptr;    // E, Mx, My, Mz
    float* d_xface = nullptr;   // x-face copies of the tile kernel, valid for tile size xface_T (0: stale)
    size_t xface_bytes = 0;
    int xface_T = 0;
    const char* last_path = "none";
    int force_generic = 0;
};

namespace ising {

namespace {

constexpr uint32_t kTagHeisSweep = 5u;   // H4
constexpr uint32_t kTagHeisInit = 6u;    // H3

struct f3 { float x, y, z; };

// H2: 40 bits of two random words -> a uniform direction (the low 24 bits of wb are the acceptance number).
__device__ __forceinline__ f3 heis_direction(uint32_t wa, uint32_t wb) {
    constexpr float PI_4 = (float)0.78539816339744830962;
    constexpr float S3 = (float)(-1.0 / 6.0), S5 = (float)(1.0 / 120.0), S7 = (float)(-1.0 / 5040.0), S9 = (float)(1.0 / 362880.0);
    constexpr float C2 = (float)(-1.0 / 2.0), C4 = (float)(1.0 / 24.0), C6 = (float)(-1.0 / 720.0), C8 = (float)(1.0 / 40320.0),
                    C10 = (float)(-1.0 / 3628800.0);
    const uint32_t phi20 = __funnelshift_l(wb, wa, 8) & 0xfffffu;       // ((wa & 0xfff) << 8) | (wb >> 24)
    const float z = __fmaf_rn(__uint2float_rn(wa >> 12), 0x1p-19f, -1.0f);
    const float rho = __fsqrt_rn(__fmaf_rn(-z, z, 1.0f));
    const uint32_t q = phi20 >> 17;
    float t = __fmul_rn(__uint2float_rn(phi20 & 0x1ffffu), 0x1p-17f);
    if (q & 1u) t = __fsub_rn(t, 1.0f);
    const float x = __fmul_rn(t, PI_4);
    const float x2 = __fmul_rn(x, x);
    const float x3 = __fmul_rn(x2, x);
    float ps = __fmaf_rn(x2, S9, S7);
    ps = __fmaf_rn(x2, ps, S5);
    ps = __fmaf_rn(x2, ps, S3);
    const float sn = __fmaf_rn(x3, ps, x);
    float pc = __fmaf_rn(x2, C10, C8);
    pc = __fmaf_rn(x2, pc, C6);
    pc = __fmaf_rn(x2, pc, C4);
    pc = __fmaf_rn(x2, pc, C2);
    const float cs = __fmaf_rn(x2, pc, 1.0f);
    const uint32_t Q = ((q + 1u) >> 1) & 3u;
    float c = (Q & 1u) ? sn : cs;          // Q: 0 (cs, sn)  1 (-sn, cs)  2 (-cs, -sn)  3 (sn, -cs)
    float s = (Q & 1u) ? cs : sn;
    if (Q == 1u || Q == 2u) c = -c;
    if (Q >= 2u) s = -s;
    return f3{__fmul_rn(rho, c), __fmul_rn(rho, s), z};
}

// H6: acceptance probability for a < 0.
__device__ __forceinline__ float heis_accept_probability(float a) {
    constexpr float LOG2E = (float)1.4426950408889634074, LN2 = (float)0.69314718055994530942;
    constexpr float E2 = (float)(1.0 / 2.0), E3 = (float)(1.0 / 6.0), E4 = (float)(1.0 / 24.0), E5 = (float)(1.0 / 120.0),
                    E6 = (float)(1.0 / 720.0), E7 = (float)(1.0 / 5040.0);
    const float tt = __fmul_rn(a, LOG2E);
    const float n = rintf(tt);
    const float f = __fsub_rn(tt, n);
    const float g = __fmul_rn(f, LN2);
    float p = __fmaf_rn(g, E7, E6);
    p = __fmaf_rn(g, p, E5);
    p = __fmaf_rn(g, p, E4);
    p = __fmaf_rn(g, p, E3);
    p = __fmaf_rn(g, p, E2);
    p = __fmaf_rn(g, p, 1.0f);
    p = __fmaf_rn(g, p, 1.0f);
    const float P = __fmul_rn(p, __uint_as_float((uint32_t)(__float2int_rn(n) + 127) << 23));
    return tt < -64.0f ? 0.0f : P;        // (for tt outside [-64, 0] P is meaningless and not used)
}

// H5 given the two random words, the old spin and the local field; returns true and the new spin if the move is accepted.
__device__ __forceinline__ bool heis_update(uint32_t wa, uint32_t wb, float betaf, const f3& s, const f3& h, f3& sp) {
    sp = heis_direction(wa, wb);
    const float dx = __fsub_rn(sp.x, s.x), dy = __fsub_rn(sp.y, s.y), dz = __fsub_rn(sp.z, s.z);
    float e = __fmul_rn(dx, h.x);
    e = __fmaf_rn(dy, h.y, e);
    e = __fmaf_rn(dz, h.z, e);
    // both sides of "e >= 0 or u < P" are evaluated (a warp nearly always holds both cases): for e >= 0 the value
    // of P is not used
    const float u = __fmul_rn(__uint2float_rn(wb & 0xffffffu), 0x1p-24f);
    const float P = heis_accept_probability(__fmul_rn(betaf, e));
    return (e >= 0.0f) | (u < P);
}

// ---- H3 ----------------------------------------------------------------------------------------------
__global__ void k_heis_hot_start(float* __restrict__ s, uint64_t N, uint32_t k0, uint32_t k1) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const u32x4 w = philox4x32_10((uint32_t)(i >> 1), kTagHeisInit, 0u, 0u, k0, k1);
    const f3 v = (i & 1) ? heis_direction(w.z, w.w) : heis_direction(w.x, w.y);
    s[i] = v.x; s[N + i] = v.y; s[2 * N + i] = v.z;
}

// ---- generic half-sweep: one thread per 2x2 block of the xy plane (= one Philox call, H4), live neighbours --------
struct GenArgs {
    float* s;
    uint64_t N, H;
    int L, dim, T, C, c;     // T == L: one tile (phase C = 1 is never launched)
    uint32_t k0, k1;
    float betaf;
};

__global__ void k_heis_generic(GenArgs A) {
    const uint64_t g = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= A.N / 4) return;
    const int L = A.L, hl = L / 2;
    const int bx = (int)(g % hl), by = (int)((g / hl) % hl), z = (int)(g / ((uint64_t)hl * hl));
    // T is even: the block lies in one tile
    if (A.T != L && (((2 * bx) / A.T + (2 * by) / A.T + z / A.T) & 1) != A.C) return;
    const u32x4 w = philox4x32_10((uint32_t)g, kTagHeisSweep, (uint32_t)A.H, (uint32_t)(A.H >> 32), A.k0, A.k1);
    const uint64_t N = A.N;
    const float* sx = A.s;
    const float* sy = A.s + N;
    const float* sz = A.s + 2 * N;
    for (int hw = 0; hw < 2; ++hw) {         // the two rows of the block; their active sites are not neighbours
        const int y = 2 * by + hw;
        const int x = 2 * bx + ((y + z + A.c) & 1);
        const uint64_t i = ((uint64_t)z * L + y) * L + x;
        const uint64_t xm = i - x + (x == 0 ? L - 1 : x - 1), xp = i - x + (x == L - 1 ? 0 : x + 1);
        f3 h{__fadd_rn(sx[xm], sx[xp]), __fadd_rn(sy[xm], sy[xp]), __fadd_rn(sz[xm], sz[xp])};
        const uint64_t row = (uint64_t)L;
        const uint64_t ym = y == 0 ? i + row * (L - 1) : i - row, yp = y == L - 1 ? i - row * (L - 1) : i + row;
        h.x = __fadd_rn(h.x, sx[ym]); h.y = __fadd_rn(h.y, sy[ym]); h.z = __fadd_rn(h.z, sz[ym]);
        h.x = __fadd_rn(h.x, sx[yp]); h.y = __fadd_rn(h.y, sy[yp]); h.z = __fadd_rn(h.z, sz[yp]);
        if (A.dim > 2) {
            const uint64_t pl = (uint64_t)L * L;
            const uint64_t zm = z == 0 ? i + pl * (L - 1) : i - pl, zp = z == L - 1 ? i - pl * (L - 1) : i + pl;
            h.x = __fadd_rn(h.x, sx[zm]); h.y = __fadd_rn(h.y, sy[zm]); h.z = __fadd_rn(h.z, sz[zm]);
            h.x = __fadd_rn(h.x, sx[zp]); h.y = __fadd_rn(h.y, sy[zp]); h.z = __fadd_rn(h.z, sz[zp]);
        }
        const f3 s{sx[i], sy[i], sz[i]};
        f3 sp;
        if (heis_update(hw ? w.z : w.x, hw ? w.w : w.y, A.betaf, s, h, sp)) {
            A.s[i] = sp.x; A.s[N + i] = sp.y; A.s[2 * N + i] = sp.z;
        }
    }
}

// ---- tile kernel -------------------------------------------------------------------------------------------
// Shared-memory tile of one component: [ZP][YP][XP] floats, interior site (lx, ly, lz) at (lz+1, ly+1, lx+4) (2D:
// ZP = 1, no z offset): column 3 and column T+4 are the x halos, and the interior rows start 16-byte aligned.
// XP is even, so that the active sites of a row and those of the next row, which have the other parity, fall
// into different banks; the pitches and the order in which a thread takes the two rows of its block (swap_rows) were
// chosen by enumerating the banks a warp touches: no conflicts in the update loop for any supported (dim, T).
template <int DIM, int T>
struct HG {
    static constexpr int XP = T <= 16 ? T + 4 : T + 8;          // T + 4: the right halo of a row sits in the unused column 0 of the next
    static constexpr int YP = T + 2;
    static constexpr int ZP = DIM == 3 ? T + 2 : 1;
    static constexpr int ZS = XP * YP + (DIM == 3 && T == 4 ? 4 : 0);   // layer pitch
    static constexpr int COMP = ZS * ZP + 4;                    // floats per component
    static constexpr int SITES = DIM == 3 ? T * T * T : T * T;
    static constexpr int THREADS = SITES / 4 < 32 ? 32 : (SITES / 4 > 512 ? 512 : SITES / 4);
    // update loop: an item = a 2x2 block of the xy plane (one Philox call, two active sites per half-sweep, H4);
    // thread = (pair column px, row pair rp[, layer lz]) takes IPT items, THREADS / (T/2) row pairs (2D) or
    // THREADS / (T*T/4) layers (3D) apart; both are even, so the parities a thread sees are fixed.
    static constexpr int HALF = T / 2;
    static constexpr int ITEMS = SITES / 4;
    static constexpr int IPT = ITEMS / THREADS > 0 ? ITEMS / THREADS : 1;
    static constexpr int RSTEP = THREADS / HALF;                       // row pairs per round of THREADS items
    static constexpr int OSTEP = DIM == 3 ? (RSTEP / HALF) * ZS : 2 * RSTEP * XP;
    // 1: the thread takes row 2rp+1 of its block first
    __device__ static constexpr int swap_rows(int px, int rp) {
        return DIM == 2 && T == 64 ? (px >> 4) & 1 : (DIM == 3 && T == 8 ? 0 : rp & 1);
    }
    static_assert(THREADS % HALF == 0 && (ITEMS < THREADS || IPT * THREADS == ITEMS), "thread mapping");
    static_assert(IPT == 1 || (DIM == 3 ? (RSTEP % HALF == 0 && (RSTEP / HALF) % 2 == 0) : RSTEP % 2 == 0), "fixed parity per thread");
    // 2D T=64: 42 registers for a third 512-thread CTA per SM (+15 % at k=1, -3 % at k=16); 0 = the compiler's own choice
    static constexpr int MIN_CTAS = DIM == 2 && T == 64 ? 3 : 0;
    static constexpr int FACE = SITES / T;                       // sites of one face
    // shared memory: three components of the tile + halo, then the staged x faces XF[c][side][FACE]
    static constexpr size_t SMEM = (size_t)(3 * COMP + 6 * FACE) * sizeof(float);
    __device__ static constexpr int at(int lx, int ly, int lz) {
        return (DIM == 3 ? lz + 1 : 0) * ZS + (ly + 1) * XP + lx + 4;
    }
};

struct TileArgs {
    float* s;
    float* xface;        // x-face copies, see below
    uint64_t N, t_first;
    int L, B, C, k;
    uint32_t ntiles;     // all tiles, both colours
    uint32_t k0, k1;
    float betaf;
};

// x-face copies.  The x halos of a tile are single floats T apart in a row: read from the spin planes each would
// cost a whole 64-byte DRAM access.  So every tile also keeps copies of its own two x faces (the columns lx = 0 and
// lx = T-1, FACE = T^(dim-1) floats each, ordered (lz, ly)) in a side array
//     xface[((c * ntiles + tile) * 2 + side) * FACE + lz * T + ly],   tile = (tz * B + ty) * B + tx,
// written with the tile's write-back and read by the two x neighbours as contiguous 16-byte copies.  The spin planes
// stay complete and current; the host rebuilds the copies (k_heis_build_xface) when something else wrote the spins.
__device__ __forceinline__ void cp_async16_addr(uint32_t smem_addr, const float* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <int DIM, int T>
__global__ void k_heis_build_xface(const float* __restrict__ s, float* __restrict__ xface, uint64_t N, int L, int B, uint32_t ntiles) {
    constexpr int FACE = HG<DIM, T>::FACE;
    const uint64_t e = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;     // entry of xface
    if (e >= (uint64_t)3 * ntiles * 2 * FACE) return;
    const int f = (int)(e % FACE), side = (int)((e / FACE) & 1);
    const uint32_t tile = (uint32_t)((e / (2 * FACE)) % ntiles);
    const int c = (int)(e / ((uint64_t)2 * FACE * ntiles));
    const int tx = tile % B, ty = (tile / B) % B, tz = DIM == 3 ? tile / (B * B) : 0;
    const int ly = f % T, lz = f / T;
    const uint64_t i = (uint64_t)(tz * T + lz) * L * L * (DIM == 3) + (uint64_t)(ty * T + ly) * L + (uint64_t)(tx * T + (side ? T - 1 : 0));
    xface[e] = s[(uint64_t)c * N + i];
}

// One CTA per tile of the launch's coarse colour (job -> (tx/2, ty, tz) row-major).
template <int DIM, int T>
__global__ void __launch_bounds__(HG<DIM, T>::THREADS, HG<DIM, T>::MIN_CTAS) k_heis_tile(TileArgs A) {
    using G = HG<DIM, T>;
    extern __shared__ __align__(16) float sm[];
    const int tid = threadIdx.x;
    const int L = A.L, B = A.B;
    const int hb = B / 2;
    const int txh = blockIdx.x % hb;
    const int ty = (blockIdx.x / hb) % B;
    const int tz = DIM == 3 ? blockIdx.x / (hb * B) : 0;
    const int tx = 2 * txh + ((ty + tz + A.C) & 1);
    const int x0 = tx * T, y0 = ty * T, z0 = tz * T;
    const uint64_t N = A.N;
    const uint64_t row = (uint64_t)L, plane = (uint64_t)L * L;
    constexpr int Q = T / 4;
    constexpr int FACE = G::FACE;
    const uint32_t tile_row = (uint32_t)(tz * B + ty) * (uint32_t)B;
    const uint32_t t_self = tile_row + tx, t_left = tile_row + (tx == 0 ? B - 1 : tx - 1), t_right = tile_row + (tx == B - 1 ? 0 : tx + 1);
    float* const XF = sm + 3 * G::COMP;

    // a3: interior rows, the y / z faces and the x-face copies as 16-byte asynchronous copies.  Every offset is worked
    // out once per thread, the loop over the three components is innermost.  Float offsets inside one component are
    // below N <= 2^32.
    const uint32_t sm_addr = (uint32_t)__cvta_generic_to_shared(sm);
    const uint32_t origin = (uint32_t)((DIM == 3 ? (uint64_t)z0 * plane : 0) + (uint64_t)y0 * row + (uint64_t)x0);
    constexpr int INT_ROUNDS = (G::SITES / 4 + G::THREADS - 1) / G::THREADS;
    uint32_t int_g[INT_ROUNDS], int_s[INT_ROUNDS];                    // interior 16-byte pieces of this thread (write-back too)
#pragma unroll
    for (int n = 0; n < INT_ROUNDS; ++n) {
        const int idx = tid + n * G::THREADS;
        const int q = idx % Q, yy = (idx / Q) % T, zz = idx / (Q * T);
        int_g[n] = origin + (uint32_t)(DIM == 3 ? zz : 0) * (uint32_t)plane + (uint32_t)yy * (uint32_t)L + 4u * q;
        int_s[n] = (uint32_t)G::at(4 * q, yy, zz);
    }
    const bool int_live = G::SITES / 4 >= G::THREADS || tid < G::SITES / 4;
    if (int_live) {
#pragma unroll
        for (int n = 0; n < INT_ROUNDS; ++n)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                cp_async16_addr(sm_addr + 4u * (c * G::COMP + int_s[n]), A.s + (uint64_t)c * N + int_g[n]);
    }
    // faces: FQ = FACE/4 pieces per face; kinds 0,1 = y faces, 2,3 = x-face copies, 4,5 = z faces (3D): one per thread
    constexpr int FQ = FACE / 4;
    constexpr int NFACE = (DIM == 3 ? 6 : 4) * FQ;
    static_assert(NFACE <= G::THREADS, "one face piece per thread");
    if (tid < NFACE) {
        const int kind = tid / FQ, r = tid % FQ, side = kind & 1;
        const float* src;
        uint64_t cstride;                                             // floats between the components at the source
        uint32_t dst;
        if ((kind >> 1) == 1) {
            // left halo = right face (side 1) of the left neighbour, right halo = left face (side 0) of the right one
            src = A.xface + ((uint64_t)(side ? t_right : t_left) * 2 + (side ? 0 : 1)) * FACE + 4 * r;
            cstride = (uint64_t)A.ntiles * 2 * FACE;
            dst = (uint32_t)(3 * G::COMP + side * FACE + 4 * r);     // XF[c][side][.]: component stride 2*FACE, see below
        } else {
            const int q = r % Q, w = r / Q;                          // w = lz for a y face, ly for a z face
            uint32_t off;
            if (kind < 2) {
                const uint32_t y = side ? (y0 + T == L ? 0u : (uint32_t)(y0 + T)) : (y0 == 0 ? (uint32_t)(L - 1) : (uint32_t)(y0 - 1));
                off = (uint32_t)(DIM == 3 ? z0 + w : 0) * (uint32_t)plane + y * (uint32_t)L + (uint32_t)x0 + 4u * q;
                dst = (uint32_t)G::at(4 * q, side ? T : -1, w);
            } else {
                const uint32_t z = side ? (z0 + T == L ? 0u : (uint32_t)(z0 + T)) : (z0 == 0 ? (uint32_t)(L - 1) : (uint32_t)(z0 - 1));
                off = z * (uint32_t)plane + (uint32_t)(y0 + w) * (uint32_t)L + (uint32_t)x0 + 4u * q;
                dst = (uint32_t)G::at(4 * q, w, side ? T : -1);
            }
            src = A.s + off;
            cstride = N;
        }
        const uint32_t dstride = (kind >> 1) == 1 ? 2u * FACE : (uint32_t)G::COMP;
#pragma unroll
        for (int c = 0; c < 3; ++c) cp_async16_addr(sm_addr + 4u * (dst + c * dstride), src + c * cstride);
    }
    cp_async_commit();
    cp_async_wait_all();
    __syncthreads();
    static_assert(2 * FACE <= G::THREADS, "one x-halo site per thread");
    uint32_t halo_s = 0, edge_s = 0;                                  // this thread's x-halo site and own edge site
    if (tid < 2 * FACE) {                                             // staged x faces -> halo columns
        const int f = tid % FACE, side = tid / FACE;
        halo_s = (uint32_t)G::at(side ? T : -1, f % T, f / T);
        edge_s = (uint32_t)G::at(side ? T - 1 : 0, f % T, f / T);
#pragma unroll
        for (int c = 0; c < 3; ++c) sm[c * G::COMP + halo_s] = XF[c * 2 * FACE + tid];
    }
    __syncthreads();

    // a5/a6: k inner sweeps, fine colour 0 then 1; the halo stays as loaded
    float* const SX = sm;
    float* const SY = sm + G::COMP;
    float* const SZ = sm + 2 * G::COMP;
    // thread -> block (px, rp, lz); some threads take their two rows in the order (2rp+1, 2rp), so that the lanes of a
    // warp touch rows of both parities at the same time (different banks)
    const int px = tid % G::HALF, rp = (tid / G::HALF) % G::HALF, lz = tid / (G::HALF * G::HALF);
    const int sw = G::swap_rows(px, rp);
    const int rowA = 2 * rp + sw, rowB = 2 * rp + 1 - sw;
    const int parA = (rowA + lz) & 1;                                  // x0, y0, z0 are even
    const int oA_row = G::at(2 * px, rowA, lz), oB_row = G::at(2 * px, rowB, lz);
    const uint32_t hl = (uint32_t)(L >> 1);
    const uint32_t g_base = ((uint32_t)(z0 + lz) * hl * (DIM == 3) + (uint32_t)(y0 >> 1) + (uint32_t)rp) * hl + (uint32_t)(x0 >> 1) + (uint32_t)px;
    const uint32_t g_step = DIM == 3 ? (uint32_t)(G::RSTEP / G::HALF) * hl * hl : (uint32_t)G::RSTEP * hl;
    const bool live = G::ITEMS >= G::THREADS || tid < G::ITEMS;
    for (int j = 0; j < A.k; ++j) {
        for (int c = 0; c < 2; ++c) {
            const uint64_t H = 2 * (A.t_first + (uint64_t)j) + (uint64_t)c;
            const int aA = (parA + c) & 1;
            if (live) {
#pragma unroll
                for (int n = 0; n < G::IPT; ++n) {
                    const u32x4 w = philox4x32_10(g_base + (uint32_t)n * g_step, kTagHeisSweep, (uint32_t)H, (uint32_t)(H >> 32), A.k0, A.k1);
#pragma unroll
                    for (int second = 0; second < 2; ++second) {
                        const int o = (second ? oB_row + 1 - aA : oA_row + aA) + n * G::OSTEP;
                        const bool odd_row = (second != 0) != (sw != 0);            // row 2rp+1 takes words 2, 3
                        f3 h{__fadd_rn(SX[o - 1], SX[o + 1]), __fadd_rn(SY[o - 1], SY[o + 1]), __fadd_rn(SZ[o - 1], SZ[o + 1])};
                        h.x = __fadd_rn(h.x, SX[o - G::XP]); h.y = __fadd_rn(h.y, SY[o - G::XP]); h.z = __fadd_rn(h.z, SZ[o - G::XP]);
                        h.x = __fadd_rn(h.x, SX[o + G::XP]); h.y = __fadd_rn(h.y, SY[o + G::XP]); h.z = __fadd_rn(h.z, SZ[o + G::XP]);
                        if (DIM == 3) {
                            constexpr int ZS = G::ZS;
                            h.x = __fadd_rn(h.x, SX[o - ZS]); h.y = __fadd_rn(h.y, SY[o - ZS]); h.z = __fadd_rn(h.z, SZ[o - ZS]);
                            h.x = __fadd_rn(h.x, SX[o + ZS]); h.y = __fadd_rn(h.y, SY[o + ZS]); h.z = __fadd_rn(h.z, SZ[o + ZS]);
                        }
                        const f3 s{SX[o], SY[o], SZ[o]};
                        f3 sp;
                        if (heis_update(odd_row ? w.z : w.x, odd_row ? w.w : w.y, A.betaf, s, h, sp)) {
                            SX[o] = sp.x; SY[o] = sp.y; SZ[o] = sp.z;
                        }
                    }
                }
            }
            __syncthreads();
        }
    }

    // a7: interior back to HBM, and the tile's own x faces into the side array
    if (int_live) {
#pragma unroll
        for (int n = 0; n < INT_ROUNDS; ++n)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                *reinterpret_cast<float4*>(A.s + (uint64_t)c * N + int_g[n]) = *reinterpret_cast<const float4*>(sm + c * G::COMP + int_s[n]);
    }
    if (tid < 2 * FACE) {
        float* dst = A.xface + (uint64_t)t_self * 2 * FACE + tid;
#pragma unroll
        for (int c = 0; c < 3; ++c) dst[(uint64_t)c * A.ntiles * 2 * FACE] = sm[c * G::COMP + edge_s];
    }
}

// ---- H8 ----------------------------------------------------------------------------------------------
__global__ void k_heis_observables(const float* __restrict__ s, uint64_t N, int L, int dim, double* __restrict__ out) {
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (uint64_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % L);
        const int y = dim > 1 ? (int)((i / L) % L) : 0;
        const int z = dim > 2 ? (int)(i / ((uint64_t)L * L)) : 0;
        const uint64_t xp = x == L - 1 ? i - (L - 1) : i + 1;
        const uint64_t yp = y == L - 1 ? i - (uint64_t)L * (L - 1) : i + L;
        const uint64_t zp = z == L - 1 ? i - (uint64_t)L * L * (L - 1) : i + (uint64_t)L * L;
        for (int c = 0; c < 3; ++c) {
            const float* p = s + (uint64_t)c * N;
            const double v = (double)p[i];
            double nb = (double)p[xp];
            if (dim > 1) nb += (double)p[yp];
            if (dim > 2) nb += (double)p[zp];
            acc[0] -= v * nb;
            acc[1 + c] += v;
        }
    }
    __shared__ double red[4][8];
    for (int q = 0; q < 4; ++q) {
        double v = acc[q];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) red[q][threadIdx.x >> 5] = v;
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double v = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += red[threadIdx.x][w];
        atomicAdd(out + threadIdx.x, v);
    }
}

bool is_device_ptr(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

bool tile_valid(const heis_ctx* h, int T) {
    if (T < 2 || (T & 1) || h->L % T) return false;
    const int B = h->L / T;
    return B == 1 || (B % 2 == 0);
}

template <int DIM, int T>
int launch_tile(heis_ctx* h, TileArgs A) {
    using G = HG<DIM, T>;
    if (int rc = set_max_dynamic_smem<k_heis_tile<DIM, T>>((int)G::SMEM)) return rc;
    A.ntiles = (uint32_t)A.B * A.B * (DIM == 3 ? A.B : 1);
    const size_t entries = (size_t)3 * A.ntiles * 2 * G::FACE;
    if (h->xface_T != T) {                       // (re)build the x-face copies from the spin planes
        if (h->xface_bytes < entries * sizeof(float)) {
            dev_free(h->d_xface);
            h->xface_bytes = 0;
            h->d_xface = (float*)dev_alloc(entries * sizeof(float));
            if (!h->d_xface) return ISING_ENOMEM;
            h->xface_bytes = entries * sizeof(float);
        }
        k_heis_build_xface<DIM, T><<<(unsigned)((entries + 255) / 256), 256, 0, hooks().stream>>>(h->d_s, h->d_xface, h->N, h->L, A.B, A.ntiles);
        count_launch();
        h->xface_T = T;
    }
    A.xface = h->d_xface;
    for (int C = 0; C < 2; ++C) {
        A.C = C;
        k_heis_tile<DIM, T><<<A.ntiles / 2, G::THREADS, G::SMEM, hooks().stream>>>(A);
        count_launch();
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// 0: launched; 1: no tile kernel for this (dim, T)
int tile_pass(heis_ctx* h, const TileArgs& A, int T) {
    if (h->L % 4 || h->L / T < 2) return 1;
    if (h->dim == 2) {
        switch (T) {
            case 16: return launch_tile<2, 16>(h, A);
            case 32: return launch_tile<2, 32>(h, A);
            case 64: return launch_tile<2, 64>(h, A);
            default: return 1;
        }
    }
    switch (T) {
        case 4: return launch_tile<3, 4>(h, A);
        case 8: return launch_tile<3, 8>(h, A);
        case 16: return launch_tile<3, 16>(h, A);
        default: return 1;
    }
}

}  // namespace
}  // namespace ising

using namespace ising;

extern "C" {

heis_handle heis_create(int dim, int L, uint64_t seed) {
    if (dim < 2 || dim > 3 || L < 2 || (L & 1)) {
        set_error("heis_create: need dim in {2,3} and even L >= 2 (got dim=%d L=%d)", dim, L);
        return nullptr;
    }
    double n = 1.0;
    for (int d = 0; d < dim; ++d) n *= (double)L;
    if (n > 4294967296.0) {
        set_error("heis_create: N = L^dim must not exceed 2^32");
        return nullptr;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        set_error("no CUDA device: libising_b200 has no CPU path");
        return nullptr;
    }
    heis_ctx* h = new (std::nothrow) heis_ctx;
    if (!h) { set_error("out of host memory"); return nullptr; }
    h->dim = dim; h->L = L; h->seed = seed; h->N = (uint64_t)n;
    h->d_s = (float*)dev_alloc(3 * h->N * sizeof(float));
    h->d_obs = (double*)dev_alloc(4 * sizeof(double));
    if (!h->d_s || !h->d_obs) { heis_destroy(h); return nullptr; }
    const unsigned blocks = (unsigned)((h->N + 255) / 256);
    k_heis_hot_start<<<blocks, 256, 0, hooks().stream>>>(h->d_s, h->N, (uint32_t)seed, (uint32_t)(seed >> 32));
    count_launch();
    if (cudaGetLastError() != cudaSuccess) { set_error("hot-start launch failed"); heis_destroy(h); return nullptr; }
    return h;
}

void heis_destroy(heis_handle h) {
    if (!h) return;
    cudaStreamSynchronize(hooks().stream);
    dev_free(h->d_s);
    dev_free(h->d_obs);
    dev_free(h->d_xface);
    delete h;
}

static int heis_sweep_impl(heis_handle h, double beta, int n_sweeps, int tile, int k_inner, double* d_series) {
    if (!h) { set_error("heis_sweep: NULL handle"); return ISING_EINVAL; }
    if (!(beta >= 0.0) || !std::isfinite(beta) || n_sweeps < 0 || k_inner < 1) {
        set_error("heis_sweep: need finite beta >= 0, n_sweeps >= 0, k_inner >= 1");
        return ISING_EINVAL;
    }
    const int T = tile == 0 ? h->L : tile;
    if (!tile_valid(h, T)) {
        set_error("heis_sweep: tile %d invalid for L=%d (T even, T | L, L/T even or T == L)", T, h->L);
        return ISING_EINVAL;
    }
    const float betaf = (float)beta;
    const uint32_t k0 = (uint32_t)h->seed, k1 = (uint32_t)(h->seed >> 32);
    for (int pass = 0; pass < n_sweeps; ++pass) {
        const uint64_t t_first = h->t + (uint64_t)pass * k_inner;
        int rc = 1;
        if (!h->force_generic) {
            TileArgs A{h->d_s, nullptr, h->N, t_first, h->L, h->L / T, 0, k_inner, 0u, k0, k1, betaf};
            rc = tile_pass(h, A, T);
            if (rc < 0) return rc;
            if (rc == 0) h->last_path = "heis_tile";
        }
        if (rc == 1) {
            h->last_path = "heis_generic";
            h->xface_T = 0;
            const unsigned blocks = (unsigned)((h->N / 4 + 255) / 256);
            for (int C = 0; C < (T == h->L ? 1 : 2); ++C)
                for (int j = 0; j < k_inner; ++j)
                    for (int c = 0; c < 2; ++c) {
                        GenArgs G{h->d_s, h->N, 2 * (t_first + (uint64_t)j) + (uint64_t)c, h->L, h->dim, T, C, c, k0, k1, betaf};
                        k_heis_generic<<<blocks, 256, 0, hooks().stream>>>(G);
                        count_launch();
                    }
            ISING_CUDA_OK(cudaGetLastError());
        }
        if (d_series) {
            const unsigned blocks = (unsigned)std::min<uint64_t>((h->N + 255) / 256, 148 * 8);
            k_heis_observables<<<blocks, 256, 0, hooks().stream>>>(h->d_s, h->N, h->L, h->dim, d_series + (size_t)pass * 4);
            count_launch();
        }
    }
    h->t += (uint64_t)n_sweeps * k_inner;
    return 0;
}

int heis_sweep(heis_handle h, double beta, int n_sweeps, int tile, int k_inner) {
    return heis_sweep_impl(h, beta, n_sweeps, tile, k_inner, nullptr);
}

int heis_sweep_series(heis_handle h, double beta, int n_sweeps, int tile, int k_inner, double* E, double* M) {
    if (!h) { set_error("heis_sweep_series: NULL handle"); return ISING_EINVAL; }
    if (n_sweeps <= 0 || (!E && !M)) return heis_sweep_impl(h, beta, n_sweeps, tile, k_inner, nullptr);
    cudaStream_t st = hooks().stream;
    double* d_series = (double*)dev_alloc((size_t)n_sweeps * 4 * sizeof(double));      // {E, Mx, My, Mz} per pass
    if (!d_series) return ISING_ENOMEM;
    int rc = 0;
    if (cudaMemsetAsync(d_series, 0, (size_t)n_sweeps * 4 * sizeof(double), st) != cudaSuccess) { set_error("heis_sweep_series: memset failed"); rc = ISING_ECUDA; }
    if (!rc) rc = heis_sweep_impl(h, beta, n_sweeps, tile, k_inner, d_series);
    if (!rc && E && cudaMemcpy2DAsync(E, sizeof(double), d_series, 4 * sizeof(double), sizeof(double), (size_t)n_sweeps,
                                      is_device_ptr(E) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = ISING_ECUDA;
    if (!rc && M && cudaMemcpy2DAsync(M, 3 * sizeof(double), d_series + 1, 4 * sizeof(double), 3 * sizeof(double), (size_t)n_sweeps,
                                      is_device_ptr(M) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = ISING_ECUDA;
    if (rc == ISING_ECUDA) { set_error("heis_sweep_series: copy of the series failed: %s", cudaGetErrorString(cudaGetLastError())); }
    cudaStreamSynchronize(st);
    dev_free(d_series);
    return rc;
}

int heis_observables(heis_handle h, double* E, double* M) {
    if (!h) { set_error("heis_observables: NULL handle"); return ISING_EINVAL; }
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemsetAsync(h->d_obs, 0, 4 * sizeof(double), st));
    const unsigned blocks = (unsigned)std::min<uint64_t>((h->N + 255) / 256, 148 * 8);
    k_heis_observables<<<blocks, 256, 0, st>>>(h->d_s, h->N, h->L, h->dim, h->d_obs);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    if (E) ISING_CUDA_OK(cudaMemcpyAsync(E, h->d_obs, sizeof(double), is_device_ptr(E) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st));
    if (M) ISING_CUDA_OK(cudaMemcpyAsync(M, h->d_obs + 1, 3 * sizeof(double), is_device_ptr(M) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st));
    ISING_CUDA_OK(cudaStreamSynchronize(st));
    return 0;
}

int heis_copy_spins(heis_handle h, float* dst) {
    if (!h || !dst) { set_error("heis_copy_spins: NULL argument"); return ISING_EINVAL; }
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemcpyAsync(dst, h->d_s, 3 * h->N * sizeof(float), is_device_ptr(dst) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st));
    ISING_CUDA_OK(cudaStreamSynchronize(st));
    return 0;
}

int heis_set_spins(heis_handle h, const float* src) {
    if (!h || !src) { set_error("heis_set_spins: NULL argument"); return ISING_EINVAL; }
    cudaStream_t st = hooks().stream;
    h->xface_T = 0;
    ISING_CUDA_OK(cudaMemcpyAsync(h->d_s, src, 3 * h->N * sizeof(float), is_device_ptr(src) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
    ISING_CUDA_OK(cudaStreamSynchronize(st));
    return 0;
}

int heis_get_counter(heis_handle h, uint64_t* t) {
    if (!h || !t) { set_error("heis_get_counter: NULL argument"); return ISING_EINVAL; }
    *t = h->t;
    return 0;
}

int heis_set_counter(heis_handle h, uint64_t t) {
    if (!h) { set_error("heis_set_counter: NULL handle"); return ISING_EINVAL; }
    h->t = t;
    return 0;
}

const char* heis_sweep_path(heis_handle h) { return h ? h->last_path : "none"; }

int heis_force_generic(heis_handle h, int on) {
    if (!h) { set_error("heis_force_generic: NULL handle"); return ISING_EINVAL; }
    h->force_generic = on ? 1 : 0;
    return 0;
}

}  // extern "C"
