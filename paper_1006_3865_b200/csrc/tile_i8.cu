// tile_i8.cu — the 2D double-checkerboard tile kernel on int8 tile records (a1, a3-a7).
//
// HBM layout ("tile records"): the lattice is stored tile by tile so that a
// tile and each piece of its halo are contiguous, 16-byte aligned runs:
//   record(r, ty, tx) at ((r*B + ty)*B + tx) * (T*T + 2T) bytes, B = L/T, holding
//     rows rr = 0..T-1, T bytes each: [T/2 bytes fine colour 0][T/2 bytes fine colour 1];
//       byte j of part c is the site x = 2j + ((rr + c) & 1)   (colour-split row)
//     left  edge column (x = 0),   T bytes by rr      — read by the tile to the left as halo
//     right edge column (x = T-1), T bytes by rr      — read by the tile to the right
//   bytes are 0/1 (1 = spin +1).  A tile visit reads T*T + 4T bytes and writes T*T + 2T,
//   against the algorithmic 2*T*T + 4T (S8d): no sector is fetched for a single halo byte.
//
// Kernel: one launch per coarse colour.  A warp owns 64 tile rows at a time
// (one 64x64 tile or two 32x32 tiles); lane l owns rows 2m, 2m+1 so that within a
// half-sweep the x-offset of the other colour is warp-uniform.  Staging (a3) is a
// per-warp cp.async pipeline into shared memory, so neither a block barrier nor an
// mbarrier is needed: k x {even sites, __syncwarp, odd sites, __syncwarp},
// then the rows and the two edge columns go back with 128-bit stores (a7).
//
// Arithmetic per 32-bit word = 4 same-colour sites = one Philox4x32-10 call (S8c.3):
//   u    = up + down + left + right neighbour bytes (0..4 per byte)
//   tot  = n_sat + 3 + #{m : r >= thr[m]},  n_sat = s ? u : 4 - u
//   flip <=> tot <= 7  <=> n_sat + #{...} <= 4   (common.cuh: equals S8c.5)
//   r >= thr[m] is the carry of r + (2^32 - thr[m]), taken as the high word of one
//   IMAD.WIDE.U32 so that the compare runs on the FMA pipe next to Philox's multiplies.
#include "kernels.h"
#include "philox.cuh"

namespace ising {

namespace {

template <int T>
struct TG {
    static constexpr int W = T / 8;                    // 32-bit words per row part
    static constexpr int NT = 64 / T;                  // tiles per warp job
    static constexpr int HALF = T / 2;                 // bytes per row part
    static constexpr int P = T + 16;                   // smem slot pitch (one spare granule)
    static constexpr int IMG = (T + 2) * P + 2 * T;    // smem image of one tile + halo
    static constexpr int REC = T * T + 2 * T;          // HBM record bytes
    static constexpr int GR = T / 16;                  // 16-byte granules per row
    static constexpr int CH = T * GR + 4 * GR;         // cp.async chunks per tile
};

// Row rho (0 = top halo row, 1..T = tile rows, T+1 = bottom halo) lives in slot rho, shifted
// by one granule on every second group of 8 rows: with lanes owning rows 2m, 2m+1 this makes
// every quarter-warp LDS.128/STS.128 hit 8 distinct 16-byte bank groups.
template <int T>
__device__ __forceinline__ uint32_t slot_off(int rho) {
    return (uint32_t)rho * TG<T>::P + (((uint32_t)rho >> 3) & 1u) * 16u;
}

__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void* gptr) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

struct AcceptDev {
    uint32_t thr1, thr2;  // r >= thr[m] counts one (thr[m] == 0 counts always, as it must);
                          // thr[m] == 2^32 (beta = 0) is not representable: api.cu routes it to generic.cu
    uint32_t base;        // 3 in each byte
};

// One word = 4 sites.  S: own spins (0/1 bytes); U, D, X, Xs: the four neighbour words.
//   n_sat = number of neighbours equal to s;  tot = n_sat + 3 + #{m : r >= thr[m]}
//   flip <=> tot <= 7 <=> bit 3 of the byte clear.
__device__ __forceinline__ uint32_t metropolis_word(uint32_t S, uint32_t U, uint32_t D, uint32_t X, uint32_t Xs,
                                                    const u32x4& rnd, const AcceptDev& a) {
    constexpr uint32_t ONES = 0x01010101u;
    const uint32_t eU = U ^ S ^ ONES, eD = D ^ S ^ ONES, eX = X ^ S ^ ONES, eXs = Xs ^ S ^ ONES;
    uint32_t tot = eU + eD + eX;
    tot = tot + eXs + a.base;
    if (rnd.x >= a.thr1) tot += 0x00000001u;
    if (rnd.x >= a.thr2) tot += 0x00000001u;
    if (rnd.y >= a.thr1) tot += 0x00000100u;
    if (rnd.y >= a.thr2) tot += 0x00000100u;
    if (rnd.z >= a.thr1) tot += 0x00010000u;
    if (rnd.z >= a.thr2) tot += 0x00010000u;
    if (rnd.w >= a.thr1) tot += 0x01000000u;
    if (rnd.w >= a.thr2) tot += 0x01000000u;
    return S ^ (~(tot >> 3) & ONES);
}

template <int W>
__device__ __forceinline__ void lds_part(uint32_t addr, uint32_t (&v)[W]) {
#pragma unroll
    for (int i = 0; i < W; i += 4)
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];\n"
                     : "=r"(v[i]), "=r"(v[i + 1]), "=r"(v[i + 2]), "=r"(v[i + 3])
                     : "r"(addr + 4u * i)
                     : "memory");
}
template <int W>
__device__ __forceinline__ void sts_part(uint32_t addr, const uint32_t (&v)[W]) {
#pragma unroll
    for (int i = 0; i < W; i += 4)
        asm volatile("st.shared.v4.u32 [%4], {%0,%1,%2,%3};\n" ::"r"(v[i]), "r"(v[i + 1]), "r"(v[i + 2]),
                     "r"(v[i + 3]), "r"(addr + 4u * i)
                     : "memory");
}
__device__ __forceinline__ uint32_t lds_u8(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];\n" : "=r"(v) : "r"(addr) : "memory");
    return v;
}

// Update one row part.  Q = (row + colour) & 1: Q = 0 -> site x = 2j, neighbours X[j-1], X[j]
// (halo byte hb = site x = -1); Q = 1 -> x = 2j+1, neighbours X[j], X[j+1] (hb = site x = T).
template <int W, int Q>
__device__ __forceinline__ void update_part(uint32_t (&O)[W], const uint32_t (&U)[W],
                                            const uint32_t (&D)[W], const uint32_t (&X)[W], uint32_t hb,
                                            uint32_t group0, uint32_t Hlo, uint32_t Hhi, uint32_t k0,
                                            uint32_t k1, const AcceptDev& a) {
#pragma unroll
    for (int w = 0; w < W; ++w) {
        uint32_t xs;
        if (Q == 0) xs = (w == 0) ? ((X[0] << 8) | hb) : __funnelshift_l(X[w - 1], X[w], 8);
        else xs = (w == W - 1) ? ((X[w] >> 8) | (hb << 24)) : __funnelshift_r(X[w], X[w + 1], 8);
        const u32x4 rnd = philox4x32_10(group0 + (uint32_t)w, kTagSweep, Hlo, Hhi, k0, k1);
        O[w] = metropolis_word(O[w], U[w], D[w], X[w], xs, rnd, a);
    }
}

struct TileArgs {
    uint8_t* tiles;              // records, replica-major
    const uint64_t* seeds;
    int L, B, R;
    int C;                       // coarse colour of this launch
    int k;
    uint64_t t_first;            // inner-sweep index of the first of the k sweeps
    uint32_t njobs;              // warp jobs in this launch
    AcceptDev acc;
};

template <int T>
__device__ __forceinline__ void job_tile(const TileArgs& A, uint32_t job, int sub, int& r, int& tx, int& ty) {
    // colour-C tiles enumerated row by row: index q -> ty = q / (B/2), tx = 2*(q % (B/2)) + ((ty + C) & 1)
    const uint32_t per_rep = (uint32_t)A.B * (uint32_t)A.B / 2u;
    const uint32_t q = job * TG<T>::NT + (uint32_t)sub;
    r = (int)(q / per_rep);
    const uint32_t qq = q - (uint32_t)r * per_rep;
    const uint32_t hb = (uint32_t)A.B >> 1;
    ty = (int)(qq / hb);
    tx = (int)(2u * (qq - (uint32_t)ty * hb)) + ((ty + A.C) & 1);
}

__device__ __forceinline__ const uint8_t* rec_ptr(const TileArgs& A, int rec_bytes, int r, int tx, int ty) {
    return A.tiles + ((size_t)((size_t)r * A.B + ty) * A.B + tx) * (size_t)rec_bytes;
}

// a3: stage one job (NT tiles + halos) with 16-byte cp.async, chunk i -> lane i % 32.
template <int T>
__device__ __forceinline__ void stage_job(const TileArgs& A, uint32_t job, uint32_t stage_addr, int lane) {
    using G = TG<T>;
    for (int idx = lane; idx < G::NT * G::CH; idx += 32) {
        const int sub = idx / G::CH;
        const int ch = idx - sub * G::CH;
        int r, tx, ty;
        job_tile<T>(A, job, sub, r, tx, ty);
        const uint32_t img = stage_addr + (uint32_t)sub * G::IMG;
        const uint8_t* src;
        uint32_t dst;
        if (ch < T * G::GR) {                                  // interior rows
            const int row = ch / G::GR, g = ch - row * G::GR;
            src = rec_ptr(A, G::REC, r, tx, ty) + ch * 16;
            dst = img + slot_off<T>(row + 1) + g * 16;
        } else {
            const int e = ch - T * G::GR;
            const int which = e / G::GR, g = e - which * G::GR;
            const int B = A.B;
            if (which == 0) {                                  // top halo row = last row of the tile above
                src = rec_ptr(A, G::REC, r, tx, ty == 0 ? B - 1 : ty - 1) + (T - 1) * T + g * 16;
                dst = img + slot_off<T>(0) + g * 16;
            } else if (which == 1) {                           // bottom halo row = first row of the tile below
                src = rec_ptr(A, G::REC, r, tx, ty == B - 1 ? 0 : ty + 1) + g * 16;
                dst = img + slot_off<T>(T + 1) + g * 16;
            } else if (which == 2) {                           // left halo column = right edge of the left tile
                src = rec_ptr(A, G::REC, r, tx == 0 ? B - 1 : tx - 1, ty) + T * T + T + g * 16;
                dst = img + (T + 2) * G::P + g * 16;
            } else {                                           // right halo column = left edge of the right tile
                src = rec_ptr(A, G::REC, r, tx == B - 1 ? 0 : tx + 1, ty) + T * T + g * 16;
                dst = img + (T + 2) * G::P + T + g * 16;
            }
        }
        cp_async16(dst, src);
    }
}

// a4-a6: the k inner sweeps of one staged job, entirely in shared memory + registers.
template <int T>
__device__ __forceinline__ void sweep_job(const TileArgs& A, uint32_t job, uint32_t stage_addr, int lane) {
    using G = TG<T>;
    constexpr int W = G::W;
    const int sub = lane / G::HALF;
    const int m = lane - sub * G::HALF;
    int r, tx, ty;
    job_tile<T>(A, job, sub, r, tx, ty);
    const uint32_t img = stage_addr + (uint32_t)sub * G::IMG;
    const uint64_t seed = A.seeds[r];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    // Philox group of word 0 of row rr: (L/8)*(ty*T + rr) + tx*(T/8)   (S8c.3, p = i >> 1)
    const uint32_t gA = (uint32_t)(A.L >> 3) * (uint32_t)(ty * T + 2 * m) + (uint32_t)tx * W;
    const uint32_t gB = gA + (uint32_t)(A.L >> 3);
    const uint32_t sA = img + slot_off<T>(2 * m + 1);      // row 2m
    const uint32_t sB = img + slot_off<T>(2 * m + 2);      // row 2m+1
    const uint32_t sU = img + slot_off<T>(2 * m);          // row 2m-1 (or top halo)
    const uint32_t sD = img + slot_off<T>(2 * m + 3);      // row 2m+2 (or bottom halo)
    const uint32_t hcL = img + (T + 2) * G::P, hcR = hcL + T;
    for (int j = 0; j < A.k; ++j) {
        const uint64_t t = A.t_first + (uint64_t)j;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const uint64_t H = 2 * t + (uint64_t)c;
            const uint32_t Hlo = (uint32_t)H, Hhi = (uint32_t)(H >> 32);
            const uint32_t act = (uint32_t)c * G::HALF, oth = (uint32_t)(1 - c) * G::HALF;
            uint32_t OA[W], OB[W], XA[W], XB[W], UA[W], DB[W];
            lds_part<W>(sA + act, OA);
            lds_part<W>(sA + oth, XA);
            lds_part<W>(sB + act, OB);
            lds_part<W>(sB + oth, XB);
            lds_part<W>(sU + oth, UA);
            lds_part<W>(sD + oth, DB);
            if (c == 0) {   // row 2m: Q = 0 (halo x = -1); row 2m+1: Q = 1 (halo x = T)
                const uint32_t hA = lds_u8(hcL + 2 * m), hB = lds_u8(hcR + 2 * m + 1);
                update_part<W, 0>(OA, UA, XB, XA, hA, gA, Hlo, Hhi, k0, k1, A.acc);
                update_part<W, 1>(OB, XA, DB, XB, hB, gB, Hlo, Hhi, k0, k1, A.acc);
            } else {        // row 2m: Q = 1; row 2m+1: Q = 0
                const uint32_t hA = lds_u8(hcR + 2 * m), hB = lds_u8(hcL + 2 * m + 1);
                update_part<W, 1>(OA, UA, XB, XA, hA, gA, Hlo, Hhi, k0, k1, A.acc);
                update_part<W, 0>(OB, XA, DB, XB, hB, gB, Hlo, Hhi, k0, k1, A.acc);
            }
            sts_part<W>(sA + act, OA);
            sts_part<W>(sB + act, OB);
            __syncwarp();
        }
    }
}

// a7: rows back to the records with 16-byte stores (chunk i -> lane i % 32), then the edge columns.
template <int T>
__device__ __forceinline__ void writeback_job(const TileArgs& A, uint32_t job, uint32_t stage_addr, int lane) {
    using G = TG<T>;
    for (int idx = lane; idx < G::NT * T * G::GR; idx += 32) {
        const int sub = idx / (T * G::GR);
        const int ch = idx - sub * (T * G::GR);
        int r, tx, ty;
        job_tile<T>(A, job, sub, r, tx, ty);
        const int row = ch / G::GR, g = ch - row * G::GR;
        uint32_t v[4];
        lds_part<4>(stage_addr + (uint32_t)sub * G::IMG + slot_off<T>(row + 1) + g * 16, v);
        uint8_t* dst = const_cast<uint8_t*>(rec_ptr(A, G::REC, r, tx, ty)) + ch * 16;
        *reinterpret_cast<uint4*>(dst) = make_uint4(v[0], v[1], v[2], v[3]);
    }
    {
        const int sub = lane / G::HALF;
        const int m = lane - sub * G::HALF;
        int r, tx, ty;
        job_tile<T>(A, job, sub, r, tx, ty);
        const uint32_t img = stage_addr + (uint32_t)sub * G::IMG;
        const uint32_t sA = img + slot_off<T>(2 * m + 1), sB = img + slot_off<T>(2 * m + 2);
        // x = 0 is colour (rr & 1), byte 0 of that part; x = T-1 is colour ((rr+1) & 1), last byte.
        const uint32_t lA = lds_u8(sA), lB = lds_u8(sB + G::HALF);
        const uint32_t rA = lds_u8(sA + G::HALF + G::HALF - 1), rB = lds_u8(sB + G::HALF - 1);
        uint8_t* rec = const_cast<uint8_t*>(rec_ptr(A, G::REC, r, tx, ty));
        *reinterpret_cast<uint16_t*>(rec + T * T + 2 * m) = (uint16_t)(lA | (lB << 8));
        *reinterpret_cast<uint16_t*>(rec + T * T + T + 2 * m) = (uint16_t)(rA | (rB << 8));
    }
}

template <int T, int S>
__global__ void __launch_bounds__(128) k_tile_i8(TileArgs A) {
    using G = TG<T>;
    extern __shared__ __align__(16) uint8_t smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int wpb = blockDim.x >> 5;
    constexpr uint32_t STAGE = G::NT * G::IMG;
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(smem) + (uint32_t)warp * S * STAGE;
    const uint32_t first = blockIdx.x * wpb + warp;
    const uint32_t stride = gridDim.x * wpb;
    // prologue: S-1 jobs in flight
#pragma unroll
    for (int s = 0; s < S - 1; ++s) {
        const uint32_t job = first + (uint32_t)s * stride;
        if (job < A.njobs) stage_job<T>(A, job, base + (uint32_t)s * STAGE, lane);
        cp_async_commit();
    }
    uint32_t it = 0;
    for (uint32_t job = first; job < A.njobs; job += stride, ++it) {
        const uint32_t nxt = job + (uint32_t)(S - 1) * stride;
        if (nxt < A.njobs) stage_job<T>(A, nxt, base + ((it + S - 1) % S) * STAGE, lane);
        cp_async_commit();
        cp_async_wait<S - 1>();
        __syncwarp();
        const uint32_t st = base + (it % S) * STAGE;
        sweep_job<T>(A, job, st, lane);
        writeback_job<T>(A, job, st, lane);
        __syncwarp();
    }
    cp_async_wait<0>();
}

// ---- layout converters (a11); not on the timed path ------------------------------------
template <bool TO_TILES>
__global__ void k_convert_i8(int8_t* __restrict__ canon, uint8_t* __restrict__ tiles, int L, int T, int R) {
    const uint64_t N = (uint64_t)L * L;
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= N * (uint64_t)R) return;
    const int r = (int)(gid / N);
    const uint64_t i = gid - (uint64_t)r * N;
    const int x = (int)(i % L), y = (int)(i / L);
    const int B = L / T;
    const int tx = x / T, ty = y / T, lx = x - tx * T, ly = y - ty * T;
    const int c = (lx + ly) & 1, j = lx >> 1;
    uint8_t* rec = tiles + ((size_t)((size_t)r * B + ty) * B + tx) * (size_t)(T * T + 2 * T);
    if (TO_TILES) {
        const uint8_t v = canon[gid] > 0 ? 1 : 0;
        rec[ly * T + c * (T / 2) + j] = v;
        if (lx == 0) rec[T * T + ly] = v;
        if (lx == T - 1) rec[T * T + T + ly] = v;
    } else {
        canon[gid] = rec[ly * T + c * (T / 2) + j] ? 1 : -1;
    }
}

template <int T, int S>
int launch_colour(ising_ctx* h, TileArgs& A, int warps, int ctas_per_sm) {
    using G = TG<T>;
    const size_t smem = (size_t)warps * S * G::NT * G::IMG;
    if (int rc = set_max_dynamic_smem<k_tile_i8<T, S>>(200 * 1024)) return rc;
    const uint32_t need = (A.njobs + warps - 1) / warps;
    uint32_t grid = 148u * (uint32_t)ctas_per_sm;
    if (grid > need) grid = need;
    k_tile_i8<T, S><<<grid, warps * 32, smem, hooks().stream>>>(A);
    count_launch();
    return 0;
}

int env_int(const char* name, int dflt) {
    const char* v = getenv(name);
    return v ? atoi(v) : dflt;
}

}  // namespace

bool tile_i8_supported(const ising_ctx* h, int T) {
    if (h->dim != 2 || h->has_J) return false;
    if (T != 32 && T != 64) return false;
    if (h->L % T) return false;
    const int B = h->L / T;
    return B >= 2 && (B % 2 == 0);
}

size_t tile_i8_bytes(const ising_ctx* h, int T) {
    const size_t B = (size_t)(h->L / T);
    return (size_t)h->R * B * B * (size_t)(T * T + 2 * T);
}

int launch_canon_to_tile_i8(ising_ctx* h, int T, const int8_t* d_canon, void* d_tiles) {
    const uint64_t total = h->N * (uint64_t)h->R;
    k_convert_i8<true><<<(unsigned)((total + 255) / 256), 256, 0, hooks().stream>>>(
        const_cast<int8_t*>(d_canon), (uint8_t*)d_tiles, h->L, T, h->R);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_tile_i8_to_canon(ising_ctx* h, int T, const void* d_tiles, int8_t* d_canon) {
    const uint64_t total = h->N * (uint64_t)h->R;
    k_convert_i8<false><<<(unsigned)((total + 255) / 256), 256, 0, hooks().stream>>>(
        d_canon, (uint8_t*)const_cast<void*>(d_tiles), h->L, T, h->R);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// a1: one outer pass = colour-0 launch, colour-1 launch, k inner sweeps each.
int launch_tile_i8_pass(ising_ctx* h, const Accept& acc, int T, int k, uint64_t t_first) {
    TileArgs A;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.L = h->L; A.B = h->L / T; A.R = h->R; A.k = k; A.t_first = t_first;
    const uint32_t tiles_per_colour = (uint32_t)((size_t)h->R * A.B * A.B / 2);
    A.njobs = tiles_per_colour / (uint32_t)(64 / T);
    A.acc.thr1 = acc.thr[0];
    A.acc.thr2 = acc.thr[1];
    A.acc.base = 3u * 0x01010101u;
    static const int warps = env_int("ISING_TILE_WARPS", 4);
    static const int stages = env_int("ISING_TILE_STAGES", 3);
    static const int cps_env = env_int("ISING_TILE_CTAS_PER_SM", 0);
    const int cps = cps_env > 0 ? cps_env : (T == 64 ? 3 : 5);
    for (int C = 0; C < 2; ++C) {
        A.C = C;
        int rc;
        if (T == 64) rc = stages == 2 ? launch_colour<64, 2>(h, A, warps, cps) : launch_colour<64, 3>(h, A, warps, cps);
        else rc = stages == 2 ? launch_colour<32, 2>(h, A, warps, cps) : launch_colour<32, 3>(h, A, warps, cps);
        if (rc) return rc;
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

}  // namespace ising
