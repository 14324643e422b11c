// tile3d_planes.cu — the 3D double-checkerboard tile kernel (8x8x8 tiles, "completely
// analogous"; BASELINE config 4) in multi-spin form, RNG mapping "planes".
//
// A 32-bit word holds the 32 same-colour sites of one z-slice of a tile = one RNG block of the 3D
// planes mapping (4 pairs p_x x 8 rows y): bit j = 4*ly + p_x.  A tile is 8 slices x 2 colours =
// 16 words; a warp owns 4 tiles, lane = (tile, lz) holds the two words of its slice.  Neighbours of
// the 32 active sites: z-1 / z+1 = the other colour's word of the lane below / above (shuffle; halo
// word at the tile faces), y-1 / y+1 = the same word shifted by one row (4 bits; 4 halo bits from
// the tile in front / behind), x-1 / x+1 = the same word and the word shifted by one pair inside
// each row, left in rows where the active site is the left one of its pair, right in the others
// (one halo bit per row).  6-input bit adder, three thresholds (dE = 4, 8, 12), otherwise as 2D.
//
// HBM tile record = body + 96 bytes of bit-packed face copies written by the tile itself, so that
// a neighbour reads every halo as a few contiguous bytes and needs no unpacking:
//   int8 body 512 B: the 16 bytes (slice lz, colour cc, rows 4h..4h+3) at ((cc*2+h)*8 + lz)*16, byte piece_byte(4*(ly&3)+p_x)
//   bits body  64 B: word (cc, lz) at (cc*8 + lz)*4
//   faces: XL[8] words (sites x=0 of slice lz, row ly at bit 4ly+3), XR[8] words (x=7, bit 4ly),
//          YL[8] bytes (row y=0: colour 0 pairs in bits 0-3, colour 1 in 4-7), YR[8] bytes (y=7),
//          ZL 2 words (slice 0, colour 0 and 1), ZR 2 words (slice 7).
#include <cooperative_groups.h>

#include <cstdlib>

#include "kernels.h"
#include "tile3d_planes_device.cuh"
#include "grid3d_device.cuh"

namespace ising {

namespace {

// ---- layout converters (a11).  MODE 0/2: canonical -> int8 / bit records (face copies included; bit
// fields by atomicOr into zeroed storage), MODE 1/3: records -> canonical.  One thread per site.
template <int MODE>
__global__ void k_convert3d(int8_t* __restrict__ canon, uint8_t* __restrict__ tiles, int L, int R) {
    const uint64_t N = (uint64_t)L * L * L;
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= N * (uint64_t)R) return;
    const int r = (int)(gid / N);
    const uint64_t i = gid - (uint64_t)r * N;
    const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / ((uint64_t)L * L));
    const int B = L / kT3;
    const int tx = x >> 3, ty = y >> 3, tz = z >> 3, lx = x & 7, ly = y & 7, lz = z & 7;
    const int cc = (lx + ly + lz) & 1, px = lx >> 1, j = 4 * ly + px;
    constexpr bool BITS = MODE >= 2;
    constexpr int REC = BITS ? kRec3Bits : kRec3I8;
    constexpr int BODY = BITS ? kBody3Bits : kBody3I8;
    uint8_t* rec = tiles + ((size_t)r * B * B * B + ((size_t)tz * B + ty) * B + tx) * REC;
    uint8_t* byte = rec + ((cc * 2 + (ly >> 2)) * 8 + lz) * 16 + piece_byte(4 * (ly & 3) + px);
    uint32_t* word = reinterpret_cast<uint32_t*>(rec) + cc * 8 + lz;
    if (MODE == 1) { canon[gid] = *byte ? 1 : -1; return; }
    if (MODE == 3) { canon[gid] = ((*word >> j) & 1u) ? 1 : -1; return; }
    const bool up = canon[gid] > 0;
    if (!BITS) *byte = up ? 1 : 0;
    if (!up) return;
    if (BITS) atomicOr(word, 1u << j);
    uint8_t* f = rec + BODY;
    if (lx == 0) atomicOr(reinterpret_cast<uint32_t*>(f + kXL) + lz, 1u << (4 * ly + 3));
    if (lx == 7) atomicOr(reinterpret_cast<uint32_t*>(f + kXR) + lz, 1u << (4 * ly));
    // byte-wide face fields live in 4-byte aligned words: set the bit through the containing word
    if (ly == 0) atomicOr(reinterpret_cast<uint32_t*>(f + kYL) + (lz >> 2), 1u << (8 * (lz & 3) + 4 * cc + px));
    if (ly == 7) atomicOr(reinterpret_cast<uint32_t*>(f + kYR) + (lz >> 2), 1u << (8 * (lz & 3) + 4 * cc + px));
    if (lz == 0) atomicOr(reinterpret_cast<uint32_t*>(f + kZL) + cc, 1u << j);
    if (lz == 7) atomicOr(reinterpret_cast<uint32_t*>(f + kZR) + cc, 1u << j);
}

// Couplings, canonical J[d][i] (bond i -> i + e_d) -> coupling records (zeroed first).  One thread per site: it owns
// the six bonds seen from that site, in the order of the neighbour words of half_sweep3 (Zm, Zp, Ym, Yp, O, X2).
__global__ void k_convert_couplings3d(const int8_t* __restrict__ J, uint32_t* __restrict__ jrec, int L) {
    const uint64_t N = (uint64_t)L * L * L;
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / ((uint64_t)L * L));
    const int B = L / kT3;
    const int tx = x >> 3, ty = y >> 3, tz = z >> 3, lx = x & 7, ly = y & 7, lz = z & 7;
    const int cc = (lx + ly + lz) & 1, px = lx >> 1, j = 4 * ly + px;
    const uint64_t ixm = i - x + (x == 0 ? L - 1 : x - 1);
    const uint64_t iym = y == 0 ? i + (uint64_t)L * (L - 1) : i - L;
    const uint64_t izm = z == 0 ? i + (uint64_t)L * L * (L - 1) : i - (uint64_t)L * L;
    const bool xp = J[i] < 0, xm = J[ixm] < 0, yp = J[N + i] < 0, ym = J[N + iym] < 0, zp = J[2 * N + i] < 0, zm = J[2 * N + izm] < 0;
    const bool left = (lx & 1) == 0;              // the other site of the aligned pair is x + 1 for a left site
    const bool b[6] = {zm, zp, ym, yp, left ? xp : xm, left ? xm : xp};
    uint32_t* w = jrec + ((((size_t)tz * B + ty) * B + tx) * 32 + (size_t)(cc * 8 + lz) * 2) * 4;
#pragma unroll
    for (int n = 0; n < 6; ++n)
        if (b[n]) atomicOr(w + n, 1u << j);
}

// a10 directly on the 3D tile records: one launch per coarse colour C adds the colour-C tiles' share to E[r], M[r]
// (zeroed by the caller); the four tiles of a warp job belong to one replica (B^3/2 is a multiple of 4).  The warps of a
// CTA meet in shared memory and one thread adds per replica (every CTA adds to the same two words: fewer, larger adds).
constexpr int kObs3Warps = 8;
template <bool BITS, bool HASJ>
__global__ void __launch_bounds__(kObs3Warps * 32) k_observables3d(Plane3Args A, long long* __restrict__ E, long long* __restrict__ M) {
    __shared__ int s_r[kObs3Warps], s_up[kObs3Warps], s_unsat[kObs3Warps];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t job = blockIdx.x * (blockDim.x >> 5) + (uint32_t)w;
    int r = -1, up = 0, unsat = 0;
    if (job < A.njobs) {                                   // warp-uniform
        const int sub = lane >> 3, lz = lane & 7;
        const Tile3 t = job_tile3(A, job * 4u + (uint32_t)sub);
        Slice s;
        load_slice<BITS>(A, t, lz, s);
        load_couplings<HASJ>(A, t, lz, s);
        count_slice<HASJ>(s, lz, up, unsat);
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            up += __shfl_xor_sync(0xffffffffu, up, d);
            unsat += __shfl_xor_sync(0xffffffffu, unsat, d);
        }
        r = __shfl_sync(0xffffffffu, t.r, 0);
    }
    if (lane == 0) { s_r[w] = r; s_up[w] = up; s_unsat[w] = unsat; }
    __syncthreads();
    if (threadIdx.x == 0) {
        const long long sites = 4ll * kT3 * kT3 * kT3;
        int cr = -1;
        long long m = 0, e = 0;
        for (int i = 0; i <= kObs3Warps; ++i) {
            const int ri = i < kObs3Warps ? s_r[i] : -1;
            if (ri != cr) {                                 // consecutive jobs: runs of equal r
                if (cr >= 0) {
                    if (M) atomicAdd(reinterpret_cast<unsigned long long*>(M + cr), (unsigned long long)m);
                    if (E) atomicAdd(reinterpret_cast<unsigned long long*>(E + cr), (unsigned long long)e);
                }
                cr = ri; m = 0; e = 0;
            }
            if (ri >= 0) {
                m += 2ll * s_up[i] - sites;
                e += 2ll * s_unsat[i] - 3ll * sites;
            }
        }
    }
}

// ---- coarse tiles other than the 8^3 register tile (Tc = 2, 4, or a power of two above 8) as masked half-sweeps, as in
// tile_planes.cu: bit j = 4 ly + px of a slice word is the site x = 8 tx + 2 px + a, y = 8 ty + ly, z = 8 tz + lz.
__device__ __forceinline__ uint32_t coarse_mask3(int Tc, const Tile3& t, int lz, int Cc) {
    if (Tc == 0) return 0xffffffffu;
    if (Tc >= kT3) {                                       // a register tile lies in one coarse tile: all or nothing
        const uint32_t par = ((uint32_t)(kT3 * t.tx) / (uint32_t)Tc + (uint32_t)(kT3 * t.ty) / (uint32_t)Tc +
                              (uint32_t)(kT3 * t.tz + lz) / (uint32_t)Tc) & 1u;
        return par == (uint32_t)Cc ? 0xffffffffu : 0u;
    }
    const uint32_t X1 = Tc == 4 ? 0xccccccccu : 0xaaaaaaaau;       // sites with odd x / Tc
    const uint32_t Y1 = Tc == 4 ? 0xffff0000u : 0xff00ff00u;       // sites with odd y / Tc
    const uint32_t tzp = ((uint32_t)lz / (uint32_t)Tc) & 1u;       // 8 / Tc is even: tz does not matter
    return ((uint32_t)Cc ^ tzp) ? (X1 ^ Y1) : ~(X1 ^ Y1);
}

template <bool HASJ>
__device__ __forceinline__ void half_sweep3_masked(const Plane3Args& A, Slice& s, int c, int lz, uint32_t g, uint32_t p_base,
                                                   uint64_t H, uint32_t k0, uint32_t k1, uint32_t mask) {
    const uint32_t old = s.S[c];
    half_sweep3<kNoSpec3, HASJ>(A, s, c, lz, g, p_base, H, k0, k1);
    s.S[c] = (s.S[c] & mask) | (old & ~mask);
}

// store_slice for a half-sweep that changed only fine colour c: that colour's pieces and the face copies.
template <bool BITS>
__device__ __forceinline__ void store_slice_colour(const Plane3Args& A, const Tile3& t, int lz, const Slice& s, const uint2* lut, int c) {
    constexpr int REC = BITS ? kRec3Bits : kRec3I8;
    constexpr int BODY = BITS ? kBody3Bits : kBody3I8;
    const int B = A.B;
    uint8_t* rec = A.tiles + ((size_t)t.r * B * B * B + ((size_t)t.tz * B + t.ty) * B + t.tx) * REC;
    const uint32_t w = c ? s.S[1] : s.S[0];
    if (BITS) {
        *reinterpret_cast<uint32_t*>(rec + (c * 8 + lz) * 4) = w;
    } else {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint2 a = __ldg(lut + ((w >> (16 * h)) & 0xffu));
            const uint2 b = __ldg(lut + ((w >> (16 * h + 8)) & 0xffu));
            stg128(rec + ((c * 2 + h) * 8 + lz) * 16, make_uint4(a.x, a.y, b.x, b.y));
        }
    }
    uint32_t XL, XR, YL, YR;
    face_words(s.S, lz, XL, XR, YL, YR);
    uint8_t* f = rec + BODY;
    reinterpret_cast<uint32_t*>(f + kXL)[lz] = XL;
    reinterpret_cast<uint32_t*>(f + kXR)[lz] = XR;
    f[kYL + lz] = (uint8_t)YL;
    f[kYR + lz] = (uint8_t)YR;
    if (lz == 0) *reinterpret_cast<uint2*>(f + kZL) = make_uint2(s.S[0], s.S[1]);
    if (lz == 7) *reinterpret_cast<uint2*>(f + kZR) = make_uint2(s.S[0], s.S[1]);
}

// a8 in 3D for L > 64: the plain checkerboard (tile == L) with a launch per half-sweep over all tiles.  Face words mix
// the two fine colours, but a word is written whole and the bits a neighbour uses in this launch (the other fine
// colour) are the same before and after.
template <bool BITS, bool HASJ>
__global__ void __launch_bounds__(kThreads3) k_tile3d_plain(Plane3Args A, int c, uint64_t tt, int Tc, int Cc) {
    const uint2* lut = kByteLutGlobal.e;
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int lane = threadIdx.x & 31;
    const uint32_t job = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (job >= A.njobs) return;
    const int sub = lane >> 3, lz = lane & 7;
    const uint32_t B = (uint32_t)A.B;
    uint32_t q = job * 4u + (uint32_t)sub;                      // all tiles, replica-major, (tz, ty, tx) row-major
    Tile3 t;
    t.r = (int)(q / (B * B * B)); q -= (uint32_t)t.r * B * B * B;
    t.tz = (int)(q / (B * B)); q -= (uint32_t)t.tz * B * B;
    t.ty = (int)(q / B); t.tx = (int)(q - (uint32_t)t.ty * B);
    Slice s;
    load_slice<BITS>(A, t, lz, s);
    load_couplings<HASJ>(A, t, lz, s);
    const uint64_t seed = A.seeds[t.r];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    const uint32_t z = (uint32_t)(t.tz * kT3 + lz);
    const uint32_t g = (z * B + (uint32_t)t.ty) * B + (uint32_t)t.tx;
    const uint32_t p_base = (uint32_t)(t.tx * 4) + (uint32_t)(A.L >> 1) * ((uint32_t)(t.ty * kT3) + (uint32_t)A.L * z);
    half_sweep3_masked<HASJ>(A, s, c, lz, g, p_base, 2 * tt + (uint64_t)c, k0, k1, coarse_mask3(Tc, t, lz, Cc));
    store_slice_colour<BITS>(A, t, lz, s, lut, c);
}

}  // namespace

static void fill_geometry3(Plane3Args& A, const ising_ctx* h) {
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = h->L; A.B = h->L / kT3; A.R = h->R;
    const uint32_t B = (uint32_t)A.B;
    A.per_rep = B * B * B / 2u; A.per_z = B * B / 2u; A.hb = B / 2u;
    A.magic_rep = fastdiv_magic(A.per_rep); A.magic_z = fastdiv_magic(A.per_z); A.magic_hb = fastdiv_magic(A.hb);
    A.njobs = (uint32_t)((size_t)h->R * A.per_rep / 4u);
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
}

static void fill_accept3(Plane3Args& A, const Accept& acc) {
    for (int m = 0; m < 3; ++m) {
        for (int q = 0; q < kHeadBits; ++q) A.u[m][q] = ((acc.thr[m] >> (31 - q)) & 1u) ? 0xffffffffu : 0u;
        A.tail[m] = acc.thr[m] & ((1u << kTailBits) - 1u);
    }
    A.force = acc.thr_is_2p32[0] ? 0xffffffffu : 0u;
}

// n passes of k plain-checkerboard sweeps in 3D: 2 n k launches.
int launch_tile3d_plain(ising_ctx* h, const Accept& acc, bool bits, int n, int k, uint64_t t_first, int Tc) {
    Plane3Args A = {};
    fill_geometry3(A, h);
    fill_accept3(A, acc);
    A.k = k; A.t_first = t_first; A.C = 0;
    A.njobs = (uint32_t)((size_t)h->R * A.B * A.B * A.B / 4u);
    const int warps = kThreads3 / 32;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((A.njobs + warps - 1) / warps); cfg.blockDim = dim3(warps * 32); cfg.stream = hooks().stream;
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
                    if (A.jrec) {
                        if (bits) ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile3d_plain<true, true>, A, c, tt, Tc, Cc));
                        else ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile3d_plain<false, true>, A, c, tt, Tc, Cc));
                    } else {
                        if (bits) ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile3d_plain<true, false>, A, c, tt, Tc, Cc));
                        else ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile3d_plain<false, false>, A, c, tt, Tc, Cc));
                    }
                    count_launch();
                }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// a10 on 3D tile records: E[r], M[r] (R values each, either may be null).
int launch_observables3d(ising_ctx* h, bool bits, long long* d_E, long long* d_M) {
    cudaStream_t st = hooks().stream;
    if (d_E) ISING_CUDA_OK(cudaMemsetAsync(d_E, 0, sizeof(long long) * h->R, st));
    if (d_M) ISING_CUDA_OK(cudaMemsetAsync(d_M, 0, sizeof(long long) * h->R, st));
    Plane3Args A = {};
    fill_geometry3(A, h);
    const int warps = kObs3Warps;
    const uint32_t grid = (A.njobs + warps - 1) / warps;
    for (int C = 0; C < 2; ++C) {
        A.C = C;
        if (A.jrec) {
            if (bits) k_observables3d<true, true><<<grid, warps * 32, 0, st>>>(A, d_E, d_M);
            else k_observables3d<false, true><<<grid, warps * 32, 0, st>>>(A, d_E, d_M);
        } else {
            if (bits) k_observables3d<true, false><<<grid, warps * 32, 0, st>>>(A, d_E, d_M);
            else k_observables3d<false, false><<<grid, warps * 32, 0, st>>>(A, d_E, d_M);
        }
        count_launch();
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

size_t coupling_record3d_bytes(const ising_ctx* h) {
    const size_t B = (size_t)(h->L / kT3);
    return B * B * B * 32 * sizeof(uint4);
}

int launch_convert_couplings3d(ising_ctx* h, void* d_jrec) {
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemsetAsync(d_jrec, 0, coupling_record3d_bytes(h), st));
    k_convert_couplings3d<<<(unsigned)((h->N + 255) / 256), 256, 0, st>>>(h->d_J, (uint32_t*)d_jrec, h->L);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

bool tile3d_supported(const ising_ctx* h, int T) {
    if (h->dim != 3 || h->J_per_replica || T != kT3 || h->L % kT3) return false;
    const int B = h->L / kT3;
    return B >= 2 && (B % 2 == 0);
}

size_t tile3d_bytes(const ising_ctx* h, bool bits) {
    const size_t B = (size_t)(h->L / kT3);
    return (size_t)h->R * B * B * B * (size_t)(bits ? kRec3Bits : kRec3I8);
}

int launch_canon_to_3d(ising_ctx* h, bool bits, const int8_t* d_canon, void* d_tiles) {
    const uint64_t total = h->N * (uint64_t)h->R;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemsetAsync(d_tiles, 0, tile3d_bytes(h, bits), st));
    if (bits) k_convert3d<2><<<blocks, 256, 0, st>>>(const_cast<int8_t*>(d_canon), (uint8_t*)d_tiles, h->L, h->R);
    else k_convert3d<0><<<blocks, 256, 0, st>>>(const_cast<int8_t*>(d_canon), (uint8_t*)d_tiles, h->L, h->R);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_3d_to_canon(ising_ctx* h, bool bits, const void* d_tiles, int8_t* d_canon) {
    const uint64_t total = h->N * (uint64_t)h->R;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    cudaStream_t st = hooks().stream;
    if (bits) k_convert3d<3><<<blocks, 256, 0, st>>>(d_canon, (uint8_t*)const_cast<void*>(d_tiles), h->L, h->R);
    else k_convert3d<1><<<blocks, 256, 0, st>>>(d_canon, (uint8_t*)const_cast<void*>(d_tiles), h->L, h->R);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// a1: one outer pass = colour-0 launch, colour-1 launch, k inner sweeps each.
int launch_tile3d_pass(ising_ctx* h, const Accept& acc, bool bits, int k, uint64_t t_first, bool use_jit) {
    Plane3Args A;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = h->L; A.B = h->L / kT3; A.R = h->R; A.k = k; A.t_first = t_first;
    const uint32_t B = (uint32_t)A.B;
    A.per_rep = B * B * B / 2u; A.per_z = B * B / 2u; A.hb = B / 2u;
    A.magic_rep = fastdiv_magic(A.per_rep); A.magic_z = fastdiv_magic(A.per_z); A.magic_hb = fastdiv_magic(A.hb);
    A.njobs = (uint32_t)((size_t)h->R * A.per_rep / 4u);
    for (int m = 0; m < 3; ++m) {
        for (int q = 0; q < kHeadBits; ++q) A.u[m][q] = ((acc.thr[m] >> (31 - q)) & 1u) ? 0xffffffffu : 0u;
        A.tail[m] = acc.thr[m] & ((1u << kTailBits) - 1u);
    }
    A.force = acc.thr_is_2p32[0] ? 0xffffffffu : 0u;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    const int warps = kThreads3 / 32;
    const uint32_t grid = (A.njobs + warps - 1) / warps;
    // specialised on the three threshold heads (planes_jit.cu) when asked for and available
    const unsigned long long hp3 = ((unsigned long long)(acc.thr[0] >> kTailBits) << 24) |
                                   ((unsigned long long)(acc.thr[1] >> kTailBits) << 12) | (unsigned long long)(acc.thr[2] >> kTailBits);
    cudaKernel_t spec = (use_jit && !A.force && !A.jrec) ? planes3d_jit_kernel(bits, hp3, 0 /* uniform key: measured -15 % on this kernel at k = 4, +2.6 % on k_grid3d */) : nullptr;
    h->last_jit = spec ? 1 : 0;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(warps * 32); cfg.stream = hooks().stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    static const int pdl = getenv("ISING_NO_PDL") ? 0 : 1;
    attr[0].val.programmaticStreamSerializationAllowed = pdl;
    cfg.attrs = attr; cfg.numAttrs = 1;
    for (int C = 0; C < 2; ++C) {
        A.C = C;
        if (spec) {
            void* args[] = {&A};
            ISING_CUDA_OK(cudaLaunchKernelExC(&cfg, (const void*)spec, args));
        } else if (A.jrec) {
            if (bits) ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile3d_planes<true, kNoSpec3, true>, A));
            else ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile3d_planes<false, kNoSpec3, true>, A));
        } else if (bits) {
            ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile3d_planes<true>, A));
        } else {
            ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile3d_planes<false>, A));
        }
        count_launch();
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// ---- whole lattice on chip, 3D (L <= 64): one thread-block cluster per replica, slices in registers, the 96-byte face
// areas of the tiles in shared memory, read by the neighbours through distributed shared memory; the design of
// k_resident_planes (tile_planes.cu) carried over.
constexpr int kRes3Warps = 4;
constexpr int kRes3MaxCluster = 16;

struct Res3Args {
    Plane3Args P;
    int n;
    uint32_t jobs_per_colour;      // per replica, 4 tiles per job
    long long* E;                  // optional series (a10 after every pass): E[pass * R + r], M[pass * R + r]
    long long* M;
    int plain;                     // 1: plain checkerboard of the whole lattice (tile == L), a barrier after every half-sweep
    int coarse;                    // with plain: coarse tile edge of a masked double checkerboard, or 0
};

template <bool BITS, bool HASJ>
__global__ void __launch_bounds__(kRes3Warps * 32) k_resident3d(Res3Args R) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    const uint32_t CL = cluster.num_blocks(), rank = cluster.block_rank();
    const Plane3Args& A = R.P;
    const int r = (int)(blockIdx.x / CL);
    const int lane = threadIdx.x & 31, wic = threadIdx.x >> 5;
    const uint32_t wg = rank * kRes3Warps + (uint32_t)wic;            // one job per warp and colour
    const int sub = lane >> 3, lz = lane & 7;
    const uint32_t B = (uint32_t)A.B, hb = B >> 1, JC = R.jobs_per_colour;
    const uint2* lut = kByteLutGlobal.e;
    __shared__ __align__(16) uint8_t faces[2][kRes3Warps][4][kFaces3];
    __shared__ int acc[2][2];          // rank 0 only: {#up, #unsatisfied bonds} of the replica, for even / odd passes
    if (threadIdx.x < 4) (&acc[0][0])[threadIdx.x] = 0;
    int* const acc0 = cluster.map_shared_rank(&acc[0][0], 0);
    const bool series = R.E != nullptr || R.M != nullptr;
    const long long nsites = (long long)A.L * A.L * A.L;
    auto write_series = [&](int pass) {                                // one thread of the cluster, a barrier after the atomics
        if (rank == 0 && threadIdx.x == 0) {
            int* a = &acc[pass & 1][0];
            if (R.M) R.M[(size_t)pass * A.R + r] = 2ll * a[0] - nsites;
            if (R.E) R.E[(size_t)pass * A.R + r] = 2ll * a[1] - 3ll * nsites;
            a[0] = 0; a[1] = 0;
        }
    };

    auto tile_of = [&](int C, uint32_t job) {
        uint32_t q = job * 4u + (uint32_t)sub;                        // colour-C tiles of the replica, (tz, ty, tx/2) row-major
        Tile3 t;
        t.r = r;
        t.tz = (int)(q / (B * hb)); q -= (uint32_t)t.tz * B * hb;
        t.ty = (int)(q / hb); q -= (uint32_t)t.ty * hb;
        t.tx = (int)(2u * q) + ((t.ty + t.tz + C) & 1);
        return t;
    };
    auto faces_of = [&](uint32_t tx, uint32_t ty, uint32_t tz) -> const uint8_t* {
        const uint32_t C = (tx + ty + tz) & 1u, q = (tz * B + ty) * hb + (tx >> 1);
        const uint32_t job = q >> 2, sb = q & 3u;                      // job < W: one job per warp and colour
        return cluster.map_shared_rank(&faces[C][job % kRes3Warps][sb][0], job / kRes3Warps);
    };
    struct Nb { const uint8_t *xm, *xp, *ym, *yp, *zm, *zp; };
    auto neighbours = [&](const Tile3& t) {
        const uint32_t tx = (uint32_t)t.tx, ty = (uint32_t)t.ty, tz = (uint32_t)t.tz;
        return Nb{faces_of(tx == 0 ? B - 1 : tx - 1, ty, tz), faces_of(tx == B - 1 ? 0 : tx + 1, ty, tz),
                  faces_of(tx, ty == 0 ? B - 1 : ty - 1, tz), faces_of(tx, ty == B - 1 ? 0 : ty + 1, tz),
                  faces_of(tx, ty, tz == 0 ? B - 1 : tz - 1), faces_of(tx, ty, tz == B - 1 ? 0 : tz + 1)};
    };
    auto publish = [&](int C, const Slice& s) {
        uint32_t XL, XR, YL, YR;
        face_words(s.S, lz, XL, XR, YL, YR);
        uint8_t* f = &faces[C][wic][sub][0];
        reinterpret_cast<uint32_t*>(f + kXL)[lz] = XL;
        reinterpret_cast<uint32_t*>(f + kXR)[lz] = XR;
        f[kYL + lz] = (uint8_t)YL;
        f[kYR + lz] = (uint8_t)YR;
        if (lz == 0) *reinterpret_cast<uint2*>(f + kZL) = make_uint2(s.S[0], s.S[1]);
        if (lz == 7) *reinterpret_cast<uint2*>(f + kZR) = make_uint2(s.S[0], s.S[1]);
    };
    auto refresh = [&](const Nb& nb, Slice& s) {
        s.x = reinterpret_cast<const uint32_t*>(nb.xm + kXR)[lz] | reinterpret_cast<const uint32_t*>(nb.xp + kXL)[lz];
        s.y = (uint32_t)nb.ym[kYR + lz] | ((uint32_t)nb.yp[kYL + lz] << 8);
        if (lz == 0) { const uint2 w = *reinterpret_cast<const uint2*>(nb.zm + kZR); s.zq[0] = w.x; s.zq[1] = w.y; }
        if (lz == 7) { const uint2 w = *reinterpret_cast<const uint2*>(nb.zp + kZL); s.zq[0] = w.x; s.zq[1] = w.y; }
    };

    const bool mine = wg < JC;
    Slice s[2];
    Tile3 t[2];
    Nb nb[2];
#pragma unroll
    for (int C = 0; C < 2; ++C)
        if (mine) {
            t[C] = tile_of(C, wg);
            nb[C] = neighbours(t[C]);
            load_slice<BITS>(A, t[C], lz, s[C]);
            load_couplings<HASJ>(A, t[C], lz, s[C]);
            publish(C, s[C]);
        }
    cluster.sync();

    const uint64_t seed = A.seeds[r];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int pass = 0; pass < R.n && R.plain; ++pass) {        // a8: fine colour 0 of every tile, barrier, fine colour 1, barrier
      for (int Cc = 0; Cc < (R.coarse ? 2 : 1); ++Cc)          // (masked double checkerboard: both coarse colours in turn)
        for (int j = 0; j < A.k; ++j) {
            const uint64_t tt = A.t_first + (uint64_t)pass * (uint64_t)A.k + (uint64_t)j;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                if (series && Cc == 0 && j == 0 && c == 1 && pass > 0) write_series(pass - 1);
#pragma unroll
                for (int C = 0; C < 2; ++C)
                    if (mine) {
                        refresh(nb[C], s[C]);
                        const uint32_t z = (uint32_t)(t[C].tz * kT3 + lz);
                        const uint32_t g = (z * B + (uint32_t)t[C].ty) * B + (uint32_t)t[C].tx;
                        const uint32_t p_base = (uint32_t)(t[C].tx * 4) + (uint32_t)(A.L >> 1) * ((uint32_t)(t[C].ty * kT3) + (uint32_t)A.L * z);
                        half_sweep3_masked<HASJ>(A, s[C], c, lz, g, p_base, 2 * tt + (uint64_t)c, k0, k1, coarse_mask3(R.coarse, t[C], lz, Cc));
                        publish(C, s[C]);
                    }
                cluster.sync();
            }
        }
        if (series) {
            int up = 0, unsat = 0;
            if (mine) {
                refresh(nb[0], s[0]);
                refresh(nb[1], s[1]);
                count_slice<HASJ>(s[0], lz, up, unsat);
                count_slice<HASJ>(s[1], lz, up, unsat);
            }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                up += __shfl_xor_sync(0xffffffffu, up, d);
                unsat += __shfl_xor_sync(0xffffffffu, unsat, d);
            }
            if (lane == 0 && mine) {
                atomicAdd(acc0 + 2 * (pass & 1), up);
                atomicAdd(acc0 + 2 * (pass & 1) + 1, unsat);
            }
        }
    }
    for (int pass = 0; pass < R.n && !R.plain; ++pass) {
#pragma unroll
        for (int C = 0; C < 2; ++C) {
            if (series && C == 1 && pass > 0) write_series(pass - 1);    // complete since the barrier just passed
            if (mine) {
                refresh(nb[C], s[C]);
                const uint32_t z = (uint32_t)(t[C].tz * kT3 + lz);
                const uint32_t g = (z * B + (uint32_t)t[C].ty) * B + (uint32_t)t[C].tx;
                const uint32_t p_base = (uint32_t)(t[C].tx * 4) + (uint32_t)(A.L >> 1) * ((uint32_t)(t[C].ty * kT3) + (uint32_t)A.L * z);
                for (int j = 0; j < A.k; ++j) {
                    const uint64_t tt = A.t_first + (uint64_t)pass * (uint64_t)A.k + (uint64_t)j;
                    half_sweep3<kNoSpec3, HASJ>(A, s[C], 0, lz, g, p_base, 2 * tt, k0, k1);
                    half_sweep3<kNoSpec3, HASJ>(A, s[C], 1, lz, g, p_base, 2 * tt + 1, k0, k1);
                }
                publish(C, s[C]);
            }
            cluster.sync();
        }
        if (series) {                       // as in k_resident_planes: count on the registers, sums to rank 0
            int up = 0, unsat = 0;
            if (mine) {
                refresh(nb[0], s[0]);       // the colour-0 tiles' halos are one phase old
                count_slice<HASJ>(s[0], lz, up, unsat);
                count_slice<HASJ>(s[1], lz, up, unsat);
            }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                up += __shfl_xor_sync(0xffffffffu, up, d);
                unsat += __shfl_xor_sync(0xffffffffu, unsat, d);
            }
            if (lane == 0 && mine) {
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
        if (mine) store_slice<BITS>(A, t[C], lz, s[C], lut);
    cluster.sync();            // no CTA leaves while its shared memory may still be read or added to
}

bool resident3d_supported(const ising_ctx* h, int T) {
    if (!tile3d_supported(h, T)) return false;
    const uint32_t B = (uint32_t)(h->L / kT3);
    return B * B * B / 2u / 4u <= (uint32_t)(kRes3MaxCluster * kRes3Warps) && (B * B * B / 2u) % 4u == 0;
}

int launch_resident3d(ising_ctx* h, const Accept& acc, bool bits, int n, int k, uint64_t t_first, long long* d_E, long long* d_M,
                      bool plain, int Tc) {
    Res3Args R;
    R.E = d_E; R.M = d_M;
    R.plain = plain ? 1 : 0;
    R.coarse = plain ? Tc : 0;
    Plane3Args& A = R.P;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_sweep_seeds;
    A.seed0 = h->shared_sweep ? h->sweep_seed : h->seeds[0];
    A.L = h->L; A.B = h->L / kT3; A.R = h->R; A.k = k; A.t_first = t_first; A.C = 0;
    A.njobs = 0; A.per_rep = A.per_z = A.hb = 0; A.magic_rep = A.magic_z = A.magic_hb = 0;
    for (int m = 0; m < 3; ++m) {
        for (int q = 0; q < kHeadBits; ++q) A.u[m][q] = ((acc.thr[m] >> (31 - q)) & 1u) ? 0xffffffffu : 0u;
        A.tail[m] = acc.thr[m] & ((1u << kTailBits) - 1u);
    }
    A.force = acc.thr_is_2p32[0] ? 0xffffffffu : 0u;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    R.n = n;
    const uint32_t B = (uint32_t)A.B;
    R.jobs_per_colour = B * B * B / 2u / 4u;
    const uint32_t want = (R.jobs_per_colour + kRes3Warps - 1) / kRes3Warps;
    unsigned cl = 1;
    while (cl < want && cl < (unsigned)kRes3MaxCluster) cl *= 2;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cl * (unsigned)h->R); cfg.blockDim = dim3(kRes3Warps * 32); cfg.dynamicSmemBytes = 0; cfg.stream = hooks().stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cl; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    auto go = [&](auto kernel) -> int {
        if (cl > 8) ISING_CUDA_OK(cudaFuncSetAttribute(kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, kernel, R));
        return 0;
    };
    const int rc = A.jrec ? (bits ? go(k_resident3d<true, true>) : go(k_resident3d<false, true>))
                          : (bits ? go(k_resident3d<true, false>) : go(k_resident3d<false, false>));
    if (rc) return rc;
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// ---- k_grid3d (grid3d_device.cuh): the whole call in one cooperative launch, slices on chip on all SMs ----
__global__ void k_grid3d_series_finish(const long long* __restrict__ acc, long long* __restrict__ E, long long* __restrict__ Mo,
                                       uint32_t count, long long nsites) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;          // pass * R + r
    if (i >= count) return;
    long long up = 0, unsat = 0;
    for (int s = 0; s < kGrid3AccSlots; ++s) { up += acc[((size_t)i * kGrid3AccSlots + s) * 2]; unsat += acc[((size_t)i * kGrid3AccSlots + s) * 2 + 1]; }
    if (Mo) Mo[i] = 2 * up - nsites;
    if (E) E[i] = 2 * unsat - 3 * nsites;
}

size_t grid3d_xedge_bytes(const ising_ctx* h) {
    const size_t B = (size_t)(h->L / kT3);
    return (size_t)h->R * B * B * B * kG3Rec * sizeof(unsigned long long);
}
size_t grid3d_acc_bytes(const ising_ctx* h, int n) { return (size_t)n * (size_t)h->R * kGrid3AccSlots * 2 * sizeof(long long); }

bool grid3d_supported(const ising_ctx* h, int T) {
    if (!tile3d_supported(h, T)) return false;
    const uint64_t B = (uint64_t)(h->L / kT3);
    return (uint64_t)h->R * B * B * B / 8u <= 148u * 32u * 16u;
}

namespace {
// One cooperative launch with M = 1 or 2 jobs of each colour per warp.  The run-time build (bits/hp3 given) is compiled
// for the CTA shape the lattice wants: ONE CTA per SM with ceil(warps / SMs) warps (rounding them up to a multiple of four gains nothing, measured), so
// that every SM and every scheduler carries the same number of jobs (config 4: 4096 jobs per colour = 28 warps on each
// SM, one job per warp, 72 registers).  Measured on config 4, k = 1 / 4 / 16: 5 CTAs of 4 warps with two jobs per warp
// 1684 / - / -; 4 CTAs of 7 warps 1917 / 2338 / 2382; 7 CTAs of 4 warps 1855 / 2201 / 2269; one CTA of 28 warps
// 1967 / 2713 / 3030 flips/ns.  The pre-compiled kernels keep their fixed shape (CTAs of up to 4 warps, 5 per SM).
template <bool BITS, bool HASJ>
int launch_grid3d_one(Grid3Args& R, bool want_jit, unsigned long long hp3, int reps, bool* fits, bool* used_jit) {
    int dev = 0, sms = 0;
    ISING_CUDA_OK(cudaGetDevice(&dev));
    ISING_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    *fits = false; *used_jit = false;
    static const uint32_t warp_cap = getenv("ISING_GRID_WARPS") ? (uint32_t)atoi(getenv("ISING_GRID_WARPS")) : 0u;   // testing aid
    static const uint32_t wsm_cap = getenv("ISING_G3_WSM") ? (uint32_t)atoi(getenv("ISING_G3_WSM")) : 28u;   // 28 warps: 72 registers each
    const uint32_t max_m = warp_cap ? 16u : 2u;              // as in launch_grid_planes: beyond two jobs per warp the per-pass kernels win
    for (uint32_t M = 1; M <= max_m; ++M) {
        const uint32_t warps_needed = (R.jobs_total + M - 1) / M;
        if (warp_cap && warps_needed > warp_cap && M < 16u) continue;
        const uint32_t w_sm = (warps_needed + (uint32_t)sms - 1) / (uint32_t)sms;
        int wpb, bps;
        const void* fn = nullptr;
        if (want_jit && !HASJ && w_sm <= wsm_cap) {
            wpb = (int)w_sm; bps = 1;         // one CTA per SM
            fn = (const void*)grid3d_jit_kernel(BITS, hp3, reps, wpb * 32, bps, R.acc != nullptr);
        }
        if (fn) *used_jit = true;
        else {
            fn = (const void*)k_grid3d<BITS, HASJ>;
            wpb = warps_needed <= (uint32_t)sms * 4u ? 1 : (warps_needed <= (uint32_t)sms * 8u ? 2 : 4);
            *used_jit = false;
        }
        ISING_CUDA_OK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        const size_t smem = (size_t)wpb * 2u * M * (size_t)kG3Slots * 32u * sizeof(uint32_t);    // words + constants of every job
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

// n passes in one cooperative launch; returns 1 (nothing launched) if the lattice does not fit on chip.
int launch_grid3d(ising_ctx* h, const Accept& acc, bool bits, int n, int k, uint64_t t_first, void* d_xedge, void* d_acc,
                  long long* d_E, long long* d_M, bool use_jit) {
    Grid3Args R;
    Plane3Args& A = R.P;
    A = Plane3Args{};
    fill_geometry3(A, h);
    fill_accept3(A, acc);
    A.k = k; A.t_first = t_first; A.C = 0;
    R.n = n;
    R.jobs_total = A.njobs;
    R.jobs_per_warp = 1;
    R.xedge = (unsigned long long*)d_xedge;
    const bool series = (d_E || d_M) && n > 0;
    R.acc = series ? (long long*)d_acc : nullptr;
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemsetAsync(d_xedge, 0, grid3d_xedge_bytes(h), st));          // version 0 = nothing published
    if (series) ISING_CUDA_OK(cudaMemsetAsync(d_acc, 0, grid3d_acc_bytes(h, n), st));
    const unsigned long long hp3 = ((unsigned long long)(acc.thr[0] >> kTailBits) << 24) |
                                   ((unsigned long long)(acc.thr[1] >> kTailBits) << 12) | (unsigned long long)(acc.thr[2] >> kTailBits);
    const bool want_jit = use_jit && !A.force && !A.jrec;
    bool fits = false, used_jit = false;
    int rc;
    if (A.jrec) rc = bits ? launch_grid3d_one<true, true>(R, false, hp3, h->R, &fits, &used_jit) : launch_grid3d_one<false, true>(R, false, hp3, h->R, &fits, &used_jit);
    else rc = bits ? launch_grid3d_one<true, false>(R, want_jit, hp3, h->R, &fits, &used_jit) : launch_grid3d_one<false, false>(R, want_jit, hp3, h->R, &fits, &used_jit);
    if (rc) return rc;
    if (!fits) return 1;
    h->last_jit = used_jit ? 1 : 0;
    if (series) {
        const uint32_t count = (uint32_t)n * (uint32_t)h->R;
        k_grid3d_series_finish<<<(count + 255) / 256, 256, 0, st>>>((const long long*)d_acc, d_E, d_M, count, (long long)h->N);
        count_launch();
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

}  // namespace ising
