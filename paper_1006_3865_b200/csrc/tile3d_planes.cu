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
#include "kernels.h"
#include "tile3d_planes_device.cuh"

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

}  // namespace

bool tile3d_supported(const ising_ctx* h, int T) {
    if (h->dim != 3 || h->has_J || T != kT3 || h->L % kT3) return false;
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
    const int warps = kThreads3 / 32;
    const uint32_t grid = (A.njobs + warps - 1) / warps;
    // specialised on the three threshold heads (planes_jit.cu) when asked for and available
    const unsigned long long hp3 = ((unsigned long long)(acc.thr[0] >> kTailBits) << 24) |
                                   ((unsigned long long)(acc.thr[1] >> kTailBits) << 12) | (unsigned long long)(acc.thr[2] >> kTailBits);
    cudaKernel_t spec = (use_jit && !A.force) ? planes3d_jit_kernel(bits, hp3) : nullptr;
    h->last_jit = spec ? 1 : 0;
    for (int C = 0; C < 2; ++C) {
        A.C = C;
        if (spec) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(grid); cfg.blockDim = dim3(warps * 32); cfg.stream = hooks().stream;
            void* args[] = {&A};
            ISING_CUDA_OK(cudaLaunchKernelExC(&cfg, (const void*)spec, args));
        } else if (bits) {
            k_tile3d_planes<true><<<grid, warps * 32, 0, hooks().stream>>>(A);
        } else {
            k_tile3d_planes<false><<<grid, warps * 32, 0, hooks().stream>>>(A);
        }
        count_launch();
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

}  // namespace ising
