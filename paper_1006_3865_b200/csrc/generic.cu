// generic.cu — kernels on the canonical layout (int8 ±1, index order): hot start,
// observables, overlap, validation, and the global-memory sweep that serves every
// (dim, L, tile, couplings, replicas) combination the fast tile kernels do not.
//
// The generic sweep is the schedule of P:64-74 / S8c.6 issued as one launch per
// (coarse colour C, inner sweep j, fine colour c): all sites of fine colour c inside tiles
// of coarse colour C are independent, so one thread per site pair updates them in
// place from the live array.  With tile == L this is the single checkerboard of P:62 (a8).
#include <algorithm>

#include "kernels.h"
#include "philox.cuh"

namespace ising {

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ void key_of(uint64_t seed, uint32_t& k0, uint32_t& k1) {
    k0 = (uint32_t)(seed & 0xffffffffull);
    k1 = (uint32_t)(seed >> 32);
}

// a11 / S8c.3: s_i = (Philox(ctr = {i>>2, 1, 0, 0}, key = seed_r)[i & 3] >> 31) ? -1 : +1.
__global__ void k_hot_start(int8_t* __restrict__ s, const uint64_t* __restrict__ seeds,
                            uint64_t groups_per_replica, int R) {
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= groups_per_replica * (uint64_t)R) return;
    const uint64_t r = gid / groups_per_replica;
    const uint64_t g = gid - r * groups_per_replica;
    uint32_t k0, k1;
    key_of(seeds[r], k0, k1);
    const u32x4 o = philox4x32_10((uint32_t)g, kTagInit, 0u, 0u, k0, k1);
    char4 v;
    v.x = (o.x >> 31) ? -1 : 1;
    v.y = (o.y >> 31) ? -1 : 1;
    v.z = (o.z >> 31) ? -1 : 1;
    v.w = (o.w >> 31) ? -1 : 1;
    reinterpret_cast<char4*>(s)[r * groups_per_replica + g] = v;
}

// The same for lattices of N % 16 == 0 sites: four independent Philox calls per thread (16 sites), interleaved by the compiler,
// and one 16-byte store (the one-call kernel above spends 323 us on 2^28 sites, 60 % of its Philox bound).
__global__ void __launch_bounds__(256) k_hot_start16(int8_t* __restrict__ s, const uint64_t* __restrict__ seeds,
                                                     uint64_t quads_per_replica, int R) {
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= quads_per_replica * (uint64_t)R) return;
    const uint64_t r = gid / quads_per_replica;
    const uint64_t q = gid - r * quads_per_replica;
    uint32_t k0, k1;
    key_of(seeds[r], k0, k1);
    uint32_t w[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const u32x4 o = philox4x32_10((uint32_t)(4 * q + j), kTagInit, 0u, 0u, k0, k1);
        // byte i of the word: sign bit set -> 0xff (-1), else 0x01 (+1)
        const uint32_t neg = (o.x >> 31) | ((o.y >> 31) << 8) | ((o.z >> 31) << 16) | ((o.w >> 31) << 24);
        w[j] = (neg * 0xfeu) + 0x01010101u;                  // per byte: 1 + 0xfe = 0xff, 0 + 0x01 (no carries between bytes)
    }
    reinterpret_cast<uint4*>(s)[r * quads_per_replica + q] = make_uint4(w[0], w[1], w[2], w[3]);
}

struct GenericGeom {
    int dim, L, T, R;
    uint64_t N;
    uint64_t Jrep;     // distance between the coupling arrays of consecutive replicas: 0 (shared J) or dim*N (R17)
};

// One thread per site pair p = i >> 1 (S8c.3): the pair (2p, 2p+1) lies in one row because
// L is even and holds exactly one site of each fine colour.
__global__ void k_generic_halfsweep(int8_t* __restrict__ spins, const int8_t* __restrict__ J,
                                    const uint64_t* __restrict__ seeds, GenericGeom g,
                                    Accept acc, uint64_t H, int C, int c) {
    const uint64_t pairs = g.N >> 1;
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= pairs * (uint64_t)g.R) return;
    const uint64_t r = gid / pairs;
    const uint64_t p = gid - r * pairs;
    const uint64_t L = (uint64_t)g.L;
    const uint64_t i0 = p << 1;
    const int x0 = (int)(i0 % L);
    const int y = (int)((i0 / L) % L);
    const int z = (int)(i0 / (L * L));
    const int x = x0 + ((x0 + y + z + c) & 1);           // the site of fine colour c in the pair
    if ((((x / g.T) + (y / g.T) + (z / g.T)) & 1) != C) return;   // S8c.1 coarse colour
    const uint64_t i = i0 + (uint64_t)(x - x0);
    int8_t* s = spins + r * g.N;
    const int coord[3] = {x, y, z};
    uint64_t stride = 1;
    const int si = s[i];
    int n_sat = 0;                                       // satisfied bonds J s_i s_j = +1
    for (int d = 0; d < g.dim; ++d) {
        const uint64_t ip = (coord[d] == g.L - 1) ? i - (L - 1) * stride : i + stride;
        const uint64_t im = (coord[d] == 0) ? i + (L - 1) * stride : i - stride;
        const int Jp = J ? (int)J[r * g.Jrep + (uint64_t)d * g.N + i] : 1;
        const int Jm = J ? (int)J[r * g.Jrep + (uint64_t)d * g.N + im] : 1;
        n_sat += (Jp * si * s[ip] > 0) + (Jm * si * s[im] > 0);
        stride *= L;
    }
    const int a = 2 * n_sat - 2 * g.dim;                 // ΔE = 2a (S8c.5)
    bool flip = true;
    if (a > 0) {
        uint32_t k0, k1;
        key_of(seeds[r], k0, k1);
        const u32x4 o = philox4x32_10((uint32_t)(p >> 2), kTagSweep, (uint32_t)(H & 0xffffffffull),
                                      (uint32_t)(H >> 32), k0, k1);
        const uint32_t w = (uint32_t)(p & 3);
        const uint32_t rnd = w == 0 ? o.x : (w == 1 ? o.y : (w == 2 ? o.z : o.w));
        const int m = a / 2 - 1;
        flip = acc.thr_is_2p32[m] || (rnd < acc.thr[m]);
    }
    if (flip) s[i] = (int8_t)(-si);
}

// RNG mapping "planes" (DESIGN.md §3 R6): one thread per (replica, block g of 32 same-colour
// sites).  The 12 head planes of the block come from three Philox calls; the thread then
// walks its 32 bits.  The 20-bit tail of a site is drawn only when its head equals the head
// of the threshold it is compared with (probability 2^-12).
__global__ void k_generic_halfsweep_planes(int8_t* __restrict__ spins, const int8_t* __restrict__ J,
                                           const uint64_t* __restrict__ seeds, GenericGeom g,
                                           Accept acc, uint64_t H, int C, int c) {
    const int BW = (g.dim == 2) ? 16 : 4, BH = (g.dim == 2) ? 2 : 8;
    const int PW = g.L >> 1;
    const int GW = (PW + BW - 1) / BW, GH = (g.L + BH - 1) / BH;
    const int Lz = (g.dim == 3) ? g.L : 1;
    const uint64_t blocks = (uint64_t)GW * GH * Lz;
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= blocks * (uint64_t)g.R) return;
    const uint64_t r = gid / blocks;
    const uint32_t blk = (uint32_t)(gid - r * blocks);
    const int pb = (int)(blk % GW), yb = (int)((blk / GW) % GH), z = (int)(blk / ((uint32_t)GW * GH));
    uint32_t k0, k1;
    key_of(seeds[r], k0, k1);
    const uint32_t Hlo = (uint32_t)(H & 0xffffffffull), Hhi = (uint32_t)(H >> 32);
    uint32_t plane[kHeadBits];
#pragma unroll
    for (int n = 0; n < kHeadBits / 4; ++n) {
        const u32x4 o = philox4x32_10(blk, kTagPlanes + 256u * n, Hlo, Hhi, k0, k1);
        plane[4 * n] = o.x; plane[4 * n + 1] = o.y; plane[4 * n + 2] = o.z; plane[4 * n + 3] = o.w;
    }
    int8_t* s = spins + r * g.N;
    const uint64_t L = (uint64_t)g.L;
    for (int j = 0; j < 32; ++j) {
        const int y = yb * BH + j / BW, px = pb * BW + j % BW;
        if (y >= g.L || px >= PW) continue;
        const int x = 2 * px + ((y + z + c) & 1);
        if ((((x / g.T) + (y / g.T) + (z / g.T)) & 1) != C) continue;
        const uint64_t i = (uint64_t)x + L * ((uint64_t)y + L * (uint64_t)z);
        const int coord[3] = {x, y, z};
        uint64_t stride = 1;
        const int si = s[i];
        int n_sat = 0;
        for (int d = 0; d < g.dim; ++d) {
            const uint64_t ip = (coord[d] == g.L - 1) ? i - (L - 1) * stride : i + stride;
            const uint64_t im = (coord[d] == 0) ? i + (L - 1) * stride : i - stride;
            const int Jp = J ? (int)J[r * g.Jrep + (uint64_t)d * g.N + i] : 1;
            const int Jm = J ? (int)J[r * g.Jrep + (uint64_t)d * g.N + im] : 1;
            n_sat += (Jp * si * s[ip] > 0) + (Jm * si * s[im] > 0);
            stride *= L;
        }
        const int a = 2 * n_sat - 2 * g.dim;
        bool flip = true;
        if (a > 0) {
            const int m = a / 2 - 1;
            if (!acc.thr_is_2p32[m]) {
                uint32_t head = 0;
#pragma unroll
                for (int q = 0; q < kHeadBits; ++q) head |= ((plane[q] >> j) & 1u) << (kHeadBits - 1 - q);
                const uint32_t th = acc.thr[m] >> kTailBits;
                if (head != th) {
                    flip = head < th;
                } else {
                    const u32x4 o = philox4x32_10((uint32_t)(i >> 1), kTagTail, Hlo, Hhi, k0, k1);
                    flip = (o.x >> kHeadBits) < (acc.thr[m] & ((1u << kTailBits) - 1u));
                }
            }
        }
        if (flip) s[i] = (int8_t)(-si);
    }
}

__device__ __forceinline__ long long warp_sum(long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// a10 / S8c.7: E = -Σ_i Σ_d J_d(i) s_i s_(i+e_d), M = Σ_i s_i; blockIdx.y = replica.
__global__ void k_observables(const int8_t* __restrict__ spins, const int8_t* __restrict__ J,
                              GenericGeom g, long long* __restrict__ E, long long* __restrict__ M) {
    const int r = blockIdx.y;
    const int8_t* s = spins + (uint64_t)r * g.N;
    const uint64_t L = (uint64_t)g.L;
    long long e = 0, m = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < g.N;
         i += (uint64_t)gridDim.x * blockDim.x) {
        const int coord[3] = {(int)(i % L), (int)((i / L) % L), (int)(i / (L * L))};
        const int si = s[i];
        m += si;
        uint64_t stride = 1;
        for (int d = 0; d < g.dim; ++d) {
            const uint64_t ip = (coord[d] == g.L - 1) ? i - (L - 1) * stride : i + stride;
            const int Jp = J ? (int)J[(uint64_t)r * g.Jrep + (uint64_t)d * g.N + i] : 1;
            e -= Jp * si * s[ip];
            stride *= L;
        }
    }
    __shared__ long long sh[2][kThreads / 32];
    e = warp_sum(e);
    m = warp_sum(m);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) { sh[0][w] = e; sh[1][w] = m; }
    __syncthreads();
    if (w == 0) {
        e = lane < kThreads / 32 ? sh[0][lane] : 0;
        m = lane < kThreads / 32 ? sh[1][lane] : 0;
        e = warp_sum(e);
        m = warp_sum(m);
        if (lane == 0) {
            if (E) atomicAdd((unsigned long long*)&E[r], (unsigned long long)e);
            if (M) atomicAdd((unsigned long long*)&M[r], (unsigned long long)m);
        }
    }
}

__global__ void k_overlap(const int8_t* __restrict__ sa, const int8_t* __restrict__ sb, uint64_t N,
                          long long* __restrict__ Q) {
    long long q = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N;
         i += (uint64_t)gridDim.x * blockDim.x)
        q += (int)sa[i] * (int)sb[i];
    __shared__ long long sh[kThreads / 32];
    q = warp_sum(q);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) sh[w] = q;
    __syncthreads();
    if (w == 0) {
        q = lane < kThreads / 32 ? sh[lane] : 0;
        q = warp_sum(q);
        if (lane == 0) atomicAdd((unsigned long long*)Q, (unsigned long long)q);
    }
}

// every byte must be +1 (0x01) or -1 (0xff); 16 bytes per thread and step, the tail byte-wise
__global__ void k_validate_pm1(const int8_t* __restrict__ d, uint64_t n, int* flag) {
    const uint64_t n16 = n / 16;
    const uint4* v = reinterpret_cast<const uint4*>(d);
    bool bad = false;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint4 w = v[i];
        const uint32_t ok = (__vcmpeq4(w.x, 0x01010101u) | __vcmpeq4(w.x, 0xffffffffu)) & (__vcmpeq4(w.y, 0x01010101u) | __vcmpeq4(w.y, 0xffffffffu)) &
                            (__vcmpeq4(w.z, 0x01010101u) | __vcmpeq4(w.z, 0xffffffffu)) & (__vcmpeq4(w.w, 0x01010101u) | __vcmpeq4(w.w, 0xffffffffu));
        bad |= ok != 0xffffffffu;
    }
    if (blockIdx.x == 0)
        for (uint64_t i = 16 * n16 + threadIdx.x; i < n; i += blockDim.x) bad |= d[i] != 1 && d[i] != -1;
    if (bad) *flag = 1;
}

// canonical +-1 bytes <-> one bit per site (bit i & 31 of word i >> 5 set = spin up); one thread per word
__global__ void k_pack_bits(const int8_t* __restrict__ canon, uint32_t* __restrict__ words, uint64_t nwords) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nwords) return;
    const uint4* v = reinterpret_cast<const uint4*>(canon) + 2 * i;
    const uint4 a = v[0], b = v[1];
    const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    uint32_t out = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const uint32_t up = ~(w[q] >> 1) & 0x01010101u;          // 0x01 -> 1, 0xff -> 0, per byte
        out |= ((up * 0x01020408u) >> 24) << (4 * q);             // the four byte flags -> four adjacent bits
    }
    words[i] = out;
}

__global__ void k_unpack_bits(const uint32_t* __restrict__ words, int8_t* __restrict__ canon, uint64_t nwords) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nwords) return;
    const uint32_t in = words[i];
    uint32_t w[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const uint32_t up = (((in >> (4 * q)) & 0xfu) * 0x00204081u) & 0x01010101u;   // four bits -> four byte flags
        w[q] = ((up ^ 0x01010101u) * 255u) | up;                  // 1 -> 0x01, 0 -> 0xff
    }
    uint4* v = reinterpret_cast<uint4*>(canon) + 2 * i;
    v[0] = make_uint4(w[0], w[1], w[2], w[3]);
    v[1] = make_uint4(w[4], w[5], w[6], w[7]);
}

int reduce_grid(uint64_t n) {
    uint64_t b = (n + kThreads - 1) / kThreads;
    const uint64_t cap = 148ull * 16ull;
    return (int)(b < cap ? (b ? b : 1) : cap);
}

}  // namespace

int launch_hot_start(ising_ctx* h) {
    const uint64_t groups = h->N / 4;
    const uint64_t total = groups * (uint64_t)h->R;
    if (h->N % 16 == 0) {
        const uint64_t quads = h->N / 16;
        k_hot_start16<<<(unsigned)((quads * (uint64_t)h->R + 255) / 256), 256, 0, hooks().stream>>>(h->d_canon, h->d_seeds, quads, h->R);
    } else {
        const unsigned blocks = (unsigned)((total + kThreads - 1) / kThreads);
        k_hot_start<<<blocks, kThreads, 0, hooks().stream>>>(h->d_canon, h->d_seeds, groups, h->R);
    }
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_observables_canon(ising_ctx* h, const int8_t* d_spins, long long* d_E, long long* d_M) {
    cudaStream_t st = hooks().stream;
    if (d_E) ISING_CUDA_OK(cudaMemsetAsync(d_E, 0, sizeof(long long) * h->R, st));
    if (d_M) ISING_CUDA_OK(cudaMemsetAsync(d_M, 0, sizeof(long long) * h->R, st));
    GenericGeom g{h->dim, h->L, h->L, h->R, h->N, h->J_per_replica ? (uint64_t)h->dim * h->N : 0};
    dim3 grid(reduce_grid(h->N), h->R);
    k_observables<<<grid, kThreads, 0, st>>>(d_spins, h->d_J, g, d_E, d_M);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_overlap_canon(ising_ctx* h, const int8_t* d_spins, int a, int b, long long* d_Q) {
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemsetAsync(d_Q, 0, sizeof(long long), st));
    k_overlap<<<reduce_grid(h->N), kThreads, 0, st>>>(d_spins + (uint64_t)a * h->N,
                                                       d_spins + (uint64_t)b * h->N, h->N, d_Q);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// ---- all pairwise overlaps Q_ab = sum_i s_i^a s_i^b (S8c.7; BASELINE config 5: "pairwise overlap q") in one pass
// over the spins wherever they live.  A replica is a sequence of chunks (tile records, or the whole canonical array) of
// which the first chunk_words 32-bit words hold spins: one bit per site, a 0/1 byte per site, or a +-1 byte per site; in
// every encoding popc(word_a ^ word_b) = bits_per_diff x (number of sites of the word in which a and b differ), and
// Q_ab = N - 2 #differing.  Block row a (blockIdx.y) compares replica a with the replicas b > a, eight at a time: D[a*R+b].
constexpr int kPairChunk = 8;

__global__ void __launch_bounds__(kThreads) k_overlap_all(const uint32_t* __restrict__ base, uint64_t rep_stride_words, uint64_t n_chunks,
                                                          uint64_t chunk_stride_words, uint64_t chunk_words, int R,
                                                          unsigned long long* __restrict__ D) {
    const int a = blockIdx.y;
    const uint64_t total = n_chunks * (uint64_t)chunk_words;
    __shared__ unsigned long long sh[kThreads / 32][kPairChunk];
    for (int b0 = a + 1; b0 < R; b0 += kPairChunk) {
        unsigned long long acc[kPairChunk];
#pragma unroll
        for (int j = 0; j < kPairChunk; ++j) acc[j] = 0;
        for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
            uint64_t off = i;
            if (n_chunks > 1) {                          // tile records: chunk sizes fit 32 bits
                const uint32_t cw = (uint32_t)chunk_words;
                const uint64_t ch = i / cw;
                off = ch * chunk_stride_words + (i - ch * cw);
            }
            const uint32_t wa = __ldg(base + (uint64_t)a * rep_stride_words + off);
#pragma unroll
            for (int j = 0; j < kPairChunk; ++j)
                if (b0 + j < R) acc[j] += (unsigned)__popc(wa ^ __ldg(base + (uint64_t)(b0 + j) * rep_stride_words + off));
        }
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
        for (int j = 0; j < kPairChunk; ++j) {
            unsigned long long v = acc[j];
            for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
            if (lane == 0) sh[w][j] = v;
        }
        __syncthreads();
        if (threadIdx.x < kPairChunk && b0 + (int)threadIdx.x < R) {
            unsigned long long v = 0;
            for (int ww = 0; ww < kThreads / 32; ++ww) v += sh[ww][threadIdx.x];
            atomicAdd(D + (size_t)a * R + (b0 + threadIdx.x), v);
        }
        __syncthreads();
    }
}

__global__ void k_overlap_finish(const unsigned long long* __restrict__ D, long long* __restrict__ Q, int R, long long nsites, int bits_per_diff) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= R * R) return;
    const int a = i / R, b = i - a * R;
    if (a == b) { Q[i] = nsites; return; }
    const unsigned long long d = a < b ? D[(size_t)a * R + b] : D[(size_t)b * R + a];
    Q[i] = nsites - 2ll * (long long)(d / (unsigned)bits_per_diff);
}

// d_D: R*R zeroed-by-us scratch words, d_Q: R*R results (both device)
int launch_overlap_all(ising_ctx* h, const void* base, uint64_t rep_stride_bytes, uint64_t n_chunks, uint64_t chunk_stride_bytes,
                       uint64_t chunk_bytes, int bits_per_diff, unsigned long long* d_D, long long* d_Q) {
    cudaStream_t st = hooks().stream;
    const int R = h->R;
    ISING_CUDA_OK(cudaMemsetAsync(d_D, 0, sizeof(unsigned long long) * (size_t)R * R, st));
    if (R > 1) {
        const uint64_t total = n_chunks * (uint64_t)(chunk_bytes / 4);
        unsigned gx = (unsigned)std::min<uint64_t>((total + kThreads - 1) / kThreads, 148u * 8u);
        if (gx < 1) gx = 1;
        k_overlap_all<<<dim3(gx, (unsigned)(R - 1)), kThreads, 0, st>>>((const uint32_t*)base, rep_stride_bytes / 4, n_chunks, chunk_stride_bytes / 4,
                                                                       chunk_bytes / 4, R, d_D);
        count_launch();
    }
    k_overlap_finish<<<(R * R + 255) / 256, 256, 0, st>>>(d_D, d_Q, R, (long long)h->N, bits_per_diff);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_validate_pm1(const int8_t* d, uint64_t n, int* d_flag, int* host_bad) {
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemsetAsync(d_flag, 0, sizeof(int), st));
    k_validate_pm1<<<reduce_grid(n), kThreads, 0, st>>>(d, n, d_flag);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    ISING_CUDA_OK(cudaMemcpyAsync(host_bad, d_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
    ISING_CUDA_OK(cudaStreamSynchronize(st));
    return 0;
}

int launch_pack_bits(const int8_t* d_canon, uint32_t* d_words, uint64_t nwords) {
    k_pack_bits<<<(unsigned)((nwords + kThreads - 1) / kThreads), kThreads, 0, hooks().stream>>>(d_canon, d_words, nwords);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_unpack_bits(const uint32_t* d_words, int8_t* d_canon, uint64_t nwords) {
    k_unpack_bits<<<(unsigned)((nwords + kThreads - 1) / kThreads), kThreads, 0, hooks().stream>>>(d_words, d_canon, nwords);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// a1/a6/a8: the whole S8c.6 schedule, one launch per (C, j, c); optional E/M after each pass.
int launch_generic_sweep(ising_ctx* h, const Accept& acc, int n, int T, int k, long long* d_E,
                         long long* d_M) {
    cudaStream_t st = hooks().stream;
    GenericGeom g{h->dim, h->L, T, h->R, h->N, h->J_per_replica ? (uint64_t)h->dim * h->N : 0};
    const uint64_t total = (h->N >> 1) * (uint64_t)h->R;
    const unsigned blocks = (unsigned)((total + kThreads - 1) / kThreads);
    const int BW = (h->dim == 2) ? 16 : 4, BH = (h->dim == 2) ? 2 : 8;
    const uint64_t nblk = (uint64_t)(((h->L >> 1) + BW - 1) / BW) * ((h->L + BH - 1) / BH) *
                          (h->dim == 3 ? h->L : 1) * (uint64_t)h->R;
    const unsigned pblocks = (unsigned)((nblk + kThreads - 1) / kThreads);
    const int ncol = (T == h->L) ? 1 : 2;   // one tile: the odd coarse phase is empty
    for (int pass = 0; pass < n; ++pass) {
        for (int C = 0; C < ncol; ++C)
            for (int j = 0; j < k; ++j) {
                const uint64_t t = h->t + (uint64_t)pass * (uint64_t)k + (uint64_t)j;
                for (int c = 0; c < 2; ++c) {
                    if (h->rng == ISING_RNG_PLANES)
                        k_generic_halfsweep_planes<<<pblocks, kThreads, 0, st>>>(h->d_canon, h->d_J, h->d_sweep_seeds,
                                                                                 g, acc, 2 * t + c, C, c);
                    else
                        k_generic_halfsweep<<<blocks, kThreads, 0, st>>>(h->d_canon, h->d_J, h->d_sweep_seeds,
                                                                         g, acc, 2 * t + c, C, c);
                    count_launch();
                }
            }
        if (d_E || d_M) {
            const int rc = launch_observables_canon(h, h->d_canon,
                                                    d_E ? d_E + (size_t)pass * h->R : nullptr,
                                                    d_M ? d_M + (size_t)pass * h->R : nullptr);
            if (rc) return rc;
        }
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

}  // namespace ising
