// amsc.cu — asynchronous multi-spin coding for the 2D +-J model (DESIGN.md §3.6 R17, §6.5).
//
// Up to 32 disorder realisations are simulated at once: bit r of the 32-bit word at site i is the spin of
// realisation r, bit r of JX[i] / JY[i] says that realisation r's bond i -> i+e_x / i+e_y is J = -1.  A site is
// updated for all realisations with a dozen bitwise operations, and — the point of the method — with ONE random
// number r(i, H) (RNG mapping "words": one Philox4x32-10 output word per site, S8c.3), so the cost of the random
// numbers, which dominates everything else in this library, is shared 32 ways.  Each realisation is exactly an
// ordinary run of the oracle with its own couplings and the shared random stream (R17).
//
// Schedule: the double checkerboard of P:62-74 unchanged.  One CTA per tile: the tile, its halo and the bonds that
// touch it are staged in shared memory (coalesced row loads), k x {even sites, barrier, odd sites, barrier}, write
// back.  A thread owns 8 consecutive columns of one row, i.e. the 4 same-colour sites that share one Philox call.
#include "kernels.h"
#include "philox.cuh"

namespace ising {

namespace {

struct AmscArgs {
    uint32_t* spins;             // word lattice, site order i = x + L*y
    const uint32_t* jx;          // bond i -> i+e_x, bit r set <=> J = -1 for realisation r
    const uint32_t* jy;          // bond i -> i+e_y
    int L, B;
    int C;                       // coarse colour of this launch
    int k;
    uint64_t t_first;
    uint32_t k0, k1;             // the shared sweep key
    uint32_t thr1, thr2;         // thresholds for dE = 4, 8
    uint32_t all1, all2;         // all-ones if the threshold is 2^32 (beta = 0)
    uint32_t rmask;              // bits of the realisations in use
};

template <int T>
__global__ void __launch_bounds__(T * T / 8) k_amsc(AmscArgs A) {
    // Pitches chosen for the access pattern of the update (a warp = 32/(T/8) rows x T/8 column groups of 8): with the
    // spin pitch = 9 and the bond pitches = 1 (mod 32) the lanes of a warp hit distinct banks (T = 32).
    // (Measured: T = 32: 11920 -> 14350 flips/ns at k = 16; T = 64, where lanes g and g+4 collide whatever the pitch,
    // is faster with the plain pitches.)
    constexpr int P = T == 32 ? T + 9 : T + 2;     // pitch of the spin image, rows -1 .. T, columns -1 .. T
    constexpr int PY = T == 32 ? T + 1 : T;        // pitch of the JY image
    extern __shared__ uint32_t smem[];
    uint32_t* S = smem;                            // (T+2) rows of spin words
    uint32_t* JX = S + (T + 2) * P;                // column -1 .. T-1 of every tile row: JX[y][x+1], pitch T+1
    uint32_t* JY = JX + T * (T + 1);               // row -1 .. T-1: JY[y+1][x], pitch PY
    const int L = A.L, B = A.B;
    // colour-C tiles row by row: q -> ty = q / (B/2), tx = 2*(q % (B/2)) + ((ty + C) & 1)
    const int hb = B >> 1;
    const int ty = blockIdx.x / hb, tx = 2 * (blockIdx.x % hb) + ((ty + A.C) & 1);
    const int x0 = tx * T, y0 = ty * T;
    const int tid = threadIdx.x, nthr = T * T / 8;
    // a3: stage, row by row with 128-bit loads (no per-element wrap arithmetic): spin rows -1 .. T, bond rows, then the
    // two halo columns and the left rim of JX.
    constexpr int V = T / 4;                                          // 16-byte chunks per tile row
    for (int idx = tid; idx < (T + 2) * V; idx += nthr) {             // spins: rows -1 .. T
        const int rr = idx / V, v = idx - rr * V;
        int gy = y0 + rr - 1;
        gy = gy < 0 ? gy + L : (gy >= L ? gy - L : gy);
        const uint4 w = *reinterpret_cast<const uint4*>(A.spins + (size_t)gy * L + x0 + 4 * v);
        uint32_t* d = S + rr * P + 1 + 4 * v;
        d[0] = w.x; d[1] = w.y; d[2] = w.z; d[3] = w.w;
    }
    for (int idx = tid; idx < T * V; idx += nthr) {                   // JX: rows 0 .. T-1, columns 0 .. T-1
        const int rr = idx / V, v = idx - rr * V;
        const uint4 w = *reinterpret_cast<const uint4*>(A.jx + (size_t)(y0 + rr) * L + x0 + 4 * v);
        uint32_t* d = JX + rr * (T + 1) + 1 + 4 * v;
        d[0] = w.x; d[1] = w.y; d[2] = w.z; d[3] = w.w;
    }
    for (int idx = tid; idx < (T + 1) * V; idx += nthr) {             // JY: rows -1 .. T-1
        const int rr = idx / V, v = idx - rr * V;
        const int gy = y0 + rr - 1 < 0 ? y0 + rr - 1 + L : y0 + rr - 1;
        const uint4 w = *reinterpret_cast<const uint4*>(A.jy + (size_t)gy * L + x0 + 4 * v);
        uint32_t* d = JY + rr * PY + 4 * v;
        d[0] = w.x; d[1] = w.y; d[2] = w.z; d[3] = w.w;
    }
    {
        const int xl = x0 == 0 ? L - 1 : x0 - 1, xr = x0 + T == L ? 0 : x0 + T;
        for (int idx = tid; idx < 3 * T; idx += nthr) {                // halo columns x = -1, x = T; JX of column -1
            const int rr = idx % T, which = idx / T;
            const size_t row = (size_t)(y0 + rr) * L;
            if (which == 0) S[(rr + 1) * P] = A.spins[row + xl];
            else if (which == 1) S[(rr + 1) * P + T + 1] = A.spins[row + xr];
            else JX[rr * (T + 1)] = A.jx[row + xl];
        }
    }
    __syncthreads();
    const int y = tid / (T / 8), g = tid % (T / 8);                  // row and 8-column group of this thread
    // Philox group of the thread's 4 same-colour sites: p = i >> 1 = Y*(L/2) + X/2, group = p >> 2 (S8c.3)
    const uint32_t grp = (uint32_t)(((size_t)(y0 + y) * (L >> 1) + (x0 >> 1)) >> 2) + (uint32_t)g;
    for (int j = 0; j < A.k; ++j) {
        const uint64_t tt = A.t_first + (uint64_t)j;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const uint64_t H = 2 * tt + (uint64_t)c;
            const u32x4 rnd = philox4x32_10(grp, kTagSweep, (uint32_t)H, (uint32_t)(H >> 32), A.k0, A.k1);
            const uint32_t r4[4] = {rnd.x, rnd.y, rnd.z, rnd.w};
            const int par = (y + c) & 1;                               // y0 and x0 are even: local parity = global parity
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                const int x = 8 * g + 2 * m + par;
                const uint32_t s = S[(y + 1) * P + x + 1];
                const uint32_t a = s ^ S[y * P + x + 1] ^ JY[y * PY + x];               // up: bond (y-1) -> y
                const uint32_t b = s ^ S[(y + 2) * P + x + 1] ^ JY[(y + 1) * PY + x];   // down: bond y -> y+1
                const uint32_t cc = s ^ S[(y + 1) * P + x] ^ JX[y * (T + 1) + x];      // left: bond (x-1) -> x
                const uint32_t d = s ^ S[(y + 1) * P + x + 2] ^ JX[y * (T + 1) + x + 1];   // right
                const uint32_t p1 = a | b, q1 = a & b, p2 = cc | d, q2 = cc & d;
                const uint32_t ge1 = p1 | p2, ge2 = (p1 & p2) | q1 | q2;               // unsatisfied bonds >= 1, >= 2
                const uint32_t R1 = (r4[m] < A.thr1 ? 0xffffffffu : 0u) | A.all1;      // the same r for every realisation
                const uint32_t R2 = (r4[m] < A.thr2 ? 0xffffffffu : 0u) | A.all2;
                const uint32_t flip = (ge2 | (ge1 & R1) | R2) & A.rmask;               // dE <= 0, dE = 4, dE = 8 (eq. (2))
                S[(y + 1) * P + x + 1] = s ^ flip;
            }
            __syncthreads();
        }
    }
    // a7: write the interior back, 128-bit stores, coalesced rows
    for (int idx = tid; idx < T * V; idx += nthr) {
        const int rr = idx / V, v = idx - rr * V;
        const uint32_t* d = S + (rr + 1) * P + 1 + 4 * v;
        *reinterpret_cast<uint4*>(A.spins + (size_t)(y0 + rr) * L + x0 + 4 * v) = make_uint4(d[0], d[1], d[2], d[3]);
    }
}

// canonical int8 +-1 (R*N, realisation-major) <-> word lattice; couplings J[R][2][N] -> JX, JY words.
__global__ void k_amsc_pack(const int8_t* __restrict__ canon, uint32_t* __restrict__ words, uint64_t N, int R, int negative) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    uint32_t w = 0;
    for (int r = 0; r < R; ++r) {
        const int8_t v = canon[(uint64_t)r * N + i];
        w |= (uint32_t)(negative ? v < 0 : v > 0) << r;
    }
    words[i] = w;
}
__global__ void k_amsc_pack_J(const int8_t* __restrict__ J, uint32_t* __restrict__ jx, uint32_t* __restrict__ jy, uint64_t N, int R) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    uint32_t wx = 0, wy = 0;
    for (int r = 0; r < R; ++r) {
        wx |= (uint32_t)(J[((uint64_t)r * 2 + 0) * N + i] < 0) << r;
        wy |= (uint32_t)(J[((uint64_t)r * 2 + 1) * N + i] < 0) << r;
    }
    jx[i] = wx; jy[i] = wy;
}
__global__ void k_amsc_unpack(const uint32_t* __restrict__ words, int8_t* __restrict__ canon, uint64_t N, int R) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint32_t w = words[i];
    for (int r = 0; r < R; ++r) canon[(uint64_t)r * N + i] = ((w >> r) & 1u) ? 1 : -1;
}

}  // namespace

bool amsc_supported(const ising_ctx* h, int T) {
    if (h->dim != 2 || !h->J_per_replica || !h->shared_sweep || h->rng != ISING_RNG_WORDS || h->R > 32) return false;
    if (T != 32 && T != 64) return false;
    if (h->L % T) return false;
    const int B = h->L / T;
    return B >= 2 && (B % 2 == 0);
}

size_t amsc_spin_bytes(const ising_ctx* h) { return (size_t)h->N * 4; }

// J word lattices (2 * N words), built once per handle.
int launch_amsc_pack_J(ising_ctx* h, void* d_jwords) {
    uint32_t* jx = (uint32_t*)d_jwords;
    k_amsc_pack_J<<<(unsigned)((h->N + 255) / 256), 256, 0, hooks().stream>>>(h->d_J, jx, jx + h->N, h->N, h->R);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_canon_to_amsc(ising_ctx* h, const int8_t* d_canon, void* d_words) {
    k_amsc_pack<<<(unsigned)((h->N + 255) / 256), 256, 0, hooks().stream>>>(d_canon, (uint32_t*)d_words, h->N, h->R, 0);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_amsc_to_canon(ising_ctx* h, const void* d_words, int8_t* d_canon) {
    k_amsc_unpack<<<(unsigned)((h->N + 255) / 256), 256, 0, hooks().stream>>>((const uint32_t*)d_words, d_canon, h->N, h->R);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// a1: one outer pass = colour-0 launch, colour-1 launch, k inner sweeps each.
int launch_amsc_pass(ising_ctx* h, const Accept& acc, int T, int k, uint64_t t_first, const void* d_jwords) {
    AmscArgs A;
    A.spins = (uint32_t*)h->d_tiles;
    A.jx = (const uint32_t*)d_jwords;
    A.jy = A.jx + h->N;
    A.L = h->L; A.B = h->L / T; A.k = k; A.t_first = t_first;
    A.k0 = (uint32_t)h->sweep_seed; A.k1 = (uint32_t)(h->sweep_seed >> 32);
    A.thr1 = acc.thr[0]; A.thr2 = acc.thr[1];
    A.all1 = acc.thr_is_2p32[0] ? 0xffffffffu : 0u;
    A.all2 = acc.thr_is_2p32[1] ? 0xffffffffu : 0u;
    A.rmask = h->R >= 32 ? 0xffffffffu : ((1u << h->R) - 1u);
    const unsigned grid = (unsigned)(A.B * A.B / 2);
    const size_t smem = sizeof(uint32_t) * (size_t)((T + 2) * (T == 32 ? T + 9 : T + 2) + T * (T + 1) + (T + 1) * (T == 32 ? T + 1 : T));
    if (int rc = set_max_dynamic_smem<k_amsc<64>>(64 * 1024)) return rc;
    for (int C = 0; C < 2; ++C) {
        A.C = C;
        if (T == 64) k_amsc<64><<<grid, 64 * 64 / 8, smem, hooks().stream>>>(A);
        else k_amsc<32><<<grid, 32 * 32 / 8, smem, hooks().stream>>>(A);
        count_launch();
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

}  // namespace ising
