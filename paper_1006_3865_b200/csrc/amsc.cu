// amsc.cu — asynchronous multi-spin coding for the 2D +-J model (DESIGN.md §3.6 R17, §6.5).
//
// 32 disorder realisations are simulated per word lattice (and up to 256 per handle, as several lattices driven by the same
// random numbers): bit r & 31 of the 32-bit word at site i is the spin of realisation r, bit r of JX[i] / JY[i] says that realisation r's bond i -> i+e_x / i+e_y is J = -1.  A site is
// updated for all realisations with a dozen bitwise operations, and — the point of the method — with ONE random
// number r(i, H) (RNG mapping "words": one Philox4x32-10 output word per site, S8c.3), so the cost of the random
// numbers, which dominates everything else in this library, is shared 32 ways (per lattice).  Each realisation is exactly an
// ordinary run of the oracle with its own couplings and the shared random stream (R17).
//
// Schedule: the double checkerboard of P:62-74 unchanged.  One CTA per tile: the tile, its halo and the bonds that
// touch it are staged in shared memory (coalesced row loads), k x {even sites, barrier, odd sites, barrier}, write
// back.  A thread owns 8 consecutive columns of one row, i.e. the 4 same-colour sites that share one Philox call.
#include "kernels.h"
#include "philox.cuh"

namespace ising {

namespace {

template <class W>
struct AmscArgs {
    W* spins;                    // word lattice, site order i = x + L*y
    const W* jx;                 // bond i -> i+e_x, bit r set <=> J = -1 for realisation r
    const W* jy;                 // bond i -> i+e_y
    int L, B;
    int C;                       // coarse colour of this launch
    int k;
    uint64_t t_first;
    uint32_t k0, k1;             // the shared sweep key
    uint32_t thr1, thr2;         // thresholds for dE = 4, 8
    uint32_t all1, all2;         // all-ones if the threshold is 2^32 (beta = 0)
    W rmask;                     // bits of the realisations in use
};

template <int T, class W>
__global__ void __launch_bounds__(T * T / 8) k_amsc(AmscArgs<W> A) {
    // Pitches chosen for the access pattern of the update (a warp = 32/(T/8) rows x T/8 column groups of 8): with the
    // spin pitch = 9 and the bond pitches = 1 (mod 32) the lanes of a warp hit distinct banks (T = 32).
    // (Measured: T = 32: 11920 -> 14350 flips/ns at k = 16; T = 64, where lanes g and g+4 collide whatever the pitch,
    // is faster with the plain pitches.)
    constexpr int P = T == 32 ? T + 9 : T + 2;     // pitch of the spin image, rows -1 .. T, columns -1 .. T
    constexpr int PY = T == 32 ? T + 1 : T;        // pitch of the JY image
    extern __shared__ __align__(16) unsigned char smem_raw[];
    W* S = reinterpret_cast<W*>(smem_raw);         // (T+2) rows of spin words
    W* JX = S + (T + 2) * P;                       // column -1 .. T-1 of every tile row: JX[y][x+1], pitch T+1
    W* JY = JX + T * (T + 1);                      // row -1 .. T-1: JY[y+1][x], pitch PY
    constexpr int WPC = 16 / (int)sizeof(W);       // words per 16-byte chunk
    const int L = A.L, B = A.B;
    // colour-C tiles row by row: q -> ty = q / (B/2), tx = 2*(q % (B/2)) + ((ty + C) & 1)
    const int hb = B >> 1;
    const int ty = blockIdx.x / hb, tx = 2 * (blockIdx.x % hb) + ((ty + A.C) & 1);
    const int x0 = tx * T, y0 = ty * T;
    const int tid = threadIdx.x, nthr = T * T / 8;
    // a3: stage, row by row with 128-bit loads (no per-element wrap arithmetic): spin rows -1 .. T, bond rows, then the
    // two halo columns and the left rim of JX.
    constexpr int V = T / WPC;                                        // 16-byte chunks per tile row
    auto put = [](W* d, const uint4& w) {                             // one chunk into (unaligned) shared memory, word by word
        if (sizeof(W) == 4) { d[0] = (W)w.x; d[1] = (W)w.y; d[2] = (W)w.z; d[3] = (W)w.w; }
        else { d[0] = (W)(((unsigned long long)w.y << 32) | w.x); d[1] = (W)(((unsigned long long)w.w << 32) | w.z); }
    };
    for (int idx = tid; idx < (T + 2) * V; idx += nthr) {             // spins: rows -1 .. T
        const int rr = idx / V, v = idx - rr * V;
        int gy = y0 + rr - 1;
        gy = gy < 0 ? gy + L : (gy >= L ? gy - L : gy);
        put(S + rr * P + 1 + WPC * v, *reinterpret_cast<const uint4*>(A.spins + (size_t)gy * L + x0 + WPC * v));
    }
    for (int idx = tid; idx < T * V; idx += nthr) {                   // JX: rows 0 .. T-1, columns 0 .. T-1
        const int rr = idx / V, v = idx - rr * V;
        put(JX + rr * (T + 1) + 1 + WPC * v, *reinterpret_cast<const uint4*>(A.jx + (size_t)(y0 + rr) * L + x0 + WPC * v));
    }
    for (int idx = tid; idx < (T + 1) * V; idx += nthr) {             // JY: rows -1 .. T-1
        const int rr = idx / V, v = idx - rr * V;
        const int gy = y0 + rr - 1 < 0 ? y0 + rr - 1 + L : y0 + rr - 1;
        put(JY + rr * PY + WPC * v, *reinterpret_cast<const uint4*>(A.jy + (size_t)gy * L + x0 + WPC * v));
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
                const W s = S[(y + 1) * P + x + 1];
                const W a = s ^ S[y * P + x + 1] ^ JY[y * PY + x];               // up: bond (y-1) -> y
                const W b = s ^ S[(y + 2) * P + x + 1] ^ JY[(y + 1) * PY + x];   // down: bond y -> y+1
                const W cc = s ^ S[(y + 1) * P + x] ^ JX[y * (T + 1) + x];      // left: bond (x-1) -> x
                const W d = s ^ S[(y + 1) * P + x + 2] ^ JX[y * (T + 1) + x + 1];   // right
                const W p1 = a | b, q1 = a & b, p2 = cc | d, q2 = cc & d;
                const W ge1 = p1 | p2, ge2 = (p1 & p2) | q1 | q2;               // unsatisfied bonds >= 1, >= 2
                const W R1 = (r4[m] < A.thr1 || A.all1) ? ~(W)0 : (W)0;          // the same r for every realisation
                const W R2 = (r4[m] < A.thr2 || A.all2) ? ~(W)0 : (W)0;
                const W flip = (ge2 | (ge1 & R1) | R2) & A.rmask;               // dE <= 0, dE = 4, dE = 8 (eq. (2))
                S[(y + 1) * P + x + 1] = s ^ flip;
            }
            __syncthreads();
        }
    }
    // a7: write the interior back, 128-bit stores, coalesced rows
    for (int idx = tid; idx < T * V; idx += nthr) {
        const int rr = idx / V, v = idx - rr * V;
        const W* d = S + (rr + 1) * P + 1 + WPC * v;
        uint4 w;
        if (sizeof(W) == 4) w = make_uint4((uint32_t)d[0], (uint32_t)d[1], (uint32_t)d[2], (uint32_t)d[3]);
        else w = make_uint4((uint32_t)d[0], (uint32_t)((unsigned long long)d[0] >> 32), (uint32_t)d[1], (uint32_t)((unsigned long long)d[1] >> 32));
        *reinterpret_cast<uint4*>(A.spins + (size_t)(y0 + rr) * L + x0 + WPC * v) = w;
    }
}

// ---- 3D (the Edwards-Anderson glass of P:100): 8^3 tiles, one CTA of 64 threads per tile.  Thread (z, y) owns the row of 8
// sites x = 0..7 = the 4 same-colour sites that share one Philox call (group i >> 3).  Six neighbours, three thresholds.
template <class W>
struct Amsc3Args {
    W* spins;                    // i = x + L*(y + L*z)
    const W* jw;                 // jw[d*N + i]: bond i -> i + e_d
    int L, B, C, k;
    uint64_t t_first;
    uint32_t k0, k1;
    uint32_t thr[3], all[3];
    W rmask;
};

template <class W>
__global__ void __launch_bounds__(64) k_amsc3d(Amsc3Args<W> A) {
    constexpr int T = 8, P = T + 2 + 1;                      // x pitch of the spin image (odd: fewer bank conflicts)
    __shared__ W S[T + 2][T + 2][P];                         // [z+1][y+1][x+1]
    __shared__ W JXs[T][T][T + 1];                           // bond (x-1) -> x at [z][y][x], x = 0..8 -> index x
    __shared__ W JYs[T][T + 1][T];                           // bond (y-1) -> y at [z][y][x]
    __shared__ W JZs[T + 1][T][T];                           // bond (z-1) -> z at [z][y][x]
    const int L = A.L, B = A.B, hb = B >> 1;
    // colour-C tiles enumerated (tz, ty, tx/2): tx = 2 * txh + ((ty + tz + C) & 1)
    int q = blockIdx.x;
    const int tz = q / (B * hb); q -= tz * B * hb;
    const int ty = q / hb; q -= ty * hb;
    const int tx = 2 * q + ((ty + tz + A.C) & 1);
    const int x0 = tx * T, y0 = ty * T, z0 = tz * T;
    const int tid = threadIdx.x;
    const size_t N = (size_t)L * L * L;
    auto wrap = [L](int v) { return v < 0 ? v + L : (v >= L ? v - L : v); };
    auto site = [L](int x, int y, int z) { return (size_t)x + (size_t)L * ((size_t)y + (size_t)L * (size_t)z); };
    for (int idx = tid; idx < (T + 2) * (T + 2) * (T + 2); idx += 64) {      // spins with halo (corners unused but harmless)
        const int xx = idx % (T + 2), yy = (idx / (T + 2)) % (T + 2), zz = idx / ((T + 2) * (T + 2));
        S[zz][yy][xx] = A.spins[site(wrap(x0 + xx - 1), wrap(y0 + yy - 1), wrap(z0 + zz - 1))];
    }
    for (int idx = tid; idx < T * T * (T + 1); idx += 64) {
        const int a = idx % (T + 1), b = (idx / (T + 1)) % T, c = idx / ((T + 1) * T);          // a runs over the long axis
        JXs[c][b][a] = A.jw[0 * N + site(wrap(x0 + a - 1), y0 + b, z0 + c)];
        JYs[c][a][b] = A.jw[1 * N + site(x0 + b, wrap(y0 + a - 1), z0 + c)];
        JZs[a][c][b] = A.jw[2 * N + site(x0 + b, y0 + c, wrap(z0 + a - 1))];
    }
    __syncthreads();
    const int z = tid >> 3, y = tid & 7;
    const uint32_t grp = (uint32_t)(site(x0, y0 + y, z0 + z) >> 3);
    for (int j = 0; j < A.k; ++j) {
        const uint64_t tt = A.t_first + (uint64_t)j;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const uint64_t H = 2 * tt + (uint64_t)c;
            const u32x4 rnd = philox4x32_10(grp, kTagSweep, (uint32_t)H, (uint32_t)(H >> 32), A.k0, A.k1);
            const uint32_t r4[4] = {rnd.x, rnd.y, rnd.z, rnd.w};
            const int par = (y + z + c) & 1;
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                const int x = 2 * m + par;
                const W s = S[z + 1][y + 1][x + 1];
                const W a = s ^ S[z][y + 1][x + 1] ^ JZs[z][y][x], b = s ^ S[z + 2][y + 1][x + 1] ^ JZs[z + 1][y][x];
                const W e = s ^ S[z + 1][y][x + 1] ^ JYs[z][y][x], f = s ^ S[z + 1][y + 2][x + 1] ^ JYs[z][y + 1][x];
                const W u = s ^ S[z + 1][y + 1][x] ^ JXs[z][y][x], v = s ^ S[z + 1][y + 1][x + 2] ^ JXs[z][y][x + 1];
                const W p1 = a | b, q1 = a & b, p2 = e | f, q2 = e & f, p3 = u | v, q3 = u & v;
                const W ge1 = p1 | p2 | p3;
                const W ge2 = q1 | q2 | q3 | (p1 & p2) | (p1 & p3) | (p2 & p3);
                const W ge3 = (q1 & (p2 | p3)) | (q2 & (p1 | p3)) | (q3 & (p1 | p2)) | (p1 & p2 & p3);      // dE <= 0
                const W R1 = (r4[m] < A.thr[0] || A.all[0]) ? ~(W)0 : (W)0;      // dE = 4: two unsatisfied bonds
                const W R2 = (r4[m] < A.thr[1] || A.all[1]) ? ~(W)0 : (W)0;      // dE = 8: one
                const W R3 = (r4[m] < A.thr[2] || A.all[2]) ? ~(W)0 : (W)0;      // dE = 12: none
                const W flip = (ge3 | (ge2 & R1) | (ge1 & R2) | R3) & A.rmask;
                S[z + 1][y + 1][x + 1] = s ^ flip;
            }
            __syncthreads();
        }
    }
    for (int x = 0; x < T; ++x) A.spins[site(x0 + x, y0 + y, z0 + z)] = S[z + 1][y + 1][x + 1];
}

// canonical int8 +-1 (R*N, realisation-major) <-> word lattice; couplings J[R][2][N] -> JX, JY words.
// Realisations are packed 32 to a word lattice ("half" h = realisations 32h .. 32h+31): words[h*N + i], bond words
// jw[(h*dim + d)*N + i].  (The kernels are templates on the word type, but only uint32_t is instantiated: with 64-bit words the
// 2D kernel, which is bound by shared memory, ran at 7560 instead of 14350 flips/ns at L = 4096, k = 16, so more than 32
// realisations are swept as several 32-bit lattices with the same random numbers — the same trajectories.)
__global__ void k_amsc_pack(const int8_t* __restrict__ canon, uint32_t* __restrict__ words, uint64_t N, int R) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    for (int h = 0; 32 * h < R; ++h) {
        uint32_t w = 0;
        for (int r = 32 * h; r < R && r < 32 * h + 32; ++r) w |= (uint32_t)(canon[(uint64_t)r * N + i] > 0) << (r & 31);
        words[(uint64_t)h * N + i] = w;
    }
}
__global__ void k_amsc_pack_J(const int8_t* __restrict__ J, uint32_t* __restrict__ jw, uint64_t N, int R, int dim) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    for (int h = 0; 32 * h < R; ++h)
        for (int d = 0; d < dim; ++d) {
            uint32_t w = 0;
            for (int r = 32 * h; r < R && r < 32 * h + 32; ++r) w |= (uint32_t)(J[((uint64_t)r * dim + d) * N + i] < 0) << (r & 31);
            jw[((uint64_t)h * dim + d) * N + i] = w;
        }
}
__global__ void k_amsc_unpack(const uint32_t* __restrict__ words, int8_t* __restrict__ canon, uint64_t N, int R) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    for (int h = 0; 32 * h < R; ++h) {
        const uint32_t w = words[(uint64_t)h * N + i];
        for (int r = 32 * h; r < R && r < 32 * h + 32; ++r) canon[(uint64_t)r * N + i] = ((w >> (r & 31)) & 1u) ? 1 : -1;
    }
}

}  // namespace

constexpr int kAmscMaxR = 256;
static int amsc_halves(const ising_ctx* h) { return (h->R + 31) / 32; }

bool amsc_supported(const ising_ctx* h, int T) {
    if (!h->J_per_replica || !h->shared_sweep || h->rng != ISING_RNG_WORDS || h->R > kAmscMaxR) return false;
    if (h->dim == 3) return amsc3d_supported(h, T);
    if (h->dim != 2) return false;
    if (T != 32 && T != 64) return false;
    if (h->L % T) return false;
    const int B = h->L / T;
    return B >= 2 && (B % 2 == 0);
}

bool amsc3d_supported(const ising_ctx* h, int T) {
    if (h->dim != 3 || T != 8 || h->L % 8) return false;
    const int B = h->L / 8;
    return B >= 2 && (B % 2 == 0);
}

size_t amsc_spin_bytes(const ising_ctx* h) { return (size_t)amsc_halves(h) * h->N * 4; }
size_t amsc_bond_bytes(const ising_ctx* h) { return (size_t)h->dim * amsc_spin_bytes(h); }

// J word lattices, built once per handle.
int launch_amsc_pack_J(ising_ctx* h, void* d_jwords) {
    k_amsc_pack_J<<<(unsigned)((h->N + 255) / 256), 256, 0, hooks().stream>>>(h->d_J, (uint32_t*)d_jwords, h->N, h->R, h->dim);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_canon_to_amsc(ising_ctx* h, const int8_t* d_canon, void* d_words) {
    k_amsc_pack<<<(unsigned)((h->N + 255) / 256), 256, 0, hooks().stream>>>(d_canon, (uint32_t*)d_words, h->N, h->R);
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

static uint32_t half_mask(const ising_ctx* h, int half) {
    const int left = h->R - 32 * half;
    return left >= 32 ? 0xffffffffu : ((1u << left) - 1u);
}

// a1: one outer pass = colour-0 launch, colour-1 launch (per 32 realisations), k inner sweeps each.
int launch_amsc_pass(ising_ctx* h, const Accept& acc, int T, int k, uint64_t t_first, const void* d_jwords) {
    typedef uint32_t W;
    const uint32_t k0 = (uint32_t)h->sweep_seed, k1 = (uint32_t)(h->sweep_seed >> 32);
    if (h->dim == 3) {
        const int B = h->L / 8;
        for (int C = 0; C < 2; ++C)
            for (int half = 0; half < amsc_halves(h); ++half) {
                Amsc3Args<W> A;
                A.spins = (W*)h->d_tiles + (size_t)half * h->N;
                A.jw = (const W*)d_jwords + (size_t)half * 3 * h->N;
                A.L = h->L; A.B = B; A.C = C; A.k = k; A.t_first = t_first; A.k0 = k0; A.k1 = k1;
                for (int m = 0; m < 3; ++m) { A.thr[m] = acc.thr[m]; A.all[m] = acc.thr_is_2p32[m] ? 1u : 0u; }
                A.rmask = half_mask(h, half);
                k_amsc3d<W><<<(unsigned)(B * B * B / 2), 64, 0, hooks().stream>>>(A);
                count_launch();
            }
        ISING_CUDA_OK(cudaGetLastError());
        return 0;
    }
    const int B = h->L / T;
    const size_t smem = sizeof(W) * (size_t)((T + 2) * (T == 32 ? T + 9 : T + 2) + T * (T + 1) + (T + 1) * (T == 32 ? T + 1 : T));
    if (int rc = set_max_dynamic_smem<k_amsc<64, W>>(64 * 1024)) return rc;
    for (int C = 0; C < 2; ++C)
        for (int half = 0; half < amsc_halves(h); ++half) {
            AmscArgs<W> A;
            A.spins = (W*)h->d_tiles + (size_t)half * h->N;
            A.jx = (const W*)d_jwords + (size_t)half * 2 * h->N;
            A.jy = A.jx + h->N;
            A.L = h->L; A.B = B; A.C = C; A.k = k; A.t_first = t_first; A.k0 = k0; A.k1 = k1;
            A.thr1 = acc.thr[0]; A.thr2 = acc.thr[1];
            A.all1 = acc.thr_is_2p32[0] ? 0xffffffffu : 0u;
            A.all2 = acc.thr_is_2p32[1] ? 0xffffffffu : 0u;
            A.rmask = half_mask(h, half);
            if (T == 64) k_amsc<64, W><<<(unsigned)(B * B / 2), 64 * 64 / 8, smem, hooks().stream>>>(A);
            else k_amsc<32, W><<<(unsigned)(B * B / 2), 32 * 32 / 8, smem, hooks().stream>>>(A);
            count_launch();
        }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

}  // namespace ising
