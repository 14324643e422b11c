#pragma once
#include "tile_planes_device.cuh"

namespace ising {

namespace ISING_DEVICE_NS {

// grid_planes_device.cuh — k_grid_planes: the whole lattice on chip across ALL SMs (the paper's own sizes, 512 < L <= 4096: P:78; BASELINE
// config 2; VERDICT round 1 "missing" 3).  Between L = 1024 and L ~ 4096 a launch per coarse colour holds fewer warps than
// the GPU has schedulers and a pass costs two launch latencies; the cluster-resident kernel above stops at 16 SMs.  Here
// ONE launch per ising_sweep call keeps every tile in registers on all SMs for all n passes: warp w of the grid owns
// the jobs w, w + W, ... (at most M) of each coarse colour and alternates between them, phase by phase.  There is no
// grid-wide barrier: a tile needs only the boundary words of its four neighbours as they stood at the end of the
// previous phase (same-colour tiles never touch), so after every phase a tile publishes its boundary words in a
// 128-byte exchange record in global memory (L2), each word as one 64-bit store {value, version}, version = number of
// phases done; a neighbour polls exactly the words it needs until their version is the phase it is about to run
// (relaxed gpu-scope loads: every word validates itself, no fence).  A tile rewrites its record only after its neighbours have
// published the next version, i.e. after they have read this one, so one buffer per tile suffices.  All CTAs must be
// co-resident (the launch is cooperative for that guarantee only).  HBM is touched twice per call.
constexpr int kGridAccSlots = 8;          // copies of the per-pass accumulators (same-address atomics spread out)

struct GridArgs {
    PlaneArgs P;
    int n;                                // outer passes
    uint32_t jobs_total;                  // R * jobs per colour
    uint32_t tiles_per_colour;            // per replica
    uint32_t jobs_per_warp;               // M: jobs of each colour a warp owns (state in shared memory between phases)
    unsigned long long* xedge;            // per tile 16 x u64: TOP[4] | COL[4] = {L0, L1, R0, R1} | BOT[4] | pad; u64 = version << 32 | word
    long long* acc;                       // optional series accumulators [n][R][kGridAccSlots][2] = {#up, #unsatisfied}, zeroed
    uint32_t magic_k;                     // PC kernels: fastdiv magic of k
};

__device__ __forceinline__ ulonglong2 ld_xedge2(const unsigned long long* p) {
    ulonglong2 v;
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0,%1}, [%2];" : "=l"(v.x), "=l"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_xedge2(unsigned long long* p, unsigned long long a, unsigned long long b) {
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1,%2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}

// ---- PC = true: producer / consumer form for lattices so small that every warp would be alone on its scheduler (one job
// per colour for fewer warps than the GPU has schedulers: L = 1024 at tile 32).  There a warp's k inner sweeps are a serial
// chain of ~800 cycles per block update, 85 % of it random numbers and compares that do not depend on the spins.  A CTA is
// then one consumer warp (warp 0: the grid worker described above) and 3 or 7 producer warps on the schedulers of the SM
// (two warps per scheduler overlap their ALU and multiplier work, a single warp cannot): the producers compute R_m = [r < thr[m]] (head planes, borrow chains, ties resolved for every site whose head
// equals a threshold head) for the consumer's coming half-sweeps, round robin, into a ring in shared memory; the consumer
// only does the spin-dependent part (neighbour words, bit adder, flip = [n>=2] | [n>=1] & R1 | R2: ~40 instructions).
constexpr int kPcRing = 16;               // half-sweeps of masks in flight per consumer

__device__ __forceinline__ uint32_t lds_acquire(uint32_t saddr) {
    uint32_t v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_release(uint32_t saddr, uint32_t v) {
    asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory");
}

// the spin-dependent part of update_block for all blocks of the lane, R1 / R2 given
template <int T, bool HASJ>
__device__ __forceinline__ void half_sweep_masks(const PlaneArgs& A, TileRegs<T>& t, const uint4 (&Jw)[2][PG<T>::NW], int c, int Y,
                                                 const uint32_t (&R1)[PG<T>::NW], const uint32_t (&R2)[PG<T>::NW]) {
    using G = PG<T>;
    uint32_t Snew[G::NW];
#pragma unroll
    for (int gx = 0; gx < G::NW; ++gx) {
        uint32_t V1, V2, H1, H2;
        neighbour_words<T, false>(t, c, gx, Y, V1, V2, H1, H2);
        const uint32_t S = t.S[c][gx];
        const uint4& J = Jw[c][gx];
        const uint32_t a = S ^ V1 ^ (HASJ ? J.x : 0u), b = S ^ V2 ^ (HASJ ? J.y : 0u);
        const uint32_t e = S ^ H1 ^ (HASJ ? J.z : 0u), d = S ^ H2 ^ (HASJ ? J.w : 0u);
        const uint32_t p1 = a | b, q1 = a & b, p2 = e | d, q2 = e & d;
        const uint32_t ge1 = p1 | p2, ge2 = (p1 & p2) | q1 | q2 | A.force;
        Snew[gx] = S ^ (ge2 | (ge1 & R1[gx]) | R2[gx]);
    }
#pragma unroll
    for (int gx = 0; gx < G::NW; ++gx) t.S[c][gx] = Snew[gx];
}

// CTA shape: the pre-compiled kernels take up to 128 threads, 5 CTAs per SM; the run-time build names its own (launch_grid_one)
#ifndef ISING_G2_THREADS
#define ISING_G2_THREADS 128
#define ISING_G2_BLOCKS 5
#endif
// ISING_G2_PARK = 0 (run-time build only): the jobs' constants are not parked beside their words but decoded again in every
// phase (a dozen instructions with the geometry known at compile time), so that shared memory holds nothing but spins:
// 28 warps x 16 jobs x 512 bytes = 229376 of the 232448 bytes of an SM hold a 16384^2 lattice on the 148 SMs of a B200.
#ifndef ISING_G2_PARK
#define ISING_G2_PARK 1
#endif
// ISING_G2_SERIES = 0 / 1 (run-time build): whether the E / M series is taken is known when the kernel is compiled (without
// the accounting code the 28-warp kernel needs 70 registers and nothing spills; with it 72 and 40 bytes of spills)
#ifndef ISING_G2_SERIES
#define ISING_G2_SERIES -1
#endif
// ISING_G2_STRIP = M > 0 (run-time build, several jobs per warp): warp w owns the M CONSECUTIVE jobs w M ... w M + M - 1 of
// each colour, i.e. a strip of 2 M (tile 64) or 4 M (tile 32) adjacent tiles of one tile row (M divides the jobs of a row),
// instead of the jobs w, w + W, ...  The left and right neighbours of a tile (other colour, same row) are then the warp's
// own jobs, except at the two ends of the strip: their boundary columns are read from the words the warp has parked in shared
// memory (same block row = same lane, or the other half-warp at tile 32) instead of being published to and polled from L2;
// only the tile rows above and below, and the strip ends, go through the exchange records.  With the colour-C tiles of a row at
// tx = 2 q + p, p = (ty + C) & 1, and the other colour's at 2 q' + 1 - p: p = 0: right neighbour q' = q, left q' = q - 1;
// p = 1: left q' = q, right q' = q + 1 (tile 32: q = 2 job + sub).
// (Tried without strips, any mapping: the other colour's job of the SAME index is always the warp's own neighbour, to the right
// where p = 0, to the left where p = 1, so one of the two columns could always come from shared memory, halving the column
// exchange.  Measured: config 3 tile 64 k = 1 2990 -> 2894 flips/ns, L = 4096 and 8192 unchanged or -1 %: dropped.)
#ifndef ISING_G2_STRIP
#define ISING_G2_STRIP 0
#endif

// tile row (its parity is all that is used) of the strip that starts at job j0: jobs of a colour are enumerated row by row
template <int T>
__device__ __forceinline__ uint32_t geom_strip_row(const PlaneArgs& A, uint32_t j0) {
    const uint32_t jobs_per_row = geom_B(A) / 2u / (uint32_t)PG<T>::TPW;
    return (j0 / jobs_per_row) % geom_B(A);
}

template <int T, bool BITS, bool HASJ, uint32_t HP = kNoSpec, bool PC = false>
__global__ void __launch_bounds__(PC ? 256 : ISING_G2_THREADS, PC ? 2 : ISING_G2_BLOCKS) k_grid_planes(GridArgs R) {
    using G = PG<T>;
    constexpr int NWORDS = 2 * G::NW;                         // words per lane and job: S[cc][gx]
    constexpr bool PARK = PC || ISING_G2_PARK;
    constexpr int NSLOT = NWORDS + (PARK ? 7 : 0);            // ... + the job's constants (decoded once): self, nU, nD, nL, nR, tx | ty << 16, r
    extern __shared__ uint32_t grid_smem[];                   // per warp: [colour][job][slot][lane]
    const PlaneArgs& A = R.P;
    const int lane = threadIdx.x & 31;
    const int wic = threadIdx.x >> 5;
    const uint32_t wg = PC ? blockIdx.x : blockIdx.x * (blockDim.x >> 5) + (uint32_t)wic, W = PC ? gridDim.x : gridDim.x * (blockDim.x >> 5);
    const int sub = lane / G::LPT, Y = lane % G::LPT;
    const uint32_t B = geom_B(A);
    constexpr uint32_t STRIP = PC ? 0u : (uint32_t)ISING_G2_STRIP;
    const uint32_t Mw = PC ? 1u : (STRIP ? STRIP : R.jobs_per_warp);
    auto job_of = [&](uint32_t m) { return STRIP ? wg * Mw + m : wg + m * W; };
    uint32_t* const ws = grid_smem + (PC ? 0u : (size_t)wic * (2u * Mw * NSLOT * 32u)) + lane;
    // PC: behind the consumer's area, the ring [slot][R1 | R2][gx][lane], its "full" words and the consumed counter
    uint32_t* const ring = grid_smem + 2u * NSLOT * 32u;
    const uint32_t flags = (uint32_t)__cvta_generic_to_shared(ring + kPcRing * 2 * G::NW * 32);
    const uint32_t total_hs = PC ? (uint32_t)R.n * 4u * (uint32_t)A.k : 0u;
    const uint2* lut = kByteLutGlobal.e;
    const bool series = ISING_G2_SERIES < 0 ? R.acc != nullptr : ISING_G2_SERIES != 0;

    struct Job { int r, tx, ty; uint32_t self, nU, nD, nL, nR; };
    auto decode = [&](uint32_t job, int C) {
        int ri, txi, tyi;
        job_tile<T>(A, job, sub, ri, txi, tyi, C);
        const uint32_t r = (uint32_t)ri, tx = (uint32_t)txi, ty = (uint32_t)tyi;
        const uint32_t base = r * B * B, row = base + ty * B;
        const uint32_t tyU = ty == 0 ? B - 1 : ty - 1, tyD = ty == B - 1 ? 0 : ty + 1;
        if (STRIP) return Job{(int)r, (int)tx, (int)ty, row + tx, base + tyU * B + tx, base + tyD * B + tx, 0u, 0u};      // nL / nR: refresh, strip ends only
        const uint32_t txL = tx == 0 ? B - 1 : tx - 1, txR = tx == B - 1 ? 0 : tx + 1;
        return Job{(int)r, (int)tx, (int)ty, row + tx, base + tyU * B + tx, base + tyD * B + tx, row + txL, row + txR};
    };
    auto jwords = [&](const Job& jb, uint4 (&Jw)[2][G::NW]) {
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int gx = 0; gx < G::NW; ++gx)
                Jw[cc][gx] = HASJ ? __ldg(A.jrec + ((size_t)jb.ty * B + jb.tx) * (2 * G::NW * G::LPT) + (cc * G::NW + gx) * G::LPT + Y)
                                  : make_uint4(0u, 0u, 0u, 0u);
    };
    // the tile's boundary words, version ver, into its exchange record
    auto publish = [&](const TileRegs<T>& tt, const Job& jb, uint32_t ver, int C, uint32_t m) {
        const uint32_t sh = (uint32_t)sub * G::LPT, msk = G::LPT == 32 ? 0xffffffffu : ((1u << G::LPT) - 1u);
        const unsigned long long v = (unsigned long long)ver << 32;
        unsigned long long* e = R.xedge + (size_t)jb.self * 16;
        // STRIP: only the tiles at the two ends of the warp's strip have a left / right neighbour in another warp (warp-uniform)
        const uint32_t par = ((uint32_t)jb.ty + (uint32_t)C) & 1u;
        const bool pubL = !STRIP || (par == 0u && m == 0u), pubR = !STRIP || (par == 1u && m + 1u == Mw);
        if (pubL) {
            const uint32_t L0 = (__ballot_sync(0xffffffffu, tt.S[0][0] & 1u) >> sh) & msk;
            const uint32_t L1 = (__ballot_sync(0xffffffffu, (tt.S[1][0] >> 16) & 1u) >> sh) & msk;
            if (Y == 0 && (!STRIP || sub == 0)) st_xedge2(e + 4, v | L0, v | L1);      // (T = 32: Y = 0 of each of the two tiles)
        }
        if (pubR) {
            const uint32_t R0 = (__ballot_sync(0xffffffffu, (tt.S[1][G::NW - 1] >> 15) & 1u) >> sh) & msk;
            const uint32_t R1 = (__ballot_sync(0xffffffffu, tt.S[0][G::NW - 1] >> 31) >> sh) & msk;
            if (Y == 0 && (!STRIP || sub == G::TPW - 1)) st_xedge2(e + 6, v | R0, v | R1);
        }
        if (Y == 0 || Y == G::LPT - 1) {
            unsigned long long* rw = e + (Y == 0 ? 0 : 8);          // TOP : BOT
            if (G::NW == 2) {
                st_xedge2(rw, v | tt.S[0][0], v | tt.S[0][1]);
                st_xedge2(rw + 2, v | tt.S[1][0], v | tt.S[1][1]);
            } else {
                st_xedge2(rw, v | tt.S[0][0], v | tt.S[1][0]);
            }
        }
    };
    // wait until the four neighbours have published version `want`, and take the halos from their words
    auto refresh = [&](TileRegs<T>& tt, const Job& jb, uint32_t want, int C, uint32_t m) {
        const unsigned long long* rowp = R.xedge + (size_t)(Y == 0 ? jb.nU : jb.nD) * 16 + (Y == 0 ? 8 : 0);   // BOT of the tile above : TOP of the tile below
        auto left_of = [&]() { return STRIP ? jb.self - (uint32_t)jb.tx + (jb.tx == 0 ? B - 1u : (uint32_t)jb.tx - 1u) : jb.nL; };
        auto right_of = [&]() { return STRIP ? jb.self - (uint32_t)jb.tx + ((uint32_t)jb.tx == B - 1u ? 0u : (uint32_t)jb.tx + 1u) : jb.nR; };
        const bool need_row = Y == 0 || Y == G::LPT - 1;
        bool extL = true, extR = true;                        // (per lane) the neighbour lives in another warp: through the exchange record
        bool edge = true;                                     // (per warp) some lane has such a neighbour
        if (STRIP) {
            if (G::TPW == 2) __syncwarp();                    // the other half-warp's parked words: written by other lanes
            // slot (of the other colour) and lane of the tiles to the left and to the right (header comment)
            const uint32_t par = ((uint32_t)jb.ty + (uint32_t)C) & 1u;
            edge = par == 0u ? m == 0u : m + 1u == Mw;
            constexpr int S = NSLOT * 32;
            const uint32_t* same = ws + (size_t)((uint32_t)(1 - C) * Mw + m) * (uint32_t)S;      // the other colour's job of the same index
            const uint32_t *ql, *qr;
            if (G::TPW == 1) {
                ql = same - (par ? 0 : S); qr = ql + S;
            } else {
                const int flip = (lane & 16) ? -16 : 16;
                if (par == 0u) { qr = same; ql = same + flip - (sub == 0 ? S : 0); }
                else { ql = same; qr = same + flip + (sub == 1 ? S : 0); }
            }
            extL = par == 0u && m == 0u && (G::TPW == 1 || sub == 0);
            extR = par == 1u && m + 1u == Mw && (G::TPW == 1 || sub == 1);
            if (!extL) { tt.hL0 = (ql[(2 * G::NW - 1) * 32] >> 15) & 1u; tt.hL1 = ql[(G::NW - 1) * 32] >> 31; }      // its R0, R1
            if (!extR) { tt.hR0 = qr[0] & 1u; tt.hR1 = (qr[G::NW * 32] >> 16) & 1u; }                               // its L0, L1
        }
        if (STRIP && !edge) {                                 // all but one job of a phase: only the tile rows above and below
            for (;;) {
                ulonglong2 r0 = make_ulonglong2(0, 0), r1 = r0;
                bool ok = true;
                if (need_row) {
                    r0 = ld_xedge2(rowp);
                    ok = (uint32_t)(r0.x >> 32) == want && (uint32_t)(r0.y >> 32) == want;
                    if (G::NW == 2) {
                        r1 = ld_xedge2(rowp + 2);
                        ok = ok && (uint32_t)(r1.x >> 32) == want && (uint32_t)(r1.y >> 32) == want;
                    }
                }
                if (__all_sync(0xffffffffu, ok)) {
                    tt.vrow[0][0] = (uint32_t)r0.x;
                    if (G::NW == 2) { tt.vrow[0][1] = (uint32_t)r0.y; tt.vrow[1][0] = (uint32_t)r1.x; tt.vrow[1][1] = (uint32_t)r1.y; }
                    else tt.vrow[1][0] = (uint32_t)r0.y;
                    return;
                }
            }
        }
        const unsigned long long* lf = R.xedge + (size_t)left_of() * 16 + 6;                                    // {R0, R1}
        const unsigned long long* rt = R.xedge + (size_t)right_of() * 16 + 4;                                   // {L0, L1}
        for (;;) {
            ulonglong2 r0 = make_ulonglong2(0, 0), r1 = r0, a = r0, b = r0;
            bool ok = true;
            if (extL) {
                a = ld_xedge2(lf);
                ok = ok && (uint32_t)(a.x >> 32) == want && (uint32_t)(a.y >> 32) == want;
            }
            if (extR) {
                b = ld_xedge2(rt);
                ok = ok && (uint32_t)(b.x >> 32) == want && (uint32_t)(b.y >> 32) == want;
            }
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
                if (extL) { tt.hL0 = ((uint32_t)a.x >> Y) & 1u; tt.hL1 = ((uint32_t)a.y >> Y) & 1u; }
                if (extR) { tt.hR0 = ((uint32_t)b.x >> Y) & 1u; tt.hR1 = ((uint32_t)b.y >> Y) & 1u; }
                return;
            }
        }
    };
    // a10 on the registers: the job's share of #up and #unsatisfied bonds of pass `pass`
    auto account = [&](const TileRegs<T>& tt, const uint4 (&Jw)[2][G::NW], int r, int pass) {
        int up = 0, unsat = 0;
        count_row<T, false>(tt, Jw, Y, up, unsat);
#pragma unroll
        for (int d = G::LPT / 2; d > 0; d >>= 1) {
            up += __shfl_xor_sync(0xffffffffu, up, d);
            unsat += __shfl_xor_sync(0xffffffffu, unsat, d);
        }
        if (Y == 0) {
            long long* a = R.acc + (((size_t)pass * A.R + r) * kGridAccSlots + (wg % kGridAccSlots)) * 2;
            atomicAdd(reinterpret_cast<unsigned long long*>(a), (unsigned long long)up);
            atomicAdd(reinterpret_cast<unsigned long long*>(a + 1), (unsigned long long)unsat);
        }
    };
    auto sm_job = [&](int C, uint32_t m) {                             // the constants parked by the prologue
        if (!PARK) return decode(job_of(m), C);
        const uint32_t* p = ws + (size_t)((uint32_t)C * Mw + m) * (NSLOT * 32u) + NWORDS * 32;
        const uint32_t xy = p[5 * 32];
        return Job{(int)p[6 * 32], (int)(xy & 0xffffu), (int)(xy >> 16), p[0], p[1 * 32], p[2 * 32], p[3 * 32], p[4 * 32]};
    };
    auto sm_put_job = [&](const Job& jb, int C, uint32_t m) {
        if (!PARK) return;
        uint32_t* p = ws + (size_t)((uint32_t)C * Mw + m) * (NSLOT * 32u) + NWORDS * 32;
        p[0] = jb.self; p[1 * 32] = jb.nU; p[2 * 32] = jb.nD; p[3 * 32] = jb.nL; p[4 * 32] = jb.nR;
        p[5 * 32] = (uint32_t)jb.tx | ((uint32_t)jb.ty << 16); p[6 * 32] = (uint32_t)jb.r;
    };
    auto sm_load = [&](TileRegs<T>& tt, int C, uint32_t m) {
        const uint32_t* p = ws + (size_t)((uint32_t)C * Mw + m) * (NSLOT * 32u);
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int gx = 0; gx < G::NW; ++gx) tt.S[cc][gx] = p[(cc * G::NW + gx) * 32];
    };
    auto sm_store = [&](const TileRegs<T>& tt, int C, uint32_t m) {
        uint32_t* p = ws + (size_t)((uint32_t)C * Mw + m) * (NSLOT * 32u);
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int gx = 0; gx < G::NW; ++gx) p[(cc * G::NW + gx) * 32] = tt.S[cc][gx];
    };

    if (PC && threadIdx.x < kPcRing + 1) ring[kPcRing * 2 * G::NW * 32 + threadIdx.x] = 0u;      // full[] and the consumed counter
    // records -> shared memory; the colour-1 tiles publish their initial boundary (version 1 = what phase 0 waits for)
    for (int C = 0; C < 2 && (!PC || wic == 0); ++C)
        for (uint32_t m = 0; m < Mw; ++m) {
            const uint32_t job = job_of(m);
            if (job >= R.jobs_total) break;                               // warp-uniform
            const Job jb = decode(job, C);
            TileRegs<T> tt;
            load_tile<T, BITS>(A, jb.r, jb.tx, jb.ty, Y, sub * G::LPT, tt);
            sm_store(tt, C, m);
            sm_put_job(jb, C, m);
            if (C == 1) publish(tt, jb, 1u, C, m);
        }

    if constexpr (PC) {
        __syncthreads();                                   // the consumer's job constants and the ring flags are in place
        if (wic > 0) {                                     // ---- producers: masks of the half-sweeps wic - 1, wic - 1 + 3, ...
            if (wg < R.jobs_total) {
                const uint32_t NP = (blockDim.x >> 5) - 1u;              // producer warps of the CTA
                for (uint32_t hs = (uint32_t)wic - 1u; hs < total_hs; hs += NP) {
                    const uint32_t c = hs & 1u, q = hs >> 1;
                    const uint32_t phq = fastdiv(q, (uint32_t)A.k, R.magic_k), j = q - phq * (uint32_t)A.k;
                    const int C = (int)(phq & 1u);
                    const Job jb = sm_job(C, 0);
                    const uint64_t seed = A.seeds[jb.r];
                    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
                    const uint32_t Yg = (uint32_t)(jb.ty * G::LPT + Y);
                    const uint32_t g0 = Yg * (B * G::NW) + (uint32_t)(jb.tx * G::NW);
                    const uint32_t p0 = 2u * Yg * (B * (uint32_t)(T / 2)) + 16u * (uint32_t)(jb.tx * G::NW);
                    const uint64_t H = 2 * (A.t_first + (uint64_t)(phq >> 1) * (uint64_t)A.k + (uint64_t)j) + (uint64_t)c;
                    uint32_t R1[G::NW], R2[G::NW], e1[G::NW], e2[G::NW], any = 0;
#pragma unroll
                    for (int gx = 0; gx < G::NW; ++gx) {
                        head_masks(A, g0 + (uint32_t)gx, (uint32_t)H, (uint32_t)(H >> 32), k0, k1, R1[gx], R2[gx], e1[gx], e2[gx]);
                        any |= e1[gx] | e2[gx];
                    }
                    if (any) {                             // ties: 2^-11 per site, whether or not the site will need that threshold
                        const uint32_t prow = B * (uint32_t)(T / 2);
#pragma unroll
                        for (int gx = 0; gx < G::NW; ++gx) {
                            uint32_t und = e1[gx] | e2[gx];
                            while (und) {
                                const int jj = __ffs(und) - 1;
                                und &= und - 1;
                                const uint32_t p = p0 + 16u * (uint32_t)gx + (uint32_t)(jj >> 4) * prow + (uint32_t)(jj & 15);
                                const u32x4 o = philox4x32_10(p, kTagTail, (uint32_t)H, (uint32_t)(H >> 32), k0, k1);
                                const uint32_t tail = o.x >> kHeadBits;
                                if ((e1[gx] >> jj) & 1u) R1[gx] |= (uint32_t)(tail < A.t1_tail) << jj;
                                if ((e2[gx] >> jj) & 1u) R2[gx] |= (uint32_t)(tail < A.t2_tail) << jj;
                            }
                        }
                    }
                    const uint32_t slot = hs % kPcRing;
                    if (hs >= kPcRing)                     // the consumer must be done with the slot's previous content
                        while ((int)(lds_acquire(flags + 4u * kPcRing) - (hs - kPcRing + 1u)) < 0) {}
                    uint32_t* dst = ring + (size_t)slot * (2 * G::NW * 32) + lane;
#pragma unroll
                    for (int gx = 0; gx < G::NW; ++gx) { dst[gx * 32] = R1[gx]; dst[(G::NW + gx) * 32] = R2[gx]; }
                    __syncwarp();
                    if (lane == 0) sts_release(flags + 4u * slot, hs + 1u);
                }
            }
            return;
        }
    }
    uint32_t hs_next = 0;                                  // PC: the consumer's running half-sweep index
    for (int pass = 0; pass < R.n; ++pass) {
        for (int C = 0; C < 2; ++C) {
            const uint32_t ph = 2u * (uint32_t)pass + (uint32_t)C;       // this phase waits for version ph + 1 and publishes ph + 2
            // (Starting each phase one band of jobs later, so that no job waits for the end of the phase before, was
            // measured: no gain at tile 32, -8 % at tile 64 where the extra state spills.)
            // STRIP: the two tiles at the ends of a strip wait for a tile of the neighbouring warp, and that one for them.  Where the
            // colour's tiles sit at even tx (p = 0) the dependent tile is m = 0, else m = M - 1: a warp walks its strip from that
            // end, so that both are the first job of their phases and each has had M - 1 jobs of time to arrive (walking always
            // from m = 0 made the first job of every phase wait for the last job of the phase before: -4 % at tile 64).
            const bool backwards = STRIP && (((geom_strip_row<T>(A, wg * Mw) + (uint32_t)C) & 1u) != 0u);
#pragma unroll 1                                                      // (unrolled by 2: tile 32 +0.6 %, tile 64 -4 %; by 4: -14 %)
            for (uint32_t mi = 0; mi < Mw; ++mi) {
                const uint32_t m = backwards ? Mw - 1u - mi : mi;
                const uint32_t job = job_of(m);
                if (job >= R.jobs_total) break;                           // warp-uniform
                const Job jb = sm_job(C, m);
                TileRegs<T> tt;
                sm_load(tt, C, m);
                uint4 Jw[2][G::NW];
                jwords(jb, Jw);
                refresh(tt, jb, ph + 1u, C, m);
                if (series && C == 0 && pass > 0) account(tt, Jw, jb.r, pass - 1);     // colour-0 tiles: the halos of the finished pass just arrived
#if defined(ISING_JIT_R) && ISING_JIT_R == 1
                const uint64_t seed = A.seed0;
#else
                const uint64_t seed = A.seeds[jb.r];
#endif
                const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
                const uint32_t Yg = (uint32_t)(jb.ty * G::LPT + Y);
                const uint32_t g0 = Yg * (B * G::NW) + (uint32_t)(jb.tx * G::NW);
                const uint32_t p0 = 2u * Yg * (B * (uint32_t)(T / 2)) + 16u * (uint32_t)(jb.tx * G::NW);
                for (int j = 0; j < A.k; ++j) {
                    const uint64_t t64 = A.t_first + (uint64_t)pass * (uint64_t)A.k + (uint64_t)j;
                    if (PC) {
#pragma unroll
                        for (int c = 0; c < 2; ++c) {
                            const uint32_t hs = hs_next++, slot = hs % kPcRing;
                            while (lds_acquire(flags + 4u * slot) != hs + 1u) {}
                            const uint32_t* src = ring + (size_t)slot * (2 * G::NW * 32) + lane;
                            uint32_t R1[G::NW], R2[G::NW];
#pragma unroll
                            for (int gx = 0; gx < G::NW; ++gx) { R1[gx] = src[gx * 32]; R2[gx] = src[(G::NW + gx) * 32]; }
                            __syncwarp();
                            if (lane == 0) sts_release(flags + 4u * kPcRing, hs + 1u);      // the slot may be refilled
                            half_sweep_masks<T, HASJ>(A, tt, Jw, c, Y, R1, R2);
                        }
                    } else {
                        half_sweep<T, HASJ, false, HP>(A, tt, Jw, 0, Y, g0, p0, 2 * t64, k0, k1);
                        half_sweep<T, HASJ, false, HP>(A, tt, Jw, 1, Y, g0, p0, 2 * t64 + 1, k0, k1);
                    }
                }
                publish(tt, jb, ph + 2u, C, m);
                if (series && C == 1) account(tt, Jw, jb.r, pass);       // colour-1 tiles: their halos (colour 0) are final for this pass
                sm_store(tt, C, m);
            }
        }
    }
    if (series && R.n > 0)
        for (uint32_t m = 0; m < Mw; ++m) {
            const uint32_t job = job_of(m);
            if (job >= R.jobs_total) break;
            const Job jb = sm_job(0, m);
            TileRegs<T> tt;
            sm_load(tt, 0, m);
            uint4 Jw[2][G::NW];
            jwords(jb, Jw);
            refresh(tt, jb, 2u * (uint32_t)R.n + 1u, 0, m);
            account(tt, Jw, jb.r, R.n - 1);
        }
    for (int C = 0; C < 2; ++C)
        for (uint32_t m = 0; m < Mw; ++m) {
            const uint32_t job = job_of(m);
            if (job >= R.jobs_total) break;
            const Job jb = sm_job(C, m);
            TileRegs<T> tt;
            sm_load(tt, C, m);
            store_tile<T, BITS>(A, jb.r, jb.tx, jb.ty, Y, sub, tt, lut);
        }
}

}  // namespace

}  // namespace ising
