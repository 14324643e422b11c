// flow_planes_device.cuh — k_flow_planes: the HBM-resident double-checkerboard sweep as ONE persistent launch per
// ising_sweep call, the kernel boundary between the coarse colours replaced by data flow.
//
// With a launch per colour every launch starts with all warps waiting for their tiles and ends with SMs running dry (ncu,
// profiles/r02b: 8 % of the SM cycles of a launch have no warp to issue from).  Here the grid is as large as the GPU holds
// and lives for all n passes; warps draw tickets from one global counter, ticket = (phase, job), phase = 2 * pass + colour,
// in phase-major order.  A tile may run phase ph as soon as its four neighbours — the only tiles it reads, all of the other
// colour — have finished phase ph - 1: every tile publishes the number of phases it has completed (prog[tile],
// release), a job polls the 4 NS counters it depends on (acquire).  The same wait covers the write-after-read hazard (a
// neighbour reads this tile's boundary copy in phase ph - 1).  Tickets are handed out in dependency order, so a waiting warp
// only ever waits for tickets already held by running warps: no deadlock, no co-residency requirement beyond "the grid fits",
// which it does by construction (grid = resident CTAs).  In row-major order a job's dependencies lie one whole phase back,
// except across the periodic wrap (tile row 0 needs row B - 1, the last of the previous phase): every phase therefore
// starts two tile rows further on than the one before, which puts every dependency at least B - 3 rows of tickets back —
// far more than the ~6000 jobs in flight — so the poll almost never spins and the tail of one phase overlaps the head of
// the next.  The int8 write-back table lives in shared memory (built once per CTA).
#pragma once
#include "tile_planes_device.cuh"

namespace ising {

namespace ISING_DEVICE_NS {

struct FlowArgs {
    PlaneArgs P;
    uint32_t n_phases;                    // 2 * passes
    uint32_t jobs_per_phase;              // R * tiles of one colour / (TPW * NS)
    uint32_t phase_shift;                 // jobs by which the start of a phase moves on from the previous one (two tile rows)
    uint32_t magic_jp;                    // fastdiv magic of jobs_per_phase
    uint32_t total;                       // n_phases * jobs_per_phase (< 2^32: the host splits longer calls)
    unsigned int* ticket;                 // zeroed
    uint32_t* prog;                       // per tile (replica-major, row-major): phases completed, zeroed
};

__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(uint32_t* p, uint32_t v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <int T, bool BITS, bool HASJ, uint32_t HP = kNoSpec, int NS = 1>
__global__ void __launch_bounds__(kPlaneThreads, 10) k_flow_planes(FlowArgs F) {
    using G = PG<T>;
    const PlaneArgs& A = F.P;
    __shared__ uint2 s_lut[256];
    for (int i = threadIdx.x; i < 256; i += blockDim.x) s_lut[i] = kByteLutGlobal.e[i];
    __syncthreads();
    const uint32_t lut_smem = (uint32_t)__cvta_generic_to_shared(s_lut);
    const int lane = threadIdx.x & 31;
    const int sub = lane / G::LPT, Y = lane % G::LPT;
    const uint32_t B = geom_B(A), JP = F.jobs_per_phase;
    const uint32_t total = F.total;
    uint32_t next = 0;
    if (lane == 0) next = atomicAdd(F.ticket, 1u);
    for (;;) {
        const uint32_t tk = __shfl_sync(0xffffffffu, next, 0);
        if (tk >= total) break;
        if (lane == 0) next = atomicAdd(F.ticket, 1u);           // the next ticket is on its way while this job runs
        const uint32_t ph = fastdiv(tk, JP, F.magic_jp), idx = tk - ph * JP;
        const int C = (int)(ph & 1u);
        // every phase starts two tile rows further on than the one before (see above)
        const uint32_t sh = ph * F.phase_shift;                  // < 2^32: n_phases * phase_shift <= total
        uint32_t job = idx + (sh - fastdiv(sh, JP, F.magic_jp) * JP);
        if (job >= JP) job -= JP;
        int r, tx0, ty;
        job_tile<T, NS>(A, job, sub, r, tx0, ty, C);
        const uint32_t uty = (uint32_t)ty, row0 = (uint32_t)r * B * B, rowc = row0 + uty * B;
        const uint32_t tyU = uty == 0 ? B - 1 : uty - 1, tyD = uty == B - 1 ? 0 : uty + 1;
        if (ph > 0) {
            // lanes Y = 0..3 of every tile poll its up / down / left / right neighbours, per slot
            bool ok;
            do {
                ok = true;
                if (Y < 4) {
#pragma unroll
                    for (int s = 0; s < NS; ++s) {
                        const uint32_t utx = (uint32_t)(tx0 + 2 * s);
                        const uint32_t txL = utx == 0 ? B - 1 : utx - 1, txR = utx == B - 1 ? 0 : utx + 1;
                        const uint32_t nb = Y == 0 ? row0 + tyU * B + utx : Y == 1 ? row0 + tyD * B + utx : Y == 2 ? rowc + txL : rowc + txR;
                        ok = ok && ld_acquire_u32(F.prog + nb) >= ph;
                    }
                }
            } while (!__all_sync(0xffffffffu, ok));     // (the vote orders the other lanes' loads behind the polling lanes' acquires;
        }                                               //  no tile data is ever allocated in L1: body no_allocate, halos .cg)
        TileRegs<T> t[NS];
        uint4 Jw[NS][2][G::NW];
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const int tx = tx0 + 2 * s;
            load_tile<T, BITS>(A, r, tx, ty, Y, sub * G::LPT, t[s]);
#pragma unroll
            for (int cc = 0; cc < 2; ++cc)
#pragma unroll
                for (int gx = 0; gx < G::NW; ++gx)
                    Jw[s][cc][gx] = HASJ ? __ldg(A.jrec + ((size_t)ty * B + tx) * (2 * G::NW * G::LPT) + (cc * G::NW + gx) * G::LPT + Y)
                                         : make_uint4(0u, 0u, 0u, 0u);
        }
#if defined(ISING_JIT_R) && ISING_JIT_R == 1
        const uint64_t seed = A.seed0;
#else
        const uint64_t seed = A.seeds[r];
#endif
        const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
        const uint32_t Yg = (uint32_t)(ty * G::LPT + Y);
        const uint32_t g0 = Yg * (B * G::NW) + (uint32_t)(tx0 * G::NW);
        const uint32_t p0 = 2u * Yg * (B * (uint32_t)(T / 2)) + 16u * (uint32_t)(tx0 * G::NW);
        const uint64_t tbase = A.t_first + (uint64_t)(ph >> 1) * (uint64_t)A.k;
        for (int j = 0; j < A.k; ++j) {
            const uint64_t tt = tbase + (uint64_t)j;
#pragma unroll
            for (int c = 0; c < 2; ++c)
#pragma unroll
                for (int s = 0; s < NS; ++s)
                    half_sweep<T, HASJ, false, HP>(A, t[s], Jw[s], c, Y, g0 + (uint32_t)(2 * s * G::NW), p0 + 32u * (uint32_t)(s * G::NW), 2 * tt + (uint64_t)c, k0, k1);
        }
#pragma unroll
        for (int s = 0; s < NS; ++s) store_tile<T, BITS, true>(A, r, tx0 + 2 * s, ty, Y, sub, t[s], nullptr, lut_smem);
        __syncwarp();
        if (Y == 0) {                                // one lane per tile: everything the warp stored happens-before this release
            __threadfence();
#pragma unroll
            for (int s = 0; s < NS; ++s) st_release_u32(F.prog + rowc + (uint32_t)(tx0 + 2 * s), ph + 1u);
        }
    }
}


// ---- k_flow_planes_staged: the same kernel with the bodies of a warp's NEXT job travel from HBM to shared memory by the TMA engine while the
// warp updates its current job (BASELINE north_star: "TMA or cp.async staging of tile plus halo into shared memory"): one
// cp.async.bulk per tile record body (contiguous T*T bytes; the 64 edge bytes of the four neighbours are fetched as before,
// they are what the progress counters guard) behind one mbarrier per warp.  A tile's body was last written two phases ago
// by whichever warp owned it then; the prefetch first waits for that (prog >= ph - 1), which is always long past — the
// host only selects STAGE when a phase holds more than twice as many jobs as there are warps.
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy) : "memory");
}

template <int T, bool BITS, bool HASJ, uint32_t HP = kNoSpec, int NS = 1>
__global__ void __launch_bounds__(kPlaneThreads, 10) k_flow_planes_staged(FlowArgs F) {
    constexpr bool STAGE = true;
    using G = PG<T>;
    constexpr uint32_t REC = BITS ? G::REC_BITS : G::REC_I8;
    constexpr uint32_t BODY = REC - G::EDGE;
    constexpr uint32_t WBUF = G::TPW * NS * BODY;                 // staged bytes per warp
    const PlaneArgs& A = F.P;
    __shared__ uint2 s_lut[256];
    __shared__ __align__(8) unsigned long long s_bar[kPlaneThreads / 32];
    extern __shared__ __align__(128) uint8_t flow_stage[];       // STAGE: WBUF bytes per warp
    for (int i = threadIdx.x; i < 256; i += blockDim.x) s_lut[i] = kByteLutGlobal.e[i];
    const int lane = threadIdx.x & 31, wic = threadIdx.x >> 5;
    const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&s_bar[wic]);
    const uint32_t wbuf = STAGE ? (uint32_t)__cvta_generic_to_shared(flow_stage) + (uint32_t)wic * WBUF : 0u;
    if (STAGE && lane == 0) {
        mbar_init(bar, 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    const uint32_t lut_smem = (uint32_t)__cvta_generic_to_shared(s_lut);
    const int sub = lane / G::LPT, Y = lane % G::LPT;
    const uint32_t B = geom_B(A), JP = F.jobs_per_phase;
    const uint32_t total = F.total;
    const uint64_t pol = body_policy(A.stream != 0);

    auto decode = [&](uint32_t tk, uint32_t& ph, int& r, int& tx0, int& ty) {
        ph = fastdiv(tk, JP, F.magic_jp);
        const uint32_t idx = tk - ph * JP;
        // every phase starts two tile rows further on than the one before (see above)
        const uint32_t sh = ph * F.phase_shift;                  // < 2^32: n_phases * phase_shift <= total
        uint32_t job = idx + (sh - fastdiv(sh, JP, F.magic_jp) * JP);
        if (job >= JP) job -= JP;
        job_tile<T, NS>(A, job, sub, r, tx0, ty, (int)(ph & 1u));
    };
    // TMA: the bodies of ticket tk's tiles -> this warp's buffer (all lanes must have finished reading it)
    auto stage = [&](uint32_t tk) {
        uint32_t ph; int r, tx0, ty;
        decode(tk, ph, r, tx0, ty);
        const uint32_t rowc = ((uint32_t)r * B + (uint32_t)ty) * B;
        if (ph >= 2) {                                           // the tiles' own last write-back (two phases ago) must have landed
            bool ok;
            do {
                ok = true;
                if (Y == 0) {
#pragma unroll
                    for (int s = 0; s < NS; ++s) ok = ok && ld_acquire_u32(F.prog + rowc + (uint32_t)(tx0 + 2 * s)) >= ph - 1u;
                }
            } while (!__all_sync(0xffffffffu, ok));
        }
        if (lane == 0) mbar_expect_tx(bar, WBUF);
        __syncwarp();
        if (Y == 0) {
            asm volatile("fence.proxy.async;" ::: "memory");     // generic-proxy writes (other SMs, acquired above) and reads (ours) before async-proxy accesses
#pragma unroll
            for (int s = 0; s < NS; ++s)
                bulk_g2s(wbuf + (uint32_t)(sub * NS + s) * BODY, A.tiles + (uint64_t)(rowc + (uint32_t)(tx0 + 2 * s)) * REC, BODY, bar, pol);
        }
    };

    uint32_t cur = 0, next = 0, parity = 0;
    if (lane == 0) { cur = atomicAdd(F.ticket, 1u); next = atomicAdd(F.ticket, 1u); }
    cur = __shfl_sync(0xffffffffu, cur, 0);
    if (STAGE && cur < total) stage(cur);
    for (;;) {
        const uint32_t tk = cur;
        if (tk >= total) break;
        const uint32_t nxt = __shfl_sync(0xffffffffu, next, 0);
        if (lane == 0) next = atomicAdd(F.ticket, 1u);           // one more ticket is on its way while this job runs
        uint32_t ph; int r, tx0, ty;
        decode(tk, ph, r, tx0, ty);
        const uint32_t uty = (uint32_t)ty, row0 = (uint32_t)r * B * B, rowc = row0 + uty * B;
        const uint32_t tyU = uty == 0 ? B - 1 : uty - 1, tyD = uty == B - 1 ? 0 : uty + 1;
        if (ph > 0) {
            // lanes Y = 0..3 of every tile poll its up / down / left / right neighbours, per slot
            bool ok;
            do {
                ok = true;
                if (Y < 4) {
#pragma unroll
                    for (int s = 0; s < NS; ++s) {
                        const uint32_t utx = (uint32_t)(tx0 + 2 * s);
                        const uint32_t txL = utx == 0 ? B - 1 : utx - 1, txR = utx == B - 1 ? 0 : utx + 1;
                        const uint32_t nb = Y == 0 ? row0 + tyU * B + utx : Y == 1 ? row0 + tyD * B + utx : Y == 2 ? rowc + txL : rowc + txR;
                        ok = ok && ld_acquire_u32(F.prog + nb) >= ph;
                    }
                }
            } while (!__all_sync(0xffffffffu, ok));     // (the vote orders the other lanes' loads behind the polling lanes' acquires;
        }                                               //  no tile data is ever allocated in L1: body no_allocate, halos .cg)
        if (STAGE) { mbar_wait(bar, parity); parity ^= 1u; }
        TileRegs<T> t[NS];
        uint4 Jw[NS][2][G::NW];
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const int tx = tx0 + 2 * s;
            load_tile<T, BITS>(A, r, tx, ty, Y, sub * G::LPT, t[s], STAGE ? wbuf + (uint32_t)(sub * NS + s) * BODY : 0u);
#pragma unroll
            for (int cc = 0; cc < 2; ++cc)
#pragma unroll
                for (int gx = 0; gx < G::NW; ++gx)
                    Jw[s][cc][gx] = HASJ ? __ldg(A.jrec + ((size_t)ty * B + tx) * (2 * G::NW * G::LPT) + (cc * G::NW + gx) * G::LPT + Y)
                                         : make_uint4(0u, 0u, 0u, 0u);
        }
        if (STAGE) {
            __syncwarp();                                // every lane has its pieces in registers: the buffer is free
            if (nxt < total) stage(nxt);
        }
#if defined(ISING_JIT_R) && ISING_JIT_R == 1
        const uint64_t seed = A.seed0;
#else
        const uint64_t seed = A.seeds[r];
#endif
        const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
        const uint32_t Yg = (uint32_t)(ty * G::LPT + Y);
        const uint32_t g0 = Yg * (B * G::NW) + (uint32_t)(tx0 * G::NW);
        const uint32_t p0 = 2u * Yg * (B * (uint32_t)(T / 2)) + 16u * (uint32_t)(tx0 * G::NW);
        const uint64_t tbase = A.t_first + (uint64_t)(ph >> 1) * (uint64_t)A.k;
        for (int j = 0; j < A.k; ++j) {
            const uint64_t tt = tbase + (uint64_t)j;
#pragma unroll
            for (int c = 0; c < 2; ++c)
#pragma unroll
                for (int s = 0; s < NS; ++s)
                    half_sweep<T, HASJ, false, HP>(A, t[s], Jw[s], c, Y, g0 + (uint32_t)(2 * s * G::NW), p0 + 32u * (uint32_t)(s * G::NW), 2 * tt + (uint64_t)c, k0, k1);
        }
#pragma unroll
        for (int s = 0; s < NS; ++s) store_tile<T, BITS, true>(A, r, tx0 + 2 * s, ty, Y, sub, t[s], nullptr, lut_smem);
        __syncwarp();
        if (Y == 0) {                                // one lane per tile: everything the warp stored happens-before this release
            __threadfence();
#pragma unroll
            for (int s = 0; s < NS; ++s) st_release_u32(F.prog + rowc + (uint32_t)(tx0 + 2 * s), ph + 1u);
        }
        cur = nxt;
    }
}

}  // namespace

}  // namespace ising
