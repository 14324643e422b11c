// tile_planes_device.cuh — device code of the 2D multi-spin tile kernel (see tile_planes.cu for the design
// notes).  Self-contained on top of philox.cuh / planes_common.cuh so that it compiles both into the library
// (nvcc) and, specialised on the head bits of the thresholds, at run time (NVRTC, planes_jit.cu).
#pragma once
#include "planes_common.cuh"

// Inside the library the kernels have internal linkage (anonymous namespace, like every other .cu file here);
// under NVRTC they need external linkage to be found by name.
#ifdef __CUDACC_RTC__
#define ISING_DEVICE_NS jit
#else
#define ISING_DEVICE_NS
#endif

namespace ising {

namespace ISING_DEVICE_NS {

template <int T>
struct PG {
    static constexpr int NW = T / 32;            // RNG blocks (words) per colour per lane
    static constexpr int LPT = T / 2;            // lanes per tile = block rows
    static constexpr int TPW = 64 / T;           // tiles per warp job
    static constexpr int NCH = 4 * NW;           // 16-byte pieces per lane
    static constexpr int BODY = T * T;
    // Every record ends with 64 bytes of bit-packed copies of the tile's own boundary, written by the tile, so
    // that a neighbour reads each halo as one 16-byte run of ready-made words (no sector per row, no unpacking):
    //   +0  TOP[cc][gx]: the words of block row 0 (low half = tile row 0)     -> the tile above reads them as "dn"
    //   +16 COL[4]: bit Y of {L0, L1, R0, R1} = spin at x = 0 of row 2Y, x = 0 of row 2Y+1, x = T-1 of row 2Y, of row 2Y+1
    //   +32 BOT[cc][gx]: the words of block row LPT-1 (high half = row T-1)   -> the tile below reads them as "up"
    //   +48 zero padding, so that both 32-byte sectors are always written whole (no read-modify-write in L2 / HBM)
    static constexpr int EDGE = 64, E_TOP = 0, E_COL = 16, E_BOT = 32;
    static constexpr int REC_I8 = T * T + EDGE;
    static constexpr int REC_BITS = T * T / 8 + EDGE;
};

struct PlaneArgs {
    uint8_t* tiles;              // records, replica-major
    const uint64_t* seeds;
    uint64_t seed0;              // seeds[0]: with one replica (known when the kernel is specialised at run time) the Philox key is a
                                 // kernel parameter, i.e. uniform: its ten-round schedule lives in uniform registers, not in 20 per lane
    int L, B, R;
    int C;                       // coarse colour of this launch
    int k;
    uint64_t t_first;            // inner-sweep index of the first of the k sweeps
    uint32_t njobs;
    uint32_t magic_rep, magic_hb; // ceil(2^32 / d) for d = tiles per colour per replica, B/2 (0xffffffff for d = 1)
    uint32_t u1[kHeadBits];      // plane q: all-ones if bit (31-q) of thr[1] is set, else 0
    uint32_t u2[kHeadBits];      // same for thr[2]
    uint32_t t1_tail, t2_tail;   // thr[m] & (2^20 - 1)
    uint32_t force;              // all-ones if beta = 0 (every thr[m] = 2^32: every proposal is accepted), else 0
    uint32_t hp;                 // head(thr[1]) << 12 | head(thr[2]) (host side: picks a specialised kernel)
    uint32_t stream;             // 1: the records exceed L2, stream the tile bodies (planes_common.cuh: body_policy)
    const uint4* jrec;           // coupling records (a9) or nullptr: per tile, uint4 (cc, gx, Y) =
                                 // {V1, V2, H1, H2}: bit j set <=> the bond from site j of that block to its
                                 // neighbour in the V1 / V2 / H1 / H2 word is J = -1.  Shared by all replicas.
};

// Lattice geometry: run-time fields of the arguments, or compile-time constants when the kernel is specialised at
// run time (planes_jit.cu defines ISING_JIT_B = tiles per side and ISING_JIT_R = replicas).
#ifdef ISING_JIT_B
__device__ __forceinline__ uint32_t geom_B(const PlaneArgs&) { return ISING_JIT_B; }
__device__ __forceinline__ uint32_t geom_R(const PlaneArgs&) { return ISING_JIT_R; }
#else
__device__ __forceinline__ uint32_t geom_B(const PlaneArgs& A) { return (uint32_t)A.B; }
__device__ __forceinline__ uint32_t geom_R(const PlaneArgs& A) { return (uint32_t)A.R; }
#endif

template <int T, int NS = 1>
__device__ __forceinline__ void job_tile(const PlaneArgs& A, uint32_t job, int sub, int& r, int& tx, int& ty, int C = -1) {
    // colour-C tiles enumerated row by row: q -> ty = q / (B/2), tx = 2*(q % (B/2)) + ((ty + C) & 1); a lane with NS slots
    // owns the tiles q, q + 1, ..., q + NS - 1 (same row: (B/2) % NS == 0)
    const uint32_t B = geom_B(A), per_rep = B * B / 2u, hb = B >> 1;
    const uint32_t q = (job * PG<T>::TPW + (uint32_t)sub) * (uint32_t)NS;
#ifdef ISING_JIT_B
    const uint32_t rr = ISING_JIT_R == 1 ? 0u : q / per_rep;      // divisions by constants
    const uint32_t qq = q - rr * per_rep;
    const uint32_t yy = qq / hb;
#else
    const uint32_t rr = fastdiv(q, per_rep, A.magic_rep);
    const uint32_t qq = q - rr * per_rep;
    const uint32_t yy = fastdiv(qq, hb, A.magic_hb);
#endif
    r = (int)rr;
    ty = (int)yy;
    tx = (int)(2u * (qq - yy * hb)) + ((ty + (C < 0 ? A.C : C)) & 1);
}

// Everything a lane keeps of its job between load and store.
template <int T>
struct TileRegs {
    uint32_t S[2][PG<T>::NW];     // S[cc][gx]: the lane's block row, colour cc
    uint32_t vrow[2][PG<T>::NW];  // lane Y = 0: block row above (high half = halo row -1), lane Y = LPT-1: block
                                  // row below (low half = halo row T), by colour; unused on the other lanes
    uint32_t hL0, hL1, hR0, hR1;  // halo column bits: x = -1 / x = T of rows 2Y (0) and 2Y+1 (1)
};

// body_smem != 0: the record body has been staged in shared memory (32-bit shared address of its first byte, same layout)
template <int T, bool BITS>
__device__ __forceinline__ void load_tile(const PlaneArgs& A, int r, int tx, int ty, int Y, int lane_base, TileRegs<T>& t,
                                          uint32_t body_smem = 0) {
    using G = PG<T>;
    constexpr uint32_t REC = BITS ? G::REC_BITS : G::REC_I8;
    constexpr uint32_t BODY = REC - G::EDGE;
    // tile indices in 32 bits, one widening multiply per record address
    const uint32_t B = geom_B(A), utx = (uint32_t)tx, uty = (uint32_t)ty;
    const uint32_t row0 = (uint32_t)r * B * B, rowc = row0 + uty * B;
    const uint32_t tyU = uty == 0 ? B - 1 : uty - 1, tyD = uty == B - 1 ? 0 : uty + 1;
    const uint32_t txL = utx == 0 ? B - 1 : utx - 1, txR = utx == B - 1 ? 0 : utx + 1;
    auto rec_of = [&](uint32_t idx) { return A.tiles + (uint64_t)idx * REC; };
    const uint8_t* rec = rec_of(rowc + utx);
    const uint64_t pol = body_policy(A.stream != 0);
    if (BITS) {
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int gx = 0; gx < G::NW; ++gx)
                t.S[cc][gx] = body_smem ? lds32(body_smem + ((cc * G::NW + gx) * G::LPT + Y) * 4) : ldg32(rec + ((cc * G::NW + gx) * G::LPT + Y) * 4);
    } else {
        uint4 v[G::NCH];
#pragma unroll
        for (int ch = 0; ch < G::NCH; ++ch)
            v[ch] = body_smem ? lds128(body_smem + (ch * G::LPT + Y) * 16) : ldg128(rec + (ch * G::LPT + Y) * 16, pol);
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int gx = 0; gx < G::NW; ++gx)
                t.S[cc][gx] = pack16(pack16(0u, v[(2 + cc) * G::NW + gx]), v[cc * G::NW + gx]);
    }
    // halo rows: the first lane of a tile takes BOT of the tile above, the last lane TOP of the tile below
    uint4 hv = make_uint4(0u, 0u, 0u, 0u);
    if (Y == 0 || Y == G::LPT - 1)
        hv = ldh128(rec_of(row0 + (Y == 0 ? tyU : tyD) * B + utx) + BODY + (Y == 0 ? G::E_BOT : G::E_TOP));
    t.vrow[0][0] = hv.x;
    if (G::NW == 2) { t.vrow[0][1] = hv.y; t.vrow[1][0] = hv.z; t.vrow[1][1] = hv.w; }
    else t.vrow[1][0] = hv.y;
    // halo columns: the left tile's right column, the right tile's left column (same address for every lane of a tile)
    const uint2 cl = ldh64(rec_of(rowc + txL) + BODY + G::E_COL + 8);   // {R0, R1}
    const uint2 cr = ldh64(rec_of(rowc + txR) + BODY + G::E_COL);       // {L0, L1}
    // bit 0 = the halo site of this lane's row; the bits above it (other rows) are never looked at: neighbour_words moves bit 0
    // to the edge of a half-word and everything else out of it
    t.hL0 = cl.x >> Y; t.hL1 = cl.y >> Y;
    t.hR0 = cr.x >> Y; t.hR1 = cr.y >> Y;
    (void)lane_base;
}

// a7: write the lane's block row back, and the bit-packed copies of the tile's boundary (see PG).
// SLUT: the table is a copy in shared memory, lut_smem = its 32-bit shared address (persistent kernels build it once per CTA)
template <int T, bool BITS, bool SLUT = false>
__device__ __forceinline__ void store_tile(const PlaneArgs& A, int r, int tx, int ty, int Y, int sub, const TileRegs<T>& t,
                                           const uint2* lut, uint32_t lut_smem = 0) {
    using G = PG<T>;
    constexpr uint32_t REC = BITS ? G::REC_BITS : G::REC_I8;
    constexpr uint32_t BODY = REC - G::EDGE;
    uint8_t* rec = A.tiles + (uint64_t)(((uint32_t)r * geom_B(A) + (uint32_t)ty) * geom_B(A) + (uint32_t)tx) * REC;
    const uint64_t pol = body_policy(A.stream != 0);
    if (BITS) {
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int gx = 0; gx < G::NW; ++gx)
                *reinterpret_cast<uint32_t*>(rec + ((cc * G::NW + gx) * G::LPT + Y) * 4) = t.S[cc][gx];
    } else {
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int gx = 0; gx < G::NW; ++gx) {
                const uint32_t w = t.S[cc][gx];
#pragma unroll
                for (int rp = 0; rp < 2; ++rp) {
                    uint2 a, b;                                                       // bits 0..7 -> bytes 0..7, bits 8..15 -> bytes 8..15
                    if (SLUT) {
                        a = lds64(lut_smem + (((w >> (16 * rp)) & 0xffu) << 3));
                        b = lds64(lut_smem + (((w >> (16 * rp + 8)) & 0xffu) << 3));
                    } else {
                        a = __ldg(lut + ((w >> (16 * rp)) & 0xffu));
                        b = __ldg(lut + ((w >> (16 * rp + 8)) & 0xffu));
                    }
                    stg128(rec + ((((rp * 2 + cc) * G::NW + gx) * G::LPT) + Y) * 16, make_uint4(a.x, a.y, b.x, b.y), pol);
                }
            }
    }
    // boundary columns: x = 0 is colour 0 on even rows (bit 0) and colour 1 on odd rows (bit 16); x = T-1 is
    // colour 1 / colour 0, last pair.  One ballot each; a warp holds 64 / T tiles, LPT bits per tile.
    // (tile 32: the tile's 16 lanes are one half of the ballot: one byte permute picks it)
    const uint32_t half = sub ? 0x4432u : 0x4410u;
    auto mine = [&](uint32_t ballot) { return G::LPT == 32 ? ballot : __byte_perm(ballot, 0u, half); };
    const uint32_t L0 = mine(__ballot_sync(0xffffffffu, t.S[0][0] & 1u));
    const uint32_t L1 = mine(__ballot_sync(0xffffffffu, (t.S[1][0] >> 16) & 1u));
    const uint32_t R0 = mine(__ballot_sync(0xffffffffu, (t.S[1][G::NW - 1] >> 15) & 1u));
    const uint32_t R1 = mine(__ballot_sync(0xffffffffu, t.S[0][G::NW - 1] >> 31));
    // first lane: TOP + COL (one sector), last lane: BOT + padding (the other sector)
    if (Y == 0 || Y == G::LPT - 1) {
        const uint4 w = G::NW == 2 ? make_uint4(t.S[0][0], t.S[0][1], t.S[1][0], t.S[1][1]) : make_uint4(t.S[0][0], t.S[1][0], 0u, 0u);
        uint8_t* e = rec + BODY + (Y == 0 ? G::E_TOP : G::E_BOT);
        stg128(e, w);
        stg128(e + 16, Y == 0 ? make_uint4(L0, L1, R0, R1) : make_uint4(0u, 0u, 0u, 0u));
    }
}

// R_m = [r < thr[m]] for the 32 sites of block g in half-sweep H: head planes + borrow chains.
// eq_m = sites whose 12 head bits equal the head of thr[m] (their tail decides).
__device__ __forceinline__ void head_masks(const PlaneArgs& A, uint32_t g, uint32_t Hlo, uint32_t Hhi, uint32_t k0,
                                           uint32_t k1, uint32_t& R1, uint32_t& R2, uint32_t& eq1, uint32_t& eq2) {
    uint32_t bw1 = 0, bw2 = 0, ne1 = 0, ne2 = 0;
#pragma unroll
    for (int n = kHeadBits / 4 - 1; n >= 0; --n) {                  // least significant planes first
        const u32x4 o = philox4x32_10(g, kTagPlanes + 256u * n, Hlo, Hhi, k0, k1);
        const uint32_t p[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
        for (int w = 3; w >= 0; --w) {
            const int q = 4 * n + w;
            bw1 = lop3<kLutChain>(p[w], bw1, A.u1[q]);
            bw2 = lop3<kLutChain>(p[w], bw2, A.u2[q]);
            ne1 = lop3<kLutNe>(ne1, p[w], A.u1[q]);
            ne2 = lop3<kLutNe>(ne2, p[w], A.u2[q]);
        }
    }
    R1 = bw1; R2 = bw2; eq1 = ~ne1; eq2 = ~ne2;
}

// ---- head compare specialised on the head bits of the two thresholds (HP = head(thr[1]) << 12 | head(thr[2])).
// Each site needs one threshold only (n_dis = 1: thr[1], n_dis = 0: thr[2]); with the head bits known at compile
// time the per-site choice folds into the LOP3 immediates: one borrow chain and one tie accumulator (2 LOP3 per
// plane instead of 4), third input = sel (sites that use thr[2]).
constexpr uint32_t kNoSpec = 0xffffffffu;
__host__ __device__ constexpr int lut_chain_sel(int u1, int u2) {        // inputs a = p, b = bw, c = sel
    int l = 0;
    for (int i = 0; i < 8; ++i) {
        const int p = (i >> 2) & 1, bw = (i >> 1) & 1, sel = i & 1, u = sel ? u2 : u1;
        l |= (((!p) && u) || ((p == u) && bw)) << i;
    }
    return l;
}
__host__ __device__ constexpr int lut_ne_sel(int u1, int u2) {           // inputs a = ne, b = p, c = sel
    int l = 0;
    for (int i = 0; i < 8; ++i) {
        const int ne = (i >> 2) & 1, p = (i >> 1) & 1, sel = i & 1, u = sel ? u2 : u1;
        l |= (ne || (p != u)) << i;
    }
    return l;
}
template <uint32_t HP, int Q>
struct HeadBit {                                   // head bit of plane Q (0 = most significant) of thr[1] / thr[2]
    static constexpr int u1 = (HP >> (12 + 11 - Q)) & 1, u2 = (HP >> (11 - Q)) & 1;
    static constexpr bool same = u1 == u2;         // the site's choice of threshold does not matter for this plane
};
// Two adjacent planes whose head bits do not depend on the choice: one LOP3 advances the borrow chain by both
// (inputs a = p_Q, the less significant plane, b = p_(Q-1), c = bw), and one LOP3 accumulates both "differs" bits.
__host__ __device__ constexpr int lut_chain_pair(int uq, int uq1) {
    int l = 0;
    for (int i = 0; i < 8; ++i) {
        const int pq = (i >> 2) & 1, pq1 = (i >> 1) & 1, bw = i & 1;
        const int b1 = ((!pq) && uq) || ((pq == uq) && bw);            // after plane Q
        const int b2 = ((!pq1) && uq1) || ((pq1 == uq1) && b1);        // after plane Q-1
        l |= b2 << i;
    }
    return l;
}
__host__ __device__ constexpr int lut_ne_pair(int ua, int ub) {          // inputs a = ne, b = p_a, c = p_b
    int l = 0;
    for (int i = 0; i < 8; ++i) {
        const int ne = (i >> 2) & 1, pa = (i >> 1) & 1, pb = i & 1;
        l |= (ne || (pa != ua) || (pb != ub)) << i;
    }
    return l;
}
// borrow chain from plane Q down to plane 0 (least significant plane first: Q = 11)
template <uint32_t HP, int Q>
__device__ __forceinline__ void chain_from(const uint32_t (&p)[kHeadBits], uint32_t sel, uint32_t& bw) {
    if constexpr (Q >= 0) {
        if constexpr (Q >= 1 && HeadBit<HP, Q>::same && HeadBit<HP, (Q >= 1 ? Q - 1 : 0)>::same) {
            bw = lop3<lut_chain_pair(HeadBit<HP, Q>::u1, HeadBit<HP, Q - 1>::u1)>(p[Q], p[Q - 1], bw);
            chain_from<HP, Q - 2>(p, sel, bw);
        } else {
            bw = lop3<lut_chain_sel(HeadBit<HP, Q>::u1, HeadBit<HP, Q>::u2)>(p[Q], bw, sel);
            chain_from<HP, Q - 1>(p, sel, bw);
        }
    }
}
// "some head bit differs from the threshold's": planes whose bit depends on the choice one by one, the others two at a
// time (PEND = a choice-independent plane waiting for a partner, or -1)
template <uint32_t HP, int Q, int PEND>
__device__ __forceinline__ void ne_from(const uint32_t (&p)[kHeadBits], uint32_t sel, uint32_t& ne) {
    if constexpr (Q >= 0) {
        if constexpr (!HeadBit<HP, Q>::same) {
            ne = lop3<lut_ne_sel(HeadBit<HP, Q>::u1, HeadBit<HP, Q>::u2)>(ne, p[Q], sel);
            ne_from<HP, Q - 1, PEND>(p, sel, ne);
        } else if constexpr (PEND < 0) {
            ne_from<HP, Q - 1, Q>(p, sel, ne);
        } else {
            ne = lop3<lut_ne_pair(HeadBit<HP, (PEND >= 0 ? PEND : 0)>::u1, HeadBit<HP, Q>::u1)>(ne, p[PEND >= 0 ? PEND : 0], p[Q]);
            ne_from<HP, Q - 1, -1>(p, sel, ne);
        }
    } else if constexpr (PEND >= 0) {
        ne = lop3<lut_ne_pair(HeadBit<HP, (PEND >= 0 ? PEND : 0)>::u1, HeadBit<HP, (PEND >= 0 ? PEND : 0)>::u1)>(ne, p[PEND >= 0 ? PEND : 0], p[PEND >= 0 ? PEND : 0]);
    }
}
template <uint32_t HP>
__device__ __forceinline__ void head_masks_sel(uint32_t g, uint32_t Hlo, uint32_t Hhi, uint32_t k0, uint32_t k1, uint32_t sel,
                                               uint32_t& R, uint32_t& eq) {
    static_assert(kHeadBits == 12, "three Philox calls");
    uint32_t p[kHeadBits];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        const u32x4 o = philox4x32_10(g, kTagPlanes + 256u * n, Hlo, Hhi, k0, k1);
        p[4 * n] = o.x; p[4 * n + 1] = o.y; p[4 * n + 2] = o.z; p[4 * n + 3] = o.w;
    }
    uint32_t bw = 0, ne = 0;
    chain_from<HP, kHeadBits - 1>(p, sel, bw);
    ne_from<HP, kHeadBits - 1, -1>(p, sel, ne);
    R = bw; eq = ~ne;
}

// a4-a5 for one block: S' = S ^ flip, neighbours V1, V2 (vertical), H1, H2 (horizontal) of the other colour.
// und selects the (rare) sites whose tail must be drawn; p_base = pair index i>>1 of bit 0, row stride L/2.
template <bool HASJ, uint32_t HP>
__device__ __forceinline__ uint32_t update_block(const PlaneArgs& A, uint32_t S, uint32_t V1, uint32_t V2, uint32_t H1,
                                                 uint32_t H2, const uint4& Jw, uint32_t g, uint32_t p_base, uint32_t prow,
                                                 uint32_t Hlo, uint32_t Hhi, uint32_t k0, uint32_t k1) {
    // unsatisfied bonds: J s_i s_j = -1  <=>  s_i != s_j for J = +1, s_i == s_j for J = -1 (eq. (1))
    const uint32_t a = S ^ V1 ^ (HASJ ? Jw.x : 0u), b = S ^ V2 ^ (HASJ ? Jw.y : 0u);
    const uint32_t c = S ^ H1 ^ (HASJ ? Jw.z : 0u), d = S ^ H2 ^ (HASJ ? Jw.w : 0u);
    const uint32_t p1 = a | b, q1 = a & b, p2 = c | d, q2 = c & d;
    const uint32_t ge1 = p1 | p2;                                     // n_dis >= 1
    // n_dis >= 2  <=>  dE <= 0: always flip (eq. (2)); beta = 0 (force) never meets a specialised kernel
    const uint32_t ge2 = (p1 & p2) | q1 | q2 | (HP == kNoSpec ? A.force : 0u);
    if (HP != kNoSpec) {
        const uint32_t sel = ~ge1;                                    // n_dis == 0: the site is compared with thr[2]
        uint32_t R, eq;
        head_masks_sel<HP>(g, Hlo, Hhi, k0, k1, sel, R, eq);
        uint32_t und = eq & ~ge2;
        while (und) {                                                 // probability 2^-12 per site
            const int j = __ffs(und) - 1;
            und &= und - 1;
            const uint32_t p = p_base + (uint32_t)(j >> 4) * prow + (uint32_t)(j & 15);
            const u32x4 o = philox4x32_10(p, kTagTail, Hlo, Hhi, k0, k1);
            R |= (uint32_t)((o.x >> kHeadBits) < (((sel >> j) & 1u) ? A.t2_tail : A.t1_tail)) << j;
        }
        return S ^ (ge2 | R);
    }
    uint32_t R1, R2, eq1, eq2;
    head_masks(A, g, Hlo, Hhi, k0, k1, R1, R2, eq1, eq2);
    uint32_t und = (eq1 & ge1 & ~ge2) | (eq2 & ~ge1);                 // n_dis == 1 needs thr[1], n_dis == 0 needs thr[2]
    while (und) {                                                     // probability 2^-12 per site
        const int j = __ffs(und) - 1;
        und &= und - 1;
        const uint32_t p = p_base + (uint32_t)(j >> 4) * prow + (uint32_t)(j & 15);
        const u32x4 o = philox4x32_10(p, kTagTail, Hlo, Hhi, k0, k1);
        const uint32_t tail = o.x >> kHeadBits;
        if ((eq1 >> j) & 1u) R1 |= (uint32_t)(tail < A.t1_tail) << j;
        if ((eq2 >> j) & 1u) R2 |= (uint32_t)(tail < A.t2_tail) << j;
    }
    const uint32_t flip = ge2 | (ge1 & R1) | R2;                      // thr[2] <= thr[1], so R2 is inside R1
    return S ^ flip;
}

// a5-a6: one half-sweep of colour c on the lane's block row; o = 1 - c is read, c is written.
// The four neighbour words of the lane's block (c, gx): V1 = other row of the block, V2 = the rows outside it
// (shuffle; halo rows on the tile's first / last lane), H1 = same pairs, H2 = pairs shifted by one with carries
// from the adjacent block or the halo column.  PERIODIC: the tile is the whole lattice (T = L, the plain
// checkerboard of P:62): "halos" are the tile's own, live, opposite edges.
template <int T, bool PERIODIC>
__device__ __forceinline__ void neighbour_words(const TileRegs<T>& t, int c, int gx, int Y, uint32_t& V1, uint32_t& V2,
                                                uint32_t& H1, uint32_t& H2) {
    using G = PG<T>;
    const int o = 1 - c;
    const uint32_t O = t.S[o][gx], Ol = t.S[o][(gx + G::NW - 1) % G::NW], Or = t.S[o][(gx + 1) % G::NW];
    uint32_t Oup, Odn;
    if (PERIODIC) {
        Oup = __shfl_sync(0xffffffffu, O, (Y + G::LPT - 1) % G::LPT);
        Odn = __shfl_sync(0xffffffffu, O, (Y + 1) % G::LPT);
    } else {
        Oup = __shfl_up_sync(0xffffffffu, O, 1);
        Odn = __shfl_down_sync(0xffffffffu, O, 1);
        if (Y == 0) Oup = t.vrow[o][gx];
        if (Y == G::LPT - 1) Odn = t.vrow[o][gx];
    }
    V1 = __byte_perm(O, O, 0x1032);               // the other row of the same block
    V2 = __byte_perm(Oup, Odn, 0x5432);           // row above the block | row below the block
    H1 = O;
    // pair-shifted word: colour 0: even rows (low half) look at pair j-1, odd rows (high half) at pair j+1; colour 1 the
    // other way round.  A half shifted by one pair with the carry from the adjacent word (or the halo column) is 16
    // consecutive bits of a 32-bit word glued from the two halves involved: one byte permute + one shift each.
    //   "pair j-1" of half X with left neighbour half Lh:  bits [30:15] of (X << 16 | Lh)
    //   "pair j+1" of half X with right neighbour half Rh: bits [16:1]  of (Rh << 16 | X)
    if (c == 0) {
        const uint32_t lf = (gx == 0 && !PERIODIC) ? (t.hL0 << 15) : Ol;                 // low half: its bit 15 is the carry in
        const uint32_t rt = (gx == G::NW - 1 && !PERIODIC) ? (t.hR1 << 16) : Or;         // high half: its bit 16 is the carry in
        const uint32_t lo = __byte_perm(lf, O, 0x5410) >> 15;                            // (O.lo16 << 16 | lf.lo16) >> 15: result in bits [15:0]
        const uint32_t hi = __byte_perm(O, rt, 0x7632) << 15;                            // (rt.hi16 << 16 | O.hi16) << 15: result in bits [31:16]
        H2 = (lo & 0x0000ffffu) | (hi & 0xffff0000u);
    } else {
        const uint32_t rt = (gx == G::NW - 1 && !PERIODIC) ? t.hR0 : Or;                 // low half looks right: carry = bit 0 of the right word's low half
        const uint32_t lf = (gx == 0 && !PERIODIC) ? (t.hL1 << 31) : Ol;                 // high half looks left: carry = bit 31 of the left word
        const uint32_t lo = __byte_perm(O, rt, 0x5410) >> 1;                             // (rt.lo16 << 16 | O.lo16) >> 1
        const uint32_t hi = __byte_perm(lf, O, 0x7632) << 1;                             // (O.hi16 << 16 | lf.hi16) << 1
        H2 = (lo & 0x0000ffffu) | (hi & 0xffff0000u);
    }
}

// a5-a6: one half-sweep of colour c on the lane's block row; o = 1 - c is read, c is written.
template <int T, bool HASJ, bool PERIODIC = false, uint32_t HP = kNoSpec>
__device__ __forceinline__ void half_sweep(const PlaneArgs& A, TileRegs<T>& t, const uint4 (&Jw)[2][PG<T>::NW], int c, int Y,
                                           uint32_t g0, uint32_t p0, uint64_t H, uint32_t k0, uint32_t k1) {
    using G = PG<T>;
    const uint32_t Hlo = (uint32_t)H, Hhi = (uint32_t)(H >> 32);
    uint32_t Snew[G::NW];
#pragma unroll
    for (int gx = 0; gx < G::NW; ++gx) {
        uint32_t V1, V2, H1, H2;
        neighbour_words<T, PERIODIC>(t, c, gx, Y, V1, V2, H1, H2);
        Snew[gx] = update_block<HASJ, HP>(A, t.S[c][gx], V1, V2, H1, H2, Jw[c][gx], g0 + (uint32_t)gx,
                                          p0 + 16u * (uint32_t)gx, geom_B(A) * (uint32_t)(T / 2), Hlo, Hhi, k0, k1);
    }
#pragma unroll
    for (int gx = 0; gx < G::NW; ++gx) t.S[c][gx] = Snew[gx];
}

// a10 on a tile held in registers: #up spins and #unsatisfied bonds of the lane's block row, every bond of the
// tile's colour-0 sites (each bond of the lattice has exactly one colour-0 end).  M = 2 #up - N, E = 2 #unsat - 2N.
template <int T, bool PERIODIC>
__device__ __forceinline__ void count_row(const TileRegs<T>& t, const uint4 (&Jw)[2][PG<T>::NW], int Y, int& up, int& unsat) {
    using G = PG<T>;
#pragma unroll
    for (int gx = 0; gx < G::NW; ++gx) {
        uint32_t V1, V2, H1, H2;
        neighbour_words<T, PERIODIC>(t, 0, gx, Y, V1, V2, H1, H2);
        const uint32_t S = t.S[0][gx];
        const uint4 Jc = Jw[0][gx];
        unsat += __popc(S ^ V1 ^ Jc.x) + __popc(S ^ V2 ^ Jc.y) + __popc(S ^ H1 ^ Jc.z) + __popc(S ^ H2 ^ Jc.w);
        up += __popc(S) + __popc(t.S[1][gx]);
    }
}

constexpr int kPlaneThreads = 128;      // 4 warps = 4 jobs per CTA

// NS = tiles per lane ("slots"): the lane's tiles are NS consecutive tiles of the colour in one tile row, (tx + 2s, ty), so
// the job's set-up (tile coordinates, record addresses, key schedule, the ballots of the boundary columns) is paid once per
// NS tiles — what makes tile 32 as cheap per site as tile 64 ("missing" 1).  Needs (B/2) % NS == 0.
template <int T, bool BITS, bool HASJ, uint32_t HP = kNoSpec, int NS = 1>
__global__ void __launch_bounds__(kPlaneThreads) k_tile_planes(PlaneArgs A) {
    using G = PG<T>;
    // int8 write-back table (8 bits -> 8 bytes of 0/1): a constant array in global memory read through the
    // read-only path (2 KB, L1-resident) — no per-CTA build, no barrier (measured +6 % at k = 1 over a shared-memory copy).
    const uint2* lut = kByteLutGlobal.e;
    // Programmatic dependent launch: the next colour's grid may be scheduled while this one drains; it
    // waits here until every store of the previous launch is visible.
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int lane = threadIdx.x & 31;
    const uint32_t job = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (job >= A.njobs) return;
    const int sub = lane / G::LPT, Y = lane % G::LPT;
    int r, tx0, ty;
    job_tile<T, NS>(A, job, sub, r, tx0, ty);
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
                Jw[s][cc][gx] = HASJ ? __ldg(A.jrec + ((size_t)ty * geom_B(A) + tx) * (2 * G::NW * G::LPT) + (cc * G::NW + gx) * G::LPT + Y)
                                     : make_uint4(0u, 0u, 0u, 0u);
    }
#if defined(ISING_JIT_R) && ISING_JIT_R == 1
    const uint64_t seed = A.seed0;
#else
    const uint64_t seed = A.seeds[r];
#endif
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    const uint32_t Yg = (uint32_t)(ty * G::LPT + Y);                         // global block row
    const uint32_t g0 = Yg * (geom_B(A) * G::NW) + (uint32_t)(tx0 * G::NW);  // RNG block of gx = 0 (L / 32 blocks per row)
    const uint32_t p0 = 2u * Yg * (geom_B(A) * (uint32_t)(T / 2)) + 16u * (uint32_t)(tx0 * G::NW);   // pair index of its bit 0
    for (int j = 0; j < A.k; ++j) {
        const uint64_t tt = A.t_first + (uint64_t)j;
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int s = 0; s < NS; ++s)
                half_sweep<T, HASJ, false, HP>(A, t[s], Jw[s], c, Y, g0 + (uint32_t)(2 * s * G::NW), p0 + 32u * (uint32_t)(s * G::NW), 2 * tt + (uint64_t)c, k0, k1);
    }
#pragma unroll
    for (int s = 0; s < NS; ++s) store_tile<T, BITS>(A, r, tx0 + 2 * s, ty, Y, sub, t[s], lut);
}


}  // namespace

}  // namespace ising
