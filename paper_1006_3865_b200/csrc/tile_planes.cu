// tile_planes.cu — the 2D double-checkerboard tile kernel in multi-spin (bit-plane) form,
// RNG mapping "planes" (DESIGN.md §3 R6, §5, §6).  Steps a1, a3-a7 of SURVEY §8(a).
//
// Arithmetic form.  A 32-bit word holds the 32 same-colour sites of one RNG block: 16 pairs
// p_x x 2 rows, bit j = (y & 1) * 16 + (p_x & 15).  For a half-sweep of colour c the four
// neighbours of all 32 sites are four words of the other colour (same block; same block with
// its halves swapped; the blocks above/below; the block shifted by one pair), so
//   disagreement masks, a 4-input bit adder, and
//   flip = [n_dis >= 2] | [n_dis >= 1] & R1 | R2,    R_m = [r < thr[m]] per site
// cost ~10 LOP3 per 32 sites.  R_m comes from the 12 head planes of the block (3 Philox calls)
// by a bit-serial borrow chain against the head bits of thr[m] (uniform operands), LSB plane
// first; a site whose head equals the head of a threshold it needs (probability 2^-12) draws its
// 20 tail bits from the per-site call.  Everything runs in registers: a warp owns 64 tile rows
// (one 64x64 tile or two 32x32 tiles), lane = block row, vertical neighbours come by shuffle,
// the k inner sweeps never touch memory.
//
// HBM layouts (tile records; PG below):
//   int8  record = T*T body + 64 edge bytes, 0/1 per spin.  Body is piece-major: the 16 bytes
//         (row 2Y+rp, colour cc, pairs 16gx..16gx+15) sit at ((rp*2+cc)*NW+gx)*LPT*16 + Y*16, so lane Y
//         loads its 4*NW pieces with fully coalesced 128-bit accesses and no shared-memory staging.
//   bits  record = T*T/8 body + 64 edge bytes: word (cc, Y, gx) at ((cc*NW+gx)*LPT + Y)*4.
//   edge  = bit-packed copies of the tile's own first / last block row and first / last column, written by
//         the tile, so that every halo is one 16-byte run of ready-made words in the neighbour's record.
#include "kernels.h"
#include "planes_common.cuh"

namespace ising {

namespace {

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
    uint32_t stream;             // 1: the records exceed L2, stream the tile bodies (planes_common.cuh: body_policy)
    const uint4* jrec;           // coupling records (a9) or nullptr: per tile, uint4 (cc, gx, Y) =
                                 // {V1, V2, H1, H2}: bit j set <=> the bond from site j of that block to its
                                 // neighbour in the V1 / V2 / H1 / H2 word is J = -1.  Shared by all replicas.
};

template <int T>
__device__ __forceinline__ void job_tile(const PlaneArgs& A, uint32_t job, int sub, int& r, int& tx, int& ty) {
    // colour-C tiles enumerated row by row: q -> ty = q / (B/2), tx = 2*(q % (B/2)) + ((ty + C) & 1)
    const uint32_t per_rep = (uint32_t)A.B * (uint32_t)A.B / 2u;
    const uint32_t q = job * PG<T>::TPW + (uint32_t)sub;
    const uint32_t rr = fastdiv(q, per_rep, A.magic_rep);
    r = (int)rr;
    const uint32_t qq = q - rr * per_rep;
    const uint32_t hb = (uint32_t)A.B >> 1;
    ty = (int)fastdiv(qq, hb, A.magic_hb);
    tx = (int)(2u * (qq - (uint32_t)ty * hb)) + ((ty + A.C) & 1);
}

// Everything a lane keeps of its job between load and store.
template <int T>
struct TileRegs {
    uint32_t S[2][PG<T>::NW];     // S[cc][gx]: the lane's block row, colour cc
    uint32_t vrow[2][PG<T>::NW];  // lane Y = 0: block row above (high half = halo row -1), lane Y = LPT-1: block
                                  // row below (low half = halo row T), by colour; unused on the other lanes
    uint32_t hL0, hL1, hR0, hR1;  // halo column bits: x = -1 / x = T of rows 2Y (0) and 2Y+1 (1)
};

template <int T, bool BITS>
__device__ __forceinline__ void load_tile(const PlaneArgs& A, int r, int tx, int ty, int Y, int lane_base, TileRegs<T>& t) {
    using G = PG<T>;
    constexpr uint32_t REC = BITS ? G::REC_BITS : G::REC_I8;
    constexpr uint32_t BODY = REC - G::EDGE;
    // tile indices in 32 bits, one widening multiply per record address
    const uint32_t B = (uint32_t)A.B, utx = (uint32_t)tx, uty = (uint32_t)ty;
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
            for (int gx = 0; gx < G::NW; ++gx) t.S[cc][gx] = ldg32(rec + ((cc * G::NW + gx) * G::LPT + Y) * 4);
    } else {
        uint4 v[G::NCH];
#pragma unroll
        for (int ch = 0; ch < G::NCH; ++ch) v[ch] = ldg128(rec + (ch * G::LPT + Y) * 16, pol);
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int gx = 0; gx < G::NW; ++gx)
                t.S[cc][gx] = pack16(pack16(0u, v[(2 + cc) * G::NW + gx]), v[cc * G::NW + gx]);
    }
    // halo rows: the first lane of a tile takes BOT of the tile above, the last lane TOP of the tile below
    uint4 hv = make_uint4(0u, 0u, 0u, 0u);
    if (Y == 0 || Y == G::LPT - 1)
        hv = __ldg(reinterpret_cast<const uint4*>(rec_of(row0 + (Y == 0 ? tyU : tyD) * B + utx) + BODY + (Y == 0 ? G::E_BOT : G::E_TOP)));
    t.vrow[0][0] = hv.x;
    if (G::NW == 2) { t.vrow[0][1] = hv.y; t.vrow[1][0] = hv.z; t.vrow[1][1] = hv.w; }
    else t.vrow[1][0] = hv.y;
    // halo columns: the left tile's right column, the right tile's left column (same address for every lane of a tile)
    const uint2 cl = __ldg(reinterpret_cast<const uint2*>(rec_of(rowc + txL) + BODY + G::E_COL + 8));   // {R0, R1}
    const uint2 cr = __ldg(reinterpret_cast<const uint2*>(rec_of(rowc + txR) + BODY + G::E_COL));       // {L0, L1}
    t.hL0 = (cl.x >> Y) & 1u; t.hL1 = (cl.y >> Y) & 1u;
    t.hR0 = (cr.x >> Y) & 1u; t.hR1 = (cr.y >> Y) & 1u;
    (void)lane_base;
}

// a7: write the lane's block row back, and the bit-packed copies of the tile's boundary (see PG).
template <int T, bool BITS>
__device__ __forceinline__ void store_tile(const PlaneArgs& A, int r, int tx, int ty, int Y, int sub, const TileRegs<T>& t,
                                           const uint2* lut) {
    using G = PG<T>;
    constexpr uint32_t REC = BITS ? G::REC_BITS : G::REC_I8;
    constexpr uint32_t BODY = REC - G::EDGE;
    uint8_t* rec = A.tiles + (uint64_t)(((uint32_t)r * (uint32_t)A.B + (uint32_t)ty) * (uint32_t)A.B + (uint32_t)tx) * REC;
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
                    const uint2 a = __ldg(lut + ((w >> (16 * rp)) & 0xffu));          // bits 0..7  -> bytes 0..7
                    const uint2 b = __ldg(lut + ((w >> (16 * rp + 8)) & 0xffu));      // bits 8..15 -> bytes 8..15
                    stg128(rec + ((((rp * 2 + cc) * G::NW + gx) * G::LPT) + Y) * 16, make_uint4(a.x, a.y, b.x, b.y), pol);
                }
            }
    }
    // boundary columns: x = 0 is colour 0 on even rows (bit 0) and colour 1 on odd rows (bit 16); x = T-1 is
    // colour 1 / colour 0, last pair.  One ballot each; a warp holds 64 / T tiles, LPT bits per tile.
    const uint32_t sh = (uint32_t)sub * G::LPT, m = G::LPT == 32 ? 0xffffffffu : ((1u << G::LPT) - 1u);
    const uint32_t L0 = (__ballot_sync(0xffffffffu, t.S[0][0] & 1u) >> sh) & m;
    const uint32_t L1 = (__ballot_sync(0xffffffffu, (t.S[1][0] >> 16) & 1u) >> sh) & m;
    const uint32_t R0 = (__ballot_sync(0xffffffffu, (t.S[1][G::NW - 1] >> 15) & 1u) >> sh) & m;
    const uint32_t R1 = (__ballot_sync(0xffffffffu, t.S[0][G::NW - 1] >> 31) >> sh) & m;
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

// a4-a5 for one block: S' = S ^ flip, neighbours V1, V2 (vertical), H1, H2 (horizontal) of the other colour.
// und selects the (rare) sites whose tail must be drawn; p_base = pair index i>>1 of bit 0, row stride L/2.
template <bool HASJ>
__device__ __forceinline__ uint32_t update_block(const PlaneArgs& A, uint32_t S, uint32_t V1, uint32_t V2, uint32_t H1,
                                                 uint32_t H2, const uint4& Jw, uint32_t g, uint32_t p_base, uint32_t Hlo,
                                                 uint32_t Hhi, uint32_t k0, uint32_t k1) {
    uint32_t R1, R2, eq1, eq2;
    head_masks(A, g, Hlo, Hhi, k0, k1, R1, R2, eq1, eq2);
    // unsatisfied bonds: J s_i s_j = -1  <=>  s_i != s_j for J = +1, s_i == s_j for J = -1 (eq. (1))
    const uint32_t a = S ^ V1 ^ (HASJ ? Jw.x : 0u), b = S ^ V2 ^ (HASJ ? Jw.y : 0u);
    const uint32_t c = S ^ H1 ^ (HASJ ? Jw.z : 0u), d = S ^ H2 ^ (HASJ ? Jw.w : 0u);
    const uint32_t p1 = a | b, q1 = a & b, p2 = c | d, q2 = c & d;
    const uint32_t ge1 = p1 | p2;                                     // n_dis >= 1
    const uint32_t ge2 = (p1 & p2) | q1 | q2 | A.force;               // n_dis >= 2  <=>  dE <= 0: always flip (eq. (2))
    uint32_t und = (eq1 & ge1 & ~ge2) | (eq2 & ~ge1);                 // n_dis == 1 needs thr[1], n_dis == 0 needs thr[2]
    while (und) {                                                     // probability 2^-12 per site
        const int j = __ffs(und) - 1;
        und &= und - 1;
        const uint32_t p = p_base + (uint32_t)(j >> 4) * (uint32_t)(A.L >> 1) + (uint32_t)(j & 15);
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
    // pair-shifted word: colour 0: even rows look at pair j-1 (carry from the left), odd rows at j+1;
    // colour 1: even rows j+1, odd rows j-1.
    if (c == 0) {
        const uint32_t cl = (gx == 0 && !PERIODIC) ? t.hL0 : ((Ol >> 15) & 1u);
        const uint32_t cr = (gx == G::NW - 1 && !PERIODIC) ? t.hR1 : ((Or >> 16) & 1u);
        H2 = ((O << 1) & 0x0000fffeu) | cl | ((O >> 1) & 0x7fff0000u) | (cr << 31);
    } else {
        const uint32_t cr = (gx == G::NW - 1 && !PERIODIC) ? t.hR0 : (Or & 1u);
        const uint32_t cl = (gx == 0 && !PERIODIC) ? t.hL1 : (Ol >> 31);
        H2 = ((O >> 1) & 0x00007fffu) | (cr << 15) | ((O << 1) & 0xfffe0000u) | (cl << 16);
    }
}

// a5-a6: one half-sweep of colour c on the lane's block row; o = 1 - c is read, c is written.
template <int T, bool HASJ, bool PERIODIC = false>
__device__ __forceinline__ void half_sweep(const PlaneArgs& A, TileRegs<T>& t, const uint4 (&Jw)[2][PG<T>::NW], int c, int Y,
                                           uint32_t g0, uint32_t p0, uint64_t H, uint32_t k0, uint32_t k1) {
    using G = PG<T>;
    const uint32_t Hlo = (uint32_t)H, Hhi = (uint32_t)(H >> 32);
    uint32_t Snew[G::NW];
#pragma unroll
    for (int gx = 0; gx < G::NW; ++gx) {
        uint32_t V1, V2, H1, H2;
        neighbour_words<T, PERIODIC>(t, c, gx, Y, V1, V2, H1, H2);
        Snew[gx] = update_block<HASJ>(A, t.S[c][gx], V1, V2, H1, H2, Jw[c][gx], g0 + (uint32_t)gx,
                                      p0 + 16u * (uint32_t)gx, Hlo, Hhi, k0, k1);
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

template <int T, bool BITS, bool HASJ>
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
    int r, tx, ty;
    job_tile<T>(A, job, sub, r, tx, ty);
    TileRegs<T> t;
    load_tile<T, BITS>(A, r, tx, ty, Y, sub * G::LPT, t);
    uint4 Jw[2][G::NW];
#pragma unroll
    for (int cc = 0; cc < 2; ++cc)
#pragma unroll
        for (int gx = 0; gx < G::NW; ++gx)
            Jw[cc][gx] = HASJ ? __ldg(A.jrec + ((size_t)ty * A.B + tx) * (2 * G::NW * G::LPT) + (cc * G::NW + gx) * G::LPT + Y)
                              : make_uint4(0u, 0u, 0u, 0u);
    const uint64_t seed = A.seeds[r];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    const uint32_t Yg = (uint32_t)(ty * G::LPT + Y);                         // global block row
    const uint32_t g0 = Yg * (uint32_t)(A.L >> 5) + (uint32_t)(tx * G::NW);  // RNG block of gx = 0
    const uint32_t p0 = 2u * Yg * (uint32_t)(A.L >> 1) + 16u * (uint32_t)(tx * G::NW);   // pair index of its bit 0
    for (int j = 0; j < A.k; ++j) {
        const uint64_t tt = A.t_first + (uint64_t)j;
        half_sweep<T, HASJ>(A, t, Jw, 0, Y, g0, p0, 2 * tt, k0, k1);
        half_sweep<T, HASJ>(A, t, Jw, 1, Y, g0, p0, 2 * tt + 1, k0, k1);
    }
    store_tile<T, BITS>(A, r, tx, ty, Y, sub, t, lut);
}

// a8: plain checkerboard of a 64x64 lattice (tile = L = 64, BASELINE config 1).  One warp holds a whole
// replica in registers and runs all n passes of the call in one launch; E and M after every pass (a10) come
// from popcounts: M = 2*#up - N, E = -(2N - 2*#unsatisfied bonds), every bond seen once from its colour-0 end.
template <bool BITS, bool HASJ>
__global__ void __launch_bounds__(32) k_plain64_planes(PlaneArgs A, int n, long long* __restrict__ E, long long* __restrict__ M) {
    constexpr int T = 64;
    using G = PG<T>;
    const uint2* lut = kByteLutGlobal.e;
    const int Y = threadIdx.x, r = blockIdx.x;
    TileRegs<T> t;
    load_tile<T, BITS>(A, r, 0, 0, Y, 0, t);
    uint4 Jw[2][G::NW];
#pragma unroll
    for (int cc = 0; cc < 2; ++cc)
#pragma unroll
        for (int gx = 0; gx < G::NW; ++gx)
            Jw[cc][gx] = HASJ ? __ldg(A.jrec + (cc * G::NW + gx) * G::LPT + Y) : make_uint4(0u, 0u, 0u, 0u);
    const uint64_t seed = A.seeds[r];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    const uint32_t g0 = (uint32_t)Y * G::NW, p0 = 2u * (uint32_t)Y * (T / 2);
    for (int pass = 0; pass < n; ++pass) {
        for (int j = 0; j < A.k; ++j) {
            const uint64_t tt = A.t_first + (uint64_t)pass * (uint64_t)A.k + (uint64_t)j;
            half_sweep<T, HASJ, true>(A, t, Jw, 0, Y, g0, p0, 2 * tt, k0, k1);
            half_sweep<T, HASJ, true>(A, t, Jw, 1, Y, g0, p0, 2 * tt + 1, k0, k1);
        }
        if (E || M) {
            int up = 0, unsat = 0;
            count_row<T, true>(t, Jw, Y, up, unsat);
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                up += __shfl_xor_sync(0xffffffffu, up, d);
                unsat += __shfl_xor_sync(0xffffffffu, unsat, d);
            }
            if (Y == 0) {
                if (M) M[(size_t)pass * A.R + r] = 2ll * up - (long long)(T * T);
                if (E) E[(size_t)pass * A.R + r] = 2ll * unsat - 2ll * (T * T);
            }
        }
    }
    store_tile<T, BITS>(A, r, 0, 0, Y, 0, t, lut);
}

// a10 directly on the tile records (no conversion to the canonical array): one launch per coarse colour C adds
// the colour-C tiles' share to E[r], M[r] (zeroed by the caller): warp shuffle reduction, two 64-bit atomics per tile.
template <int T, bool BITS, bool HASJ>
__global__ void __launch_bounds__(kPlaneThreads) k_observables_planes(PlaneArgs A, long long* __restrict__ E, long long* __restrict__ M) {
    using G = PG<T>;
    const int lane = threadIdx.x & 31;
    const uint32_t job = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (job >= A.njobs) return;
    const int sub = lane / G::LPT, Y = lane % G::LPT;
    int r, tx, ty;
    job_tile<T>(A, job, sub, r, tx, ty);
    TileRegs<T> t;
    load_tile<T, BITS>(A, r, tx, ty, Y, sub * G::LPT, t);
    uint4 Jw[2][G::NW];
#pragma unroll
    for (int cc = 0; cc < 2; ++cc)
#pragma unroll
        for (int gx = 0; gx < G::NW; ++gx)
            Jw[cc][gx] = HASJ ? __ldg(A.jrec + ((size_t)ty * A.B + tx) * (2 * G::NW * G::LPT) + (cc * G::NW + gx) * G::LPT + Y)
                              : make_uint4(0u, 0u, 0u, 0u);
    int up = 0, unsat = 0;
    count_row<T, false>(t, Jw, Y, up, unsat);
#pragma unroll
    for (int d = G::LPT / 2; d > 0; d >>= 1) {           // reduce over the lanes of one tile
        up += __shfl_xor_sync(0xffffffffu, up, d);
        unsat += __shfl_xor_sync(0xffffffffu, unsat, d);
    }
    if (Y == 0) {
        if (M) atomicAdd(reinterpret_cast<unsigned long long*>(M + r), (unsigned long long)(2ll * up - (long long)(T * T)));
        if (E) atomicAdd(reinterpret_cast<unsigned long long*>(E + r), (unsigned long long)(2ll * unsat - 2ll * (T * T)));
    }
}

// ---- layout converters (a11): canonical int8 +-1 <-> tile records; not on the timed path ----
// One thread per site; MODE 0: canonical -> int8 records, 1: int8 records -> canonical,
// 2: canonical -> bit records, 3: bit records -> canonical.  Bit fields are set by atomicOr into zeroed storage.
template <int MODE>
__global__ void k_convert_planes(int8_t* __restrict__ canon, uint8_t* __restrict__ tiles, int L, int T, int R) {
    const uint64_t N = (uint64_t)L * L;
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= N * (uint64_t)R) return;
    const int r = (int)(gid / N);
    const uint64_t i = gid - (uint64_t)r * N;
    const int x = (int)(i % L), y = (int)(i / L);
    const int B = L / T, NW = T / 32, LPT = T / 2;
    const int tx = x / T, ty = y / T, lx = x - tx * T, ly = y - ty * T;
    const int cc = (lx + ly) & 1, px = lx >> 1, gx = px >> 4, kk = px & 15, rp = ly & 1, Y = ly >> 1;
    const size_t tile = ((size_t)r * B + ty) * B + tx;
    constexpr bool BITS = MODE >= 2;
    const size_t body_bytes = BITS ? (size_t)(T * T / 8) : (size_t)(T * T);
    uint8_t* rec = tiles + tile * (body_bytes + 64);
    uint8_t* body = rec + ((((rp * 2 + cc) * NW + gx) * LPT) + Y) * 16 + piece_byte(kk);
    uint32_t* w = reinterpret_cast<uint32_t*>(rec) + ((cc * NW + gx) * LPT + Y);
    const int j = rp * 16 + kk;
    if (MODE == 1) { canon[gid] = *body ? 1 : -1; return; }
    if (MODE == 3) { canon[gid] = ((*w >> j) & 1u) ? 1 : -1; return; }
    const bool up = canon[gid] > 0;
    if (!BITS) *body = up ? 1 : 0;
    if (!up) return;
    if (BITS) atomicOr(w, 1u << j);
    uint32_t* e = reinterpret_cast<uint32_t*>(rec + body_bytes);          // boundary copies (zeroed first), see PG
    if (Y == 0) atomicOr(e + 0 + cc * NW + gx, 1u << j);                  // TOP: words of block row 0
    if (Y == LPT - 1) atomicOr(e + 8 + cc * NW + gx, 1u << j);            // BOT: words of block row LPT-1
    if (lx == 0) atomicOr(e + 4 + rp, 1u << Y);                           // COL: L0, L1
    if (lx == T - 1) atomicOr(e + 6 + rp, 1u << Y);                       //      R0, R1
}

// Couplings, canonical J[d][i] (bond i -> i + e_d) -> coupling records (zeroed first).  One thread per site:
// it owns the four bonds seen from that site, in the order of the neighbour words of update_block.
__global__ void k_convert_couplings(const int8_t* __restrict__ J, uint32_t* __restrict__ jrec, int L, int T) {
    const uint64_t N = (uint64_t)L * L;
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int x = (int)(i % L), y = (int)(i / L);
    const int B = L / T, NW = T / 32, LPT = T / 2;
    const int tx = x / T, ty = y / T, lx = x - tx * T, ly = y - ty * T;
    const int cc = (lx + ly) & 1, px = lx >> 1, gx = px >> 4, kk = px & 15, rp = ly & 1, Y = ly >> 1;
    const uint64_t iL = (uint64_t)(x == 0 ? L - 1 : x - 1) + (uint64_t)L * y;         // site to the left
    const uint64_t iU = (uint64_t)x + (uint64_t)L * (y == 0 ? L - 1 : y - 1);         // site above (y - 1)
    const bool right = J[i] < 0, left = J[iL] < 0, down = J[N + i] < 0, up = J[N + iU] < 0;
    const bool v1 = rp == 0 ? down : up;          // V1 = the other row of the block
    const bool v2 = rp == 0 ? up : down;          // V2 = the row outside the block
    const bool h1 = (x & 1) == 0 ? right : left;  // H1 = the other site of the aligned pair (2p_x, 2p_x + 1)
    const bool h2 = (x & 1) == 0 ? left : right;
    uint32_t* w = jrec + (((size_t)ty * B + tx) * (2 * NW * LPT) + (cc * NW + gx) * LPT + Y) * 4;
    const uint32_t bit = 1u << (rp * 16 + kk);
    if (v1) atomicOr(w + 0, bit);
    if (v2) atomicOr(w + 1, bit);
    if (h1) atomicOr(w + 2, bit);
    if (h2) atomicOr(w + 3, bit);
}

template <int T, bool BITS>
int launch_colour_planes(const PlaneArgs& A) {
    const int warps = kPlaneThreads / 32;
    const uint32_t grid = (A.njobs + warps - 1) / warps;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(warps * 32); cfg.dynamicSmemBytes = 0; cfg.stream = hooks().stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    static const int pdl = getenv("ISING_NO_PDL") ? 0 : 1;
    attr[0].val.programmaticStreamSerializationAllowed = pdl;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (A.jrec) ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile_planes<T, BITS, true>, A));
    else ISING_CUDA_OK(cudaLaunchKernelEx(&cfg, k_tile_planes<T, BITS, false>, A));
    count_launch();
    return 0;
}

}  // namespace

bool tile_planes_supported(const ising_ctx* h, int T) {
    if (h->dim != 2) return false;
    if (T != 32 && T != 64) return false;
    if (h->L % T) return false;
    const int B = h->L / T;
    return B >= 2 && (B % 2 == 0);
}

size_t coupling_record_bytes(const ising_ctx* h) { return (size_t)h->N / 2 * 4; }   // 4 bond bits per site

int launch_convert_couplings(ising_ctx* h, int T, void* d_jrec) {
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemsetAsync(d_jrec, 0, coupling_record_bytes(h), st));
    k_convert_couplings<<<(unsigned)((h->N + 255) / 256), 256, 0, st>>>(h->d_J, (uint32_t*)d_jrec, h->L, T);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

size_t tile_planes_bytes(const ising_ctx* h, int T, bool bits) {
    const size_t B = (size_t)(h->L / T);
    return (size_t)h->R * B * B * (size_t)((bits ? T * T / 8 : T * T) + 64);
}

int launch_canon_to_planes(ising_ctx* h, int T, bool bits, const int8_t* d_canon, void* d_tiles) {
    const uint64_t total = h->N * (uint64_t)h->R;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    cudaStream_t st = hooks().stream;
    ISING_CUDA_OK(cudaMemsetAsync(d_tiles, 0, tile_planes_bytes(h, T, bits), st));
    if (bits) {
        k_convert_planes<2><<<blocks, 256, 0, st>>>(const_cast<int8_t*>(d_canon), (uint8_t*)d_tiles, h->L, T, h->R);
    } else {
        k_convert_planes<0><<<blocks, 256, 0, st>>>(const_cast<int8_t*>(d_canon), (uint8_t*)d_tiles, h->L, T, h->R);
    }
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

int launch_planes_to_canon(ising_ctx* h, int T, bool bits, const void* d_tiles, int8_t* d_canon) {
    const uint64_t total = h->N * (uint64_t)h->R;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    cudaStream_t st = hooks().stream;
    if (bits) k_convert_planes<3><<<blocks, 256, 0, st>>>(d_canon, (uint8_t*)const_cast<void*>(d_tiles), h->L, T, h->R);
    else k_convert_planes<1><<<blocks, 256, 0, st>>>(d_canon, (uint8_t*)const_cast<void*>(d_tiles), h->L, T, h->R);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

constexpr size_t kL2StreamBytes = 96u << 20;    // records larger than this do not stay in the 126 MB L2 between passes

bool plain64_supported(const ising_ctx* h, int T) { return h->dim == 2 && h->L == 64 && T == 64; }

static void fill_accept(PlaneArgs& A, const Accept& acc) {
    for (int q = 0; q < kHeadBits; ++q) {
        A.u1[q] = ((acc.thr[0] >> (31 - q)) & 1u) ? 0xffffffffu : 0u;
        A.u2[q] = ((acc.thr[1] >> (31 - q)) & 1u) ? 0xffffffffu : 0u;
    }
    A.force = acc.thr_is_2p32[0] ? 0xffffffffu : 0u;       // thr[m] = 2^32 happens only at beta = 0, for every m at once
    A.t1_tail = acc.thr[0] & ((1u << kTailBits) - 1u);
    A.t2_tail = acc.thr[1] & ((1u << kTailBits) - 1u);
}

// a8: all n passes of a 64x64 plain-checkerboard run in one launch, one warp per replica; d_E / d_M (n*R each) optional.
int launch_plain64(ising_ctx* h, const Accept& acc, bool bits, int n, int k, uint64_t t_first, long long* d_E, long long* d_M) {
    PlaneArgs A;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_seeds;
    A.L = 64; A.B = 1; A.R = h->R; A.k = k; A.t_first = t_first; A.C = 0; A.njobs = (uint32_t)h->R;
    A.magic_rep = A.magic_hb = 0;
    A.stream = 0;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    fill_accept(A, acc);
    cudaStream_t st = hooks().stream;
    if (bits) {
        if (A.jrec) k_plain64_planes<true, true><<<h->R, 32, 0, st>>>(A, n, d_E, d_M);
        else k_plain64_planes<true, false><<<h->R, 32, 0, st>>>(A, n, d_E, d_M);
    } else {
        if (A.jrec) k_plain64_planes<false, true><<<h->R, 32, 0, st>>>(A, n, d_E, d_M);
        else k_plain64_planes<false, false><<<h->R, 32, 0, st>>>(A, n, d_E, d_M);
    }
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// a10 on tile records: E[r], M[r] (R values each, either may be null) of the state held in plane records.
int launch_observables_planes(ising_ctx* h, int T, bool bits, long long* d_E, long long* d_M) {
    cudaStream_t st = hooks().stream;
    if (d_E) ISING_CUDA_OK(cudaMemsetAsync(d_E, 0, sizeof(long long) * h->R, st));
    if (d_M) ISING_CUDA_OK(cudaMemsetAsync(d_M, 0, sizeof(long long) * h->R, st));
    PlaneArgs A = {};
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_seeds;
    A.L = h->L; A.B = h->L / T; A.R = h->R; A.k = 0; A.t_first = 0;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    const uint32_t tiles_per_colour = (uint32_t)((size_t)h->R * A.B * A.B / 2);
    A.njobs = tiles_per_colour / (uint32_t)(64 / T);
    A.magic_rep = fastdiv_magic((uint32_t)A.B * (uint32_t)A.B / 2u);
    A.magic_hb = fastdiv_magic((uint32_t)A.B / 2u);
    const int warps = kPlaneThreads / 32;
    const uint32_t grid = (A.njobs + warps - 1) / warps;
    for (int C = 0; C < 2; ++C) {
        A.C = C;
#define ISING_OBS(TT, BB)                                                                                   \
        do {                                                                                                \
            if (A.jrec) k_observables_planes<TT, BB, true><<<grid, warps * 32, 0, st>>>(A, d_E, d_M);      \
            else k_observables_planes<TT, BB, false><<<grid, warps * 32, 0, st>>>(A, d_E, d_M);            \
        } while (0)
        if (T == 64) { if (bits) ISING_OBS(64, true); else ISING_OBS(64, false); }
        else { if (bits) ISING_OBS(32, true); else ISING_OBS(32, false); }
#undef ISING_OBS
        count_launch();
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

// a1: one outer pass = colour-0 launch, colour-1 launch, k inner sweeps each.
int launch_tile_planes_pass(ising_ctx* h, const Accept& acc, int T, bool bits, int k, uint64_t t_first) {
    PlaneArgs A;
    A.tiles = (uint8_t*)h->d_tiles;
    A.seeds = h->d_seeds;
    A.L = h->L; A.B = h->L / T; A.R = h->R; A.k = k; A.t_first = t_first;
    A.jrec = h->has_J ? (const uint4*)h->d_Jtiles : nullptr;
    A.stream = tile_planes_bytes(h, T, bits) > kL2StreamBytes ? 1u : 0u;
    const uint32_t tiles_per_colour = (uint32_t)((size_t)h->R * A.B * A.B / 2);
    A.njobs = tiles_per_colour / (uint32_t)(64 / T);
    A.magic_rep = fastdiv_magic((uint32_t)A.B * (uint32_t)A.B / 2u);
    A.magic_hb = fastdiv_magic((uint32_t)A.B / 2u);
    fill_accept(A, acc);
    for (int C = 0; C < 2; ++C) {
        A.C = C;
        if (T == 64) bits ? launch_colour_planes<64, true>(A) : launch_colour_planes<64, false>(A);
        else bits ? launch_colour_planes<32, true>(A) : launch_colour_planes<32, false>(A);
    }
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}

}  // namespace ising
