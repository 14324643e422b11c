// tile3d_planes_device.cuh — device code of the 3D multi-spin tile kernel (design notes: tile3d_planes.cu).
// Self-contained on top of philox.cuh / planes_common.cuh: compiled into the library by nvcc and, specialised on
// the head bits of the three thresholds, at run time by NVRTC (planes_jit.cu).
#pragma once
#include "planes_common.cuh"

#ifdef __CUDACC_RTC__
#define ISING_DEVICE_NS3 jit
#else
#define ISING_DEVICE_NS3
#endif

namespace ising {

namespace ISING_DEVICE_NS3 {

constexpr int kT3 = 8;
constexpr int kBody3I8 = 512, kBody3Bits = 64, kFaces3 = 96;
constexpr int kRec3I8 = 640, kRec3Bits = 160;        // padded to multiples of 128 / 32 bytes
constexpr int kXL = 0, kXR = 32, kYL = 64, kYR = 72, kZL = 80, kZR = 88;   // offsets inside the face area

struct Plane3Args {
    uint8_t* tiles;              // records, replica-major; tile (tz, ty, tx) at ((tz*B + ty)*B + tx)
    const uint64_t* seeds;
    uint64_t seed0;              // seeds[0]: the (uniform) key of a single-replica handle, used by kernels compiled with ISING_JIT_R == 1
    int L, B, R;
    int C;                       // coarse colour of this launch
    int k;
    uint64_t t_first;
    uint32_t njobs;              // 4 tiles per job
    uint32_t per_rep, per_z, hb; // tiles of one colour per replica (B^3/2), per tz (B*B/2), per ty (B/2)
    uint32_t magic_rep, magic_z, magic_hb;
    uint32_t u[3][kHeadBits];    // plane q: all-ones if bit (31-q) of thr[m+1] is set
    uint32_t tail[3];            // thr[m+1] & (2^20 - 1)
    uint32_t force;              // all-ones if beta = 0 (every thr = 2^32: every proposal is accepted)
    const uint4* jrec;           // coupling records (a9) or nullptr: per tile 2 x 8 x 2 uint4, (cc, lz) -> {Zm, Zp, Ym, Yp},
                                 // {X1, X2, 0, 0}: bit j set <=> the bond from site j of that word to its neighbour in the
                                 // Zm / Zp / Ym / Yp / O / X2 word of half_sweep3 is J = -1.  Shared by the replicas.
};

struct Tile3 {
    int r, tx, ty, tz;
};

__device__ __forceinline__ Tile3 job_tile3(const Plane3Args& A, uint32_t q) {
    // colour-C tiles enumerated (tz, ty, txh): tx = 2*txh + ((ty + tz + C) & 1)
    Tile3 t;
    const uint32_t rr = fastdiv(q, A.per_rep, A.magic_rep);
    uint32_t rem = q - rr * A.per_rep;
    const uint32_t zz = fastdiv(rem, A.per_z, A.magic_z);
    rem -= zz * A.per_z;
    const uint32_t yy = fastdiv(rem, A.hb, A.magic_hb);
    rem -= yy * A.hb;
    t.r = (int)rr; t.tz = (int)zz; t.ty = (int)yy;
    t.tx = (int)(2u * rem) + (((int)yy + (int)zz + A.C) & 1);
    return t;
}

// What a lane keeps of its slice.
struct Slice {
    uint32_t S[2];        // the slice's two colour words
    uint32_t x;           // halo bits x = -1 (at 4ly) and x = 8 (at 4ly+3), every row, either colour
    uint32_t y;           // halo rows y = -1 (bits 0-7) and y = 8 (bits 8-15): colour 0 pairs in the low nibble, colour 1 in the high
    uint32_t zq[2];       // lanes lz = 0 / 7: the slice below / above, by colour (no lane is both)
    uint32_t J[2][6];     // coupling words of the slice's two colours (kernels with HASJ only)
};

template <bool HASJ>
__device__ __forceinline__ void load_couplings(const Plane3Args& A, const Tile3& t, int lz, Slice& s) {
    if (!HASJ) return;
    const uint4* rec = A.jrec + (((size_t)t.tz * A.B + t.ty) * A.B + t.tx) * 32;
#pragma unroll
    for (int cc = 0; cc < 2; ++cc) {
        const uint4 a = __ldg(rec + (cc * 8 + lz) * 2), b = __ldg(rec + (cc * 8 + lz) * 2 + 1);
        s.J[cc][0] = a.x; s.J[cc][1] = a.y; s.J[cc][2] = a.z; s.J[cc][3] = a.w; s.J[cc][4] = b.x; s.J[cc][5] = b.y;
    }
}

template <bool BITS>
__device__ __forceinline__ void load_slice(const Plane3Args& A, const Tile3& t, int lz, Slice& s) {
    constexpr int REC = BITS ? kRec3Bits : kRec3I8;
    constexpr int BODY = BITS ? kBody3Bits : kBody3I8;
    const int B = A.B;
    const uint8_t* rep = A.tiles + (size_t)t.r * B * B * B * REC;
    auto rec_of = [&](int tz, int ty, int tx) { return rep + (((size_t)tz * B + ty) * B + tx) * REC; };
    const uint8_t* rec = rec_of(t.tz, t.ty, t.tx);
    const uint8_t* fXm = rec_of(t.tz, t.ty, t.tx == 0 ? B - 1 : t.tx - 1) + BODY;
    const uint8_t* fXp = rec_of(t.tz, t.ty, t.tx == B - 1 ? 0 : t.tx + 1) + BODY;
    const uint8_t* fYm = rec_of(t.tz, t.ty == 0 ? B - 1 : t.ty - 1, t.tx) + BODY;
    const uint8_t* fYp = rec_of(t.tz, t.ty == B - 1 ? 0 : t.ty + 1, t.tx) + BODY;
    if (BITS) {
        s.S[0] = ldg32(rec + lz * 4);
        s.S[1] = ldg32(rec + (8 + lz) * 4);
    } else {
        uint4 v[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) v[c] = ldg128(rec + (c * 8 + lz) * 16, body_policy(false));
        s.S[0] = pack16(pack16(0u, v[1]), v[0]);
        s.S[1] = pack16(pack16(0u, v[3]), v[2]);
    }
    s.x = ldh32(fXm + kXR + 4 * lz) |     // left tile's x = 7 sites, bit 4ly
          ldh32(fXp + kXL + 4 * lz);      // right tile's x = 0 sites, bit 4ly+3
    s.y = ldh8(fYm + kYR + lz) |                                        // tile in front: its row y = 7
          (ldh8(fYp + kYL + lz) << 8);                                  // tile behind: its row y = 0
    s.zq[0] = s.zq[1] = 0u;
    if (lz == 0) {
        const uint2 w = ldh64(rec_of(t.tz == 0 ? B - 1 : t.tz - 1, t.ty, t.tx) + BODY + kZR);
        s.zq[0] = w.x; s.zq[1] = w.y;
    }
    if (lz == 7) {
        const uint2 w = ldh64(rec_of(t.tz == B - 1 ? 0 : t.tz + 1, t.ty, t.tx) + BODY + kZL);
        s.zq[0] = w.x; s.zq[1] = w.y;
    }
}

// The slice's own face copies: the four words / bytes its x- and y-neighbours will read.
__device__ __forceinline__ void face_words(const uint32_t (&S)[2], int lz, uint32_t& XL, uint32_t& XR, uint32_t& YL, uint32_t& YR) {
    // x = 0 is pair 0 (bit 4ly) of colour (ly+lz)&1; x = 7 is pair 3 (bit 4ly+3) of colour (ly+lz+1)&1
    const uint32_t ev = (lz & 1) ? 0x10101010u : 0x01010101u;            // bit 4ly of the rows with (ly+lz) even
    const uint32_t od = (lz & 1) ? 0x08080808u : 0x80808080u;            // bit 4ly+3 of the rows with (ly+lz) odd
    XL = ((S[0] & ev) | (S[1] & (0x11111111u ^ ev))) << 3;
    XR = ((S[0] & od) | (S[1] & (0x88888888u ^ od))) >> 3;
    YL = (S[0] & 0xfu) | ((S[1] & 0xfu) << 4);
    YR = (S[0] >> 28) | ((S[1] >> 28) << 4);
}

template <bool BITS>
__device__ __forceinline__ void store_slice(const Plane3Args& A, const Tile3& t, int lz, const Slice& s, const uint2* lut) {
    constexpr int REC = BITS ? kRec3Bits : kRec3I8;
    constexpr int BODY = BITS ? kBody3Bits : kBody3I8;
    const int B = A.B;
    uint8_t* rec = A.tiles + ((size_t)t.r * B * B * B + ((size_t)t.tz * B + t.ty) * B + t.tx) * REC;
    if (BITS) {
        *reinterpret_cast<uint32_t*>(rec + lz * 4) = s.S[0];
        *reinterpret_cast<uint32_t*>(rec + (8 + lz) * 4) = s.S[1];
    } else {
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const uint2 a = __ldg(lut + ((s.S[cc] >> (16 * h)) & 0xffu));
                const uint2 b = __ldg(lut + ((s.S[cc] >> (16 * h + 8)) & 0xffu));
                stg128(rec + ((cc * 2 + h) * 8 + lz) * 16, make_uint4(a.x, a.y, b.x, b.y));
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

// R_m = [r < thr[m]], m = 1..3, and tie masks, for the 32 sites of block g (12 head planes).
__device__ __forceinline__ void head_masks3(const Plane3Args& A, uint32_t g, uint32_t Hlo, uint32_t Hhi, uint32_t k0,
                                            uint32_t k1, uint32_t (&R)[3], uint32_t (&eq)[3]) {
    uint32_t bw[3] = {0u, 0u, 0u}, ne[3] = {0u, 0u, 0u};
#pragma unroll
    for (int n = kHeadBits / 4 - 1; n >= 0; --n) {                  // least significant planes first
        const u32x4 o = philox4x32_10(g, kTagPlanes + 256u * n, Hlo, Hhi, k0, k1);
        const uint32_t p[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
        for (int w = 3; w >= 0; --w) {
            const int q = 4 * n + w;
#pragma unroll
            for (int m = 0; m < 3; ++m) {
                bw[m] = lop3<kLutChain>(p[w], bw[m], A.u[m][q]);
                ne[m] = lop3<kLutNe>(ne[m], p[w], A.u[m][q]);
            }
        }
    }
#pragma unroll
    for (int m = 0; m < 3; ++m) { R[m] = bw[m]; eq[m] = ~ne[m]; }
}

// ---- the same compare specialised on the head bits of the three thresholds (HP3 = head(thr[1]) << 24 |
// head(thr[2]) << 12 | head(thr[3]); tile_planes_device.cuh explains the idea).  A site needs one threshold:
// thr[3] if s0 (no unsatisfied bond), thr[2] if s1 (one), else thr[1].  Per plane the threshold bit of every site is a
// compile-time function of (s0, s1); then one borrow chain and one tie accumulator.
constexpr unsigned long long kNoSpec3 = ~0ull;
// Of three binary head bits that are not all equal exactly one differs from the other two, so the site's threshold bit depends on
// ONE mask: s0 (thr[3] differs), s1 (thr[2] differs) or s0 | s1 (thr[1] differs) — the third LOP3 input of the chain and tie steps.
// Planes whose bit is the same for all three thresholds need no mask, and two of them share one LOP3 (as in 2D).
template <unsigned long long HP3, int Q>
struct HeadBit3 {
    static constexpr int u1 = (int)((HP3 >> (24 + 11 - Q)) & 1), u2 = (int)((HP3 >> (12 + 11 - Q)) & 1), u3 = (int)((HP3 >> (11 - Q)) & 1);
    static constexpr bool same = u1 == u2 && u2 == u3;
    static constexpr int which = same ? -1 : (u1 == u2 ? 0 : (u1 == u3 ? 1 : 2));     // mask: 0 = s0, 1 = s1, 2 = s0 | s1
    static constexpr int u_clear = u1;                         // the site's threshold bit where the mask is 0 (thr[1] applies, or agrees) ...
    static constexpr int u_set = u1 == u2 ? u3 : u2;           // ... and where it is 1
};
__host__ __device__ constexpr int lut_chain_mask(int u_clear, int u_set) {            // inputs a = p, b = bw, c = mask
    int l = 0;
    for (int i = 0; i < 8; ++i) {
        const int p = (i >> 2) & 1, bw = (i >> 1) & 1, m = i & 1, u = m ? u_set : u_clear;
        l |= (((!p) && u) || ((p == u) && bw)) << i;
    }
    return l;
}
__host__ __device__ constexpr int lut_ne_mask(int u_clear, int u_set) {               // inputs a = ne, b = p, c = mask
    int l = 0;
    for (int i = 0; i < 8; ++i) {
        const int ne = (i >> 2) & 1, p = (i >> 1) & 1, m = i & 1, u = m ? u_set : u_clear;
        l |= (ne || (p != u)) << i;
    }
    return l;
}
__host__ __device__ constexpr int lut_chain_pair3(int uq, int uq1) {                   // inputs a = p_Q, b = p_(Q-1), c = bw
    int l = 0;
    for (int i = 0; i < 8; ++i) {
        const int pq = (i >> 2) & 1, pq1 = (i >> 1) & 1, bw = i & 1;
        const int b1 = ((!pq) && uq) || ((pq == uq) && bw);
        const int b2 = ((!pq1) && uq1) || ((pq1 == uq1) && b1);
        l |= b2 << i;
    }
    return l;
}
__host__ __device__ constexpr int lut_ne_pair3(int ua, int ub) {                       // inputs a = ne, b = p_a, c = p_b
    int l = 0;
    for (int i = 0; i < 8; ++i) {
        const int ne = (i >> 2) & 1, pa = (i >> 1) & 1, pb = i & 1;
        l |= (ne || (pa != ua) || (pb != ub)) << i;
    }
    return l;
}
template <unsigned long long HP3, int Q>
__device__ __forceinline__ void chain3_from(const uint32_t (&p)[kHeadBits], const uint32_t (&mask)[3], uint32_t& bw) {
    if constexpr (Q >= 0) {
        using H = HeadBit3<HP3, Q>;
        if constexpr (Q >= 1 && H::same && HeadBit3<HP3, (Q >= 1 ? Q - 1 : 0)>::same) {
            bw = lop3<lut_chain_pair3(H::u1, HeadBit3<HP3, Q - 1>::u1)>(p[Q], p[Q - 1], bw);
            chain3_from<HP3, Q - 2>(p, mask, bw);
        } else {
            bw = lop3<lut_chain_mask(H::same ? H::u1 : H::u_clear, H::same ? H::u1 : H::u_set)>(p[Q], bw, mask[H::same ? 0 : H::which]);
            chain3_from<HP3, Q - 1>(p, mask, bw);
        }
    }
}
template <unsigned long long HP3, int Q, int PEND>
__device__ __forceinline__ void ne3_from(const uint32_t (&p)[kHeadBits], const uint32_t (&mask)[3], uint32_t& ne) {
    if constexpr (Q >= 0) {
        using H = HeadBit3<HP3, Q>;
        if constexpr (!H::same) {
            ne = lop3<lut_ne_mask(H::u_clear, H::u_set)>(ne, p[Q], mask[H::which]);
            ne3_from<HP3, Q - 1, PEND>(p, mask, ne);
        } else if constexpr (PEND < 0) {
            ne3_from<HP3, Q - 1, Q>(p, mask, ne);
        } else {
            ne = lop3<lut_ne_pair3(HeadBit3<HP3, (PEND >= 0 ? PEND : 0)>::u1, H::u1)>(ne, p[PEND >= 0 ? PEND : 0], p[Q]);
            ne3_from<HP3, Q - 1, -1>(p, mask, ne);
        }
    } else if constexpr (PEND >= 0) {
        constexpr int u = HeadBit3<HP3, (PEND >= 0 ? PEND : 0)>::u1;
        ne = lop3<lut_ne_pair3(u, u)>(ne, p[PEND >= 0 ? PEND : 0], p[PEND >= 0 ? PEND : 0]);
    }
}
// the twelve head planes of block g at half-sweep H (S3.4): they do not depend on the spins, so k_grid3d draws those of a
// job's first half-sweep while the neighbours' faces are still on their way
__device__ __forceinline__ void head_planes3(uint32_t g, uint32_t Hlo, uint32_t Hhi, uint32_t k0, uint32_t k1, uint32_t (&p)[kHeadBits]) {
    static_assert(kHeadBits == 12, "three Philox calls");
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        const u32x4 o = philox4x32_10(g, kTagPlanes + 256u * n, Hlo, Hhi, k0, k1);
        p[4 * n] = o.x; p[4 * n + 1] = o.y; p[4 * n + 2] = o.z; p[4 * n + 3] = o.w;
    }
}
template <unsigned long long HP3>
__device__ __forceinline__ void head_masks3_sel(const uint32_t (&p)[kHeadBits], uint32_t s0, uint32_t s1, uint32_t& R, uint32_t& eq) {
    const uint32_t mask[3] = {s0, s1, s0 | s1};
    uint32_t bw = 0, ne = 0;
    chain3_from<HP3, kHeadBits - 1>(p, mask, bw);
    ne3_from<HP3, kHeadBits - 1, -1>(p, mask, ne);
    R = bw; eq = ~ne;
}

// The six neighbour words of the lane's slice for the sites of colour c (o = 1 - c is read): z-1 / z+1 by shuffle (halo
// words at the tile faces), y-1 / y+1 by 4-bit shifts, the other site of the aligned pair (O) and the pair-shifted word (X2).
__device__ __forceinline__ void neighbour_words3(const Slice& s, int c, int lz, uint32_t& Zm, uint32_t& Zp, uint32_t& Ym,
                                                 uint32_t& Yp, uint32_t& O, uint32_t& X2) {
    const int o = 1 - c;
    O = s.S[o];
    Zm = __shfl_up_sync(0xffffffffu, O, 1);
    Zp = __shfl_down_sync(0xffffffffu, O, 1);
    if (lz == 0) Zm = s.zq[o];
    if (lz == 7) Zp = s.zq[o];
    Ym = (O << 4) | ((s.y >> (4 * o)) & 0xfu);
    Yp = (O >> 4) | (((s.y >> (8 + 4 * o)) & 0xfu) << 28);
    // rows where the active site is the left one of its pair (x = 2 p_x): ly = lz + c (mod 2); their second
    // x-neighbour is pair p_x - 1, the other rows' is pair p_x + 1
    const uint32_t m = ((lz + c) & 1) ? 0xf0f0f0f0u : 0x0f0f0f0fu;
    X2 = ((((O << 1) & 0xeeeeeeeeu) | (s.x & 0x11111111u)) & m) | ((((O >> 1) & 0x77777777u) | (s.x & 0x88888888u)) & ~m);
}

// a10 on a slice held in registers: #up spins of both colours and #unsatisfied bonds seen from the colour-0 sites (every
// bond of the lattice has exactly one colour-0 end).  M = 2 #up - N, E = 2 #unsat - 3N.
template <bool HASJ>
__device__ __forceinline__ void count_slice(const Slice& s, int lz, int& up, int& unsat) {
    uint32_t Zm, Zp, Ym, Yp, O, X2;
    neighbour_words3(s, 0, lz, Zm, Zp, Ym, Yp, O, X2);
    const uint32_t S = s.S[0];
    unsat += __popc(S ^ Zm ^ (HASJ ? s.J[0][0] : 0u)) + __popc(S ^ Zp ^ (HASJ ? s.J[0][1] : 0u)) + __popc(S ^ Ym ^ (HASJ ? s.J[0][2] : 0u)) +
             __popc(S ^ Yp ^ (HASJ ? s.J[0][3] : 0u)) + __popc(S ^ O ^ (HASJ ? s.J[0][4] : 0u)) + __popc(S ^ X2 ^ (HASJ ? s.J[0][5] : 0u));
    up += __popc(s.S[0]) + __popc(s.S[1]);
}

// One half-sweep of colour c on the lane's slice (a4-a5, 6 neighbours).
// DRAWN: p holds the head planes of (g, H) already (specialised kernels only); otherwise p is scratch.
template <unsigned long long HP3, bool HASJ, bool DRAWN>
__device__ __forceinline__ void half_sweep3(const Plane3Args& A, Slice& s, int c, int lz, uint32_t g, uint32_t p_base,
                                            uint64_t H, uint32_t k0, uint32_t k1, uint32_t (&p)[kHeadBits]) {
    const uint32_t Hlo = (uint32_t)H, Hhi = (uint32_t)(H >> 32);
    const uint32_t S = s.S[c];
    uint32_t Zm, Zp, Ym, Yp, O, X2;
    neighbour_words3(s, c, lz, Zm, Zp, Ym, Yp, O, X2);
    // disagreeing neighbours, pairwise counts, then thresholds of the sum of six
    // unsatisfied bonds: J s_i s_j = -1  <=>  s_i != s_j for J = +1, s_i == s_j for J = -1 (eq. (1))
    const uint32_t a = S ^ Zm ^ (HASJ ? s.J[c][0] : 0u), b = S ^ Zp ^ (HASJ ? s.J[c][1] : 0u);
    const uint32_t e = S ^ Ym ^ (HASJ ? s.J[c][2] : 0u), f = S ^ Yp ^ (HASJ ? s.J[c][3] : 0u);
    const uint32_t x = S ^ O ^ (HASJ ? s.J[c][4] : 0u), y = S ^ X2 ^ (HASJ ? s.J[c][5] : 0u);
    const uint32_t p1 = a | b, q1 = a & b, p2 = e | f, q2 = e & f, p3 = x | y, q3 = x & y;
    const uint32_t ge1 = p1 | p2 | p3;
    const uint32_t ge2 = q1 | q2 | q3 | (p1 & p2) | (p1 & p3) | (p2 & p3);
    const uint32_t ge3 = (q1 & (p2 | p3)) | (q2 & (p1 | p3)) | (q3 & (p1 | p2)) | (p1 & p2 & p3) | A.force;   // dE <= 0: always flip
    if (HP3 != kNoSpec3) {
        const uint32_t s0 = ~ge1, s1 = ge1 & ~ge2;                  // no / exactly one unsatisfied bond
        uint32_t R, eq;
        if (!DRAWN) head_planes3(g, Hlo, Hhi, k0, k1, p);
        head_masks3_sel<HP3>(p, s0, s1, R, eq);
        uint32_t und = eq & ~ge3;
        while (und) {                                               // probability 2^-12 per site
            const int j = __ffs(und) - 1;
            und &= und - 1;
            const uint32_t p = p_base + (uint32_t)(j >> 2) * (uint32_t)(A.L >> 1) + (uint32_t)(j & 3);
            const u32x4 t = philox4x32_10(p, kTagTail, Hlo, Hhi, k0, k1);
            const uint32_t thr_tail = ((s0 >> j) & 1u) ? A.tail[2] : (((s1 >> j) & 1u) ? A.tail[1] : A.tail[0]);
            R |= (uint32_t)((t.x >> kHeadBits) < thr_tail) << j;
        }
        s.S[c] = S ^ (ge3 | R);
        return;
    }
    uint32_t R[3], eq[3];
    head_masks3(A, g, Hlo, Hhi, k0, k1, R, eq);
    uint32_t und = (eq[0] & ge2 & ~ge3) | (eq[1] & ge1 & ~ge2) | (eq[2] & ~ge1);   // n_dis = 2, 1, 0 need thr[1], thr[2], thr[3]
    while (und) {                                                   // probability 2^-12 per site
        const int j = __ffs(und) - 1;
        und &= und - 1;
        const uint32_t p = p_base + (uint32_t)(j >> 2) * (uint32_t)(A.L >> 1) + (uint32_t)(j & 3);
        const u32x4 t = philox4x32_10(p, kTagTail, Hlo, Hhi, k0, k1);
        const uint32_t tail = t.x >> kHeadBits;
#pragma unroll
        for (int mm = 0; mm < 3; ++mm)
            if ((eq[mm] >> j) & 1u) R[mm] |= (uint32_t)(tail < A.tail[mm]) << j;
    }
    const uint32_t flip = ge3 | (ge2 & R[0]) | (ge1 & R[1]) | R[2];   // thr[3] <= thr[2] <= thr[1]
    s.S[c] = S ^ flip;
}

template <unsigned long long HP3 = kNoSpec3, bool HASJ = false>
__device__ __forceinline__ void half_sweep3(const Plane3Args& A, Slice& s, int c, int lz, uint32_t g, uint32_t p_base,
                                            uint64_t H, uint32_t k0, uint32_t k1) {
    uint32_t p[kHeadBits];
    half_sweep3<HP3, HASJ, false>(A, s, c, lz, g, p_base, H, k0, k1, p);
}

constexpr int kThreads3 = 64;        // 2 warps = 8 tiles per CTA (measured at L = 256 .. 512, k = 1 .. 16: 64 = 128 > 256 > 512 threads)

template <bool BITS, unsigned long long HP3 = kNoSpec3, bool HASJ = false>
__global__ void __launch_bounds__(kThreads3) k_tile3d_planes(Plane3Args A) {
    const uint2* lut = kByteLutGlobal.e;      // int8 write-back table, read-only path (planes_common.cuh)
    // Programmatic dependent launch, as in k_tile_planes: the next colour's grid may be scheduled while this one
    // drains; it waits here until every store of the previous launch is visible.
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int lane = threadIdx.x & 31;
    const uint32_t job = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (job >= A.njobs) return;
    const int sub = lane >> 3, lz = lane & 7;
    const Tile3 t = job_tile3(A, job * 4u + (uint32_t)sub);
    Slice s;
    load_slice<BITS>(A, t, lz, s);
    load_couplings<HASJ>(A, t, lz, s);
#if defined(ISING_JIT_R) && ISING_JIT_R == 1
    const uint64_t seed = A.seed0;
#else
    const uint64_t seed = A.seeds[t.r];
#endif
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    const uint32_t z = (uint32_t)(t.tz * kT3 + lz);
    const uint32_t g = (z * (uint32_t)A.B + (uint32_t)t.ty) * (uint32_t)A.B + (uint32_t)t.tx;     // RNG block (S3.4)
    const uint32_t p_base = (uint32_t)(t.tx * 4) + (uint32_t)(A.L >> 1) * ((uint32_t)(t.ty * kT3) + (uint32_t)A.L * z);
    for (int j = 0; j < A.k; ++j) {
        const uint64_t tt = A.t_first + (uint64_t)j;
        half_sweep3<HP3, HASJ>(A, s, 0, lz, g, p_base, 2 * tt, k0, k1);
        half_sweep3<HP3, HASJ>(A, s, 1, lz, g, p_base, 2 * tt + 1, k0, k1);
    }
    store_slice<BITS>(A, t, lz, s, lut);
}

}  // namespace

}  // namespace ising
