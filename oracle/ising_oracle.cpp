// oracle/ising_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, sequential, obviously-correct CPU restatement of the double-checkerboard
// single-spin-flip Metropolis sweep of arXiv 1006.3865 (M. Weigel, "Simulating spin
// models on GPU").  It exists to define what the CUDA path must compute bit for bit.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may call it.  It shares no code with paper_1006_3865_b200/ (own Philox, own
// thresholds, own schedule) and neither side includes or imports the other.
//
// Citation convention: P:n = /root/reference/PAPER.md line n; S8c.k = SURVEY.md §8(c)
// "Specification" item k (the reading taken wherever the paper is silent; every such
// reading is listed in DESIGN.md §3).
//
// What the paper fixes:
//   * model       H = -J Σ_<ij> s_i s_j, s_i = ±1, periodic square / simple cubic lattice
//                 of edge L (eq. (1)); J_ij = ±1 quenched for the EA glass
//   * acceptance  p_acc = min[1, exp(-β ΔE)] (eq. (2))
//   * schedule    coarse B×B tiles coloured even/odd, each T×T tile coloured even/odd
//                 (P:62); even coarse tiles first, inside a tile even sites then
//                 odd sites, repeated k times per tile load, then the odd
//                 coarse tiles.
// What the paper leaves open and DESIGN.md §3 fixes (S8c.1-8): which parity is "even",
// the random-number generator and its site mapping (Philox4x32-10, counter-based), the
// integer form of the acceptance test, the hot start, what one "sweep" is when k > 1.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Philox known-answer vectors and the
// cuRAND host generator; threshold tables against an independent long-double evaluation;
// exact enumeration of the 4×4 and 2×2×2 lattices; exhaustive single-site detailed
// balance on 2×2; Kaufman's exact finite-lattice energy at L=16; E(all up) = -dim·N;
// Z2 and gauge (Mattis) symmetry; sweep(a);sweep(b) == sweep(a+b); tile-order
// independence; SURVEY.md Appendix A trajectories produced by two unrelated programs.
// Every exported function below is reached by at least one of those pins; none is
// "parity unpinned".
//
// Two RNG->site mappings are implemented (DESIGN.md §3 reading R6; the paper is silent on
// the generator, P:78/P:84 only say that a per-thread LCG was used and is unsafe):
//   RNG_WORDS   S8c.3 verbatim: one full Philox output word per site.
//   RNG_PLANES  multi-spin form: the 12 leading bits of r come from bit-planes shared by a
//               block of 32 same-colour sites, the 20 trailing bits from a per-site call.
// Both give every (site, half-sweep) its own uniform 32-bit r compared with the same
// uint32 thresholds; they are different conventions, hence different trajectories.
//
// Build: g++ -O2 -std=c++17 -shared -fPIC ising_oracle.cpp -o liboracle_ising.so

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// ---------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) — S8c.2.  One round:
//   ctr' = { hi(M1*c2) ^ c1 ^ k0, lo(M1*c2), hi(M0*c0) ^ c3 ^ k1, lo(M0*c0) }
// ten rounds, the key bumped by (W0, W1) between rounds.
// ---------------------------------------------------------------------------------
constexpr uint32_t PHILOX_M0 = 0xD2511F53u;  // multiplies ctr[0]
constexpr uint32_t PHILOX_M1 = 0xCD9E8D57u;  // multiplies ctr[2]
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u;  // key[0] increment
constexpr uint32_t PHILOX_W1 = 0xBB67AE85u;  // key[1] increment

void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)PHILOX_M0 * c0;
        const uint64_t p1 = (uint64_t)PHILOX_M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Domain tags carried in ctr[1] (S8c.3).
constexpr uint32_t TAG_SWEEP = 0, TAG_INIT = 1, TAG_COUPLING = 2, TAG_PLANES = 3, TAG_TAIL = 4;

enum { RNG_WORDS = 0, RNG_PLANES = 1 };
constexpr int HEAD_BITS = 12;                 // leading bits of r taken from bit-planes
constexpr int TAIL_BITS = 32 - HEAD_BITS;     // trailing bits taken from the per-site call

struct Oracle {
    int dim = 2;
    int L = 0;
    uint64_t N = 0;
    int R = 1;                       // replicas sharing the couplings (S8c item 12)
    bool has_J = false;
    std::vector<int8_t> J;           // J[d*N + i] = bond from site i to i + e_d (S8b)
    std::vector<uint64_t> seeds;     // one Philox key per replica
    // Asynchronous multi-spin coding batch (DESIGN.md §3.6 R17): every replica is its own disorder
    // realisation (own couplings J[r][d][i], own hot start from seeds[r]) but all draw the SAME sweep random
    // r(i, H), keyed by sweep_seed.  Each replica is then an ordinary run whose random stream happens to be shared.
    bool J_per_replica = false;
    bool shared_sweep = false;
    uint64_t sweep_seed = 0;
    std::vector<int8_t> s;           // s[r*N + i], canonical order i = x + L*(y + L*z) (S8c.1)
    uint64_t t = 0;                  // inner sweeps done so far (S8c.6)
    int reverse_tiles = 0;           // test hook: visit the tiles of a colour in reverse order
    int rng = RNG_PLANES;            // RNG->site mapping (see header); default = the product's
    int use_memo = 1;                // test hook: 0 recomputes every Philox block (same values)
    // RNG_PLANES memo: the HEAD_BITS planes of the last few blocks (direct-mapped cache)
    struct PlaneMemo { uint64_t seed, H; uint32_t g; bool valid; uint32_t plane[HEAD_BITS]; };
    std::vector<PlaneMemo> plane_memo;
    // one-entry memo of the last Philox block, so that the four same-colour sites that
    // share a counter do not recompute it.  Purely a cache: same values either way.
    uint32_t memo_ctr[4] = {0, 0, 0, 0};
    uint32_t memo_key[2] = {0, 0};
    uint32_t memo_out[4] = {0, 0, 0, 0};
    bool memo_valid = false;
};

inline void seed_key(uint64_t seed, uint32_t key[2]) {
    key[0] = (uint32_t)(seed & 0xffffffffu);
    key[1] = (uint32_t)(seed >> 32);
}

// S8c.3, sweep stream: the random word of site i in half-sweep H = 2t + c(i).
//   p = i >> 1;  r = Philox(ctr = {p >> 2, 0, lo32(H), hi32(H)}, key = seed)[p & 3]
uint32_t sweep_random(Oracle& o, uint64_t seed, uint64_t i, uint64_t H) {
    const uint64_t p = i >> 1;
    const uint32_t ctr[4] = {(uint32_t)(p >> 2), TAG_SWEEP, (uint32_t)(H & 0xffffffffu),
                             (uint32_t)(H >> 32)};
    uint32_t key[2];
    seed_key(seed, key);
    const bool hit = o.use_memo && o.memo_valid && ctr[0] == o.memo_ctr[0] && ctr[1] == o.memo_ctr[1] &&
                     ctr[2] == o.memo_ctr[2] && ctr[3] == o.memo_ctr[3] &&
                     key[0] == o.memo_key[0] && key[1] == o.memo_key[1];
    if (!hit) {
        philox4x32_10(ctr, key, o.memo_out);
        std::memcpy(o.memo_ctr, ctr, sizeof ctr);
        std::memcpy(o.memo_key, key, sizeof key);
        o.memo_valid = true;
    }
    return o.memo_out[p & 3];
}

// RNG_PLANES geometry (DESIGN.md §3 R6).  Same-colour sites are addressed by their pair
// p_x = x >> 1 inside row (y, z) (every aligned pair (2p_x, 2p_x+1) of a row holds one site of
// each colour because L is even, S8c.3).  Rows and pairs are cut into blocks of BW pairs x
// BH rows of y: (BW, BH) = (16, 2) in 2D, (4, 8) in 3D, so a block never straddles a tile
// whose edge is a multiple of 32 (2D) or 8 (3D).  Inside a block
//     bit   j = (y % BH) * BW + (p_x % BW)                       0 <= j < 32
//     block g = ((z * GH + y / BH) * GW + p_x / BW),  GH = ceil(L / BH), GW = ceil((L/2) / BW)
void plane_geometry(const Oracle& o, uint64_t i, uint32_t* g, int* j) {
    const uint64_t L = (uint64_t)o.L;
    const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / (L * L));
    const int BW = (o.dim == 2) ? 16 : 4, BH = (o.dim == 2) ? 2 : 8;
    const int px = x >> 1;
    const int GW = ((o.L >> 1) + BW - 1) / BW, GH = (o.L + BH - 1) / BH;
    *j = (y % BH) * BW + (px % BW);
    *g = (uint32_t)(((uint64_t)z * GH + (uint64_t)(y / BH)) * GW + (uint64_t)(px / BW));
}

// RNG_PLANES, sweep stream of site i in half-sweep H = 2t + c(i):
//   plane q (q = 0..HEAD_BITS-1) of block g  =  Philox(ctr = {g, TAG_PLANES + 256*(q>>2), lo32 H, hi32 H})[q & 3]
//   head = sum_q ((plane_q >> j) & 1) << (HEAD_BITS-1-q)          (plane 0 is the most significant bit)
//   tail = Philox(ctr = {i >> 1, TAG_TAIL, lo32 H, hi32 H})[0] >> HEAD_BITS
//   r    = head << TAIL_BITS | tail
uint32_t sweep_random_planes(Oracle& o, uint64_t seed, uint64_t i, uint64_t H) {
    uint32_t g; int j;
    plane_geometry(o, i, &g, &j);
    uint32_t key[2];
    seed_key(seed, key);
    uint32_t local[HEAD_BITS];
    const uint32_t* plane = local;
    Oracle::PlaneMemo* m = nullptr;
    if (o.use_memo) {
        if (o.plane_memo.empty()) o.plane_memo.assign(4096, Oracle::PlaneMemo{0, 0, 0, false, {0}});
        m = &o.plane_memo[g & 4095u];
        if (m->valid && m->g == g && m->H == H && m->seed == seed) plane = m->plane;
    }
    if (plane == local) {
        for (int n = 0; n < HEAD_BITS / 4; ++n) {
            const uint32_t ctr[4] = {g, TAG_PLANES + 256u * (uint32_t)n, (uint32_t)(H & 0xffffffffu),
                                     (uint32_t)(H >> 32)};
            philox4x32_10(ctr, key, local + 4 * n);
        }
        if (m) {
            m->seed = seed; m->H = H; m->g = g; m->valid = true;
            std::memcpy(m->plane, local, sizeof local);
            plane = m->plane;
        }
    }
    uint32_t head = 0;
    for (int q = 0; q < HEAD_BITS; ++q) head |= ((plane[q] >> j) & 1u) << (HEAD_BITS - 1 - q);
    const uint32_t tctr[4] = {(uint32_t)(i >> 1), TAG_TAIL, (uint32_t)(H & 0xffffffffu), (uint32_t)(H >> 32)};
    uint32_t tout[4];
    philox4x32_10(tctr, key, tout);
    return (head << TAIL_BITS) | (tout[0] >> HEAD_BITS);
}

// S8c.3, hot start: s_i = (Philox(ctr = {i >> 2, 1, 0, 0}, key = seed)[i & 3] >> 31) ? -1 : +1
void hot_start(int8_t* s, uint64_t N, uint64_t seed) {
    uint32_t key[2];
    seed_key(seed, key);
    for (uint64_t i = 0; i < N; ++i) {
        const uint32_t ctr[4] = {(uint32_t)(i >> 2), TAG_INIT, 0, 0};
        uint32_t out[4];
        philox4x32_10(ctr, key, out);
        s[i] = (out[i & 3] >> 31) ? -1 : +1;
    }
}

// S8c.4: thr[m] = floor(exp(-β·4m)·2^32), m = 1..dim, in double.  ΔE = 2a = 4m (eq. (2)).
void thresholds(double beta, int dim, uint64_t thr[4]) {
    thr[0] = 0;  // unused: a <= 0 always flips
    for (int m = 1; m <= 3; ++m)
        thr[m] = (m <= dim) ? (uint64_t)std::floor(std::exp(-beta * 4.0 * (double)m) * 4294967296.0)
                            : 0;
}

inline uint64_t site_index(const Oracle& o, int x, int y, int z) {
    return (uint64_t)x + (uint64_t)o.L * ((uint64_t)y + (uint64_t)o.L * (uint64_t)z);
}

inline int wrap(int v, int L) { return v < 0 ? v + L : (v >= L ? v - L : v); }

// S8c.5: a = s_i · Σ_d [ J_d(i) s(i+e_d) + J_d(i-e_d) s(i-e_d) ];  ΔE = 2a.
// Flip if a <= 0 (ΔE <= 0 ⇒ p_acc = 1, eq. (2)); else flip iff r < thr[a/2] (strict, unsigned).
void update_site(Oracle& o, int r, int x, int y, int z, uint64_t H, const uint64_t thr[4]) {
    int8_t* s = o.s.data() + (uint64_t)r * o.N;
    const uint64_t i = site_index(o, x, y, z);
    const int coord[3] = {x, y, z};
    const int8_t* Jr = o.J.data() + (o.J_per_replica ? (uint64_t)r * o.dim * o.N : 0);
    uint64_t stride = 1;  // index distance of one step along e_d: 1, L, L^2 (S8c.1)
    int field = 0;
    for (int d = 0; d < o.dim; ++d) {
        // periodic neighbours i + e_d and i - e_d
        const uint64_t ip = (coord[d] == o.L - 1) ? i - (uint64_t)(o.L - 1) * stride : i + stride;
        const uint64_t im = (coord[d] == 0) ? i + (uint64_t)(o.L - 1) * stride : i - stride;
        const int Jp = o.has_J ? Jr[(uint64_t)d * o.N + i] : 1;     // bond i -> i+e_d
        const int Jm = o.has_J ? Jr[(uint64_t)d * o.N + im] : 1;    // bond (i-e_d) -> i
        field += Jp * s[ip] + Jm * s[im];
        stride *= (uint64_t)o.L;
    }
    const int a = s[i] * field;
    bool flip;
    if (a <= 0) {
        flip = true;
    } else {
        const uint64_t key = o.shared_sweep ? o.sweep_seed : o.seeds[r];
        const uint64_t rnd = (o.rng == RNG_PLANES) ? sweep_random_planes(o, key, i, H) : sweep_random(o, key, i, H);
        flip = rnd < thr[a / 2];
    }
    if (flip) s[i] = (int8_t)-s[i];
}

// S8c.6 — the schedule of P:64-74.
//   for pass: for C in {0,1}: for every tile of coarse colour C:
//       for j in 0..k-1: t = t0 + pass*k + j
//           for c in {0,1}: for every site of the tile with (x+y+z)&1 == c: Update(i, 2t+c)
// Neighbours are read from the live array; for an even number of tiles per edge no two
// tiles of one coarse colour touch, so this equals "halo frozen while the tile is swept k
// times".  T == L is the single checkerboard of P:62.
int sweep_passes(Oracle& o, double beta, int n, int tile, int k, int64_t* E_series,
                 int64_t* M_series);

void observables(const Oracle& o, int r, int64_t* E, int64_t* M) {
    // S8c.7: E = -Σ_i Σ_{d<dim} J_d(i) s_i s_(i+e_d),  M = Σ_i s_i
    const int8_t* s = o.s.data() + (uint64_t)r * o.N;
    int64_t e = 0, m = 0;
    const int Lz = (o.dim == 3) ? o.L : 1;
    for (int z = 0; z < Lz; ++z)
        for (int y = 0; y < o.L; ++y)
            for (int x = 0; x < o.L; ++x) {
                const uint64_t i = site_index(o, x, y, z);
                m += s[i];
                int c[3] = {x, y, z};
                for (int d = 0; d < o.dim; ++d) {
                    int cp[3] = {x, y, z};
                    cp[d] = wrap(c[d] + 1, o.L);
                    const uint64_t ip = site_index(o, cp[0], cp[1], cp[2]);
                    const int Jp = o.has_J ? o.J[(o.J_per_replica ? (uint64_t)r * o.dim * o.N : 0) + (uint64_t)d * o.N + i] : 1;
                    e -= Jp * s[i] * s[ip];
                }
            }
    *E = e;
    *M = m;
}

bool tile_ok(const Oracle& o, int T) {
    // S8b conventions: T even, T | L, and (L/T even or T == L)
    if (T < 2 || (T & 1) || o.L % T) return false;
    const int B = o.L / T;
    return B == 1 || (B % 2 == 0);
}

int sweep_passes(Oracle& o, double beta, int n, int tile, int k, int64_t* E_series,
                 int64_t* M_series) {
    const int T = (tile == 0) ? o.L : tile;
    if (!tile_ok(o, T) || k < 1 || n < 0 || !(beta >= 0.0) || !std::isfinite(beta)) return -1;
    uint64_t thr[4];
    thresholds(beta, o.dim, thr);
    const int B = o.L / T;
    const int Bz = (o.dim == 3) ? B : 1;
    const int Tz = (o.dim == 3) ? T : 1;
    const int64_t ntiles = (int64_t)B * B * Bz;
    for (int pass = 0; pass < n; ++pass) {
        for (int C = 0; C < 2; ++C) {
            for (int64_t q = 0; q < ntiles; ++q) {
                const int64_t tl = o.reverse_tiles ? (ntiles - 1 - q) : q;
                const int tx = (int)(tl % B), ty = (int)((tl / B) % B), tz = (int)(tl / ((int64_t)B * B));
                if (((tx + ty + tz) & 1) != C) continue;
                for (int r = 0; r < o.R; ++r)
                    for (int j = 0; j < k; ++j) {
                        const uint64_t t = o.t + (uint64_t)pass * (uint64_t)k + (uint64_t)j;
                        for (int c = 0; c < 2; ++c) {
                            const uint64_t H = 2 * t + (uint64_t)c;
                            for (int dz = 0; dz < Tz; ++dz)
                                for (int dy = 0; dy < T; ++dy)
                                    for (int dx = 0; dx < T; ++dx) {
                                        const int x = tx * T + dx, y = ty * T + dy, z = tz * Tz + dz;
                                        if (((x + y + z) & 1) != c) continue;
                                        update_site(o, r, x, y, z, H, thr);
                                    }
                        }
                    }
            }
        }
        if (E_series || M_series) {
            for (int r = 0; r < o.R; ++r) {
                int64_t e, m;
                observables(o, r, &e, &m);
                if (E_series) E_series[(int64_t)pass * o.R + r] = e;
                if (M_series) M_series[(int64_t)pass * o.R + r] = m;
            }
        }
    }
    o.t += (uint64_t)n * (uint64_t)k;
    return 0;
}

}  // namespace

extern "C" {

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
    philox4x32_10(ctr, key, out);
}

// out[0..2] = thr[1..3] (0 beyond dim)
void oracle_thresholds(double beta, int dim, uint64_t* out) {
    uint64_t thr[4];
    thresholds(beta, dim, thr);
    out[0] = thr[1]; out[1] = thr[2]; out[2] = thr[3];
}

// S8c.3 harness couplings: J[d][i] = (Philox(ctr={i>>2, 2, d, 0}, key=jseed)[i&3] >> 31) ? -1 : +1
void oracle_make_couplings(int dim, int L, uint64_t jseed, int8_t* out) {
    uint64_t N = 1;
    for (int d = 0; d < dim; ++d) N *= (uint64_t)L;
    uint32_t key[2];
    seed_key(jseed, key);
    for (int d = 0; d < dim; ++d)
        for (uint64_t i = 0; i < N; ++i) {
            const uint32_t ctr[4] = {(uint32_t)(i >> 2), TAG_COUPLING, (uint32_t)d, 0};
            uint32_t o4[4];
            philox4x32_10(ctr, key, o4);
            out[(uint64_t)d * N + i] = (o4[i & 3] >> 31) ? -1 : +1;
        }
}

void* oracle_create_batch(int dim, int L, const int8_t* J, const uint64_t* seeds, int R) {
    if ((dim != 2 && dim != 3) || L < 2 || (L & 1) || R < 1) return nullptr;
    Oracle* o = new Oracle;
    o->dim = dim; o->L = L; o->R = R;
    o->N = 1;
    for (int d = 0; d < dim; ++d) o->N *= (uint64_t)L;
    if (J) {
        o->has_J = true;
        o->J.assign(J, J + (uint64_t)dim * o->N);
        for (int8_t v : o->J) if (v != 1 && v != -1) { delete o; return nullptr; }
    }
    o->seeds.assign(seeds, seeds + R);
    o->s.resize((uint64_t)R * o->N);
    for (int r = 0; r < R; ++r) hot_start(o->s.data() + (uint64_t)r * o->N, o->N, seeds[r]);
    return o;
}

// Multi-realisation batch with shared sweep randoms (asynchronous multi-spin coding; R17): J = R*dim*N
// couplings (realisation-major), init_seeds[r] = hot start of realisation r, sweep_seed = key of the shared r(i, H).
void* oracle_create_multi(int dim, int L, const int8_t* J, const uint64_t* init_seeds, int R, uint64_t sweep_seed) {
    if ((dim != 2 && dim != 3) || L < 2 || (L & 1) || R < 1 || !J) return nullptr;
    Oracle* o = new Oracle;
    o->dim = dim; o->L = L; o->R = R;
    o->N = 1;
    for (int d = 0; d < dim; ++d) o->N *= (uint64_t)L;
    o->has_J = true; o->J_per_replica = true; o->shared_sweep = true; o->sweep_seed = sweep_seed;
    o->J.assign(J, J + (uint64_t)R * dim * o->N);
    for (int8_t v : o->J) if (v != 1 && v != -1) { delete o; return nullptr; }
    o->seeds.assign(init_seeds, init_seeds + R);
    o->s.resize((uint64_t)R * o->N);
    for (int r = 0; r < R; ++r) hot_start(o->s.data() + (uint64_t)r * o->N, o->N, init_seeds[r]);
    return o;
}

void* oracle_create(int dim, int L, const int8_t* J, uint64_t seed) {
    return oracle_create_batch(dim, L, J, &seed, 1);
}

void oracle_destroy(void* h) { delete (Oracle*)h; }

int oracle_sweep(void* h, double beta, int n, int tile, int k) {
    return sweep_passes(*(Oracle*)h, beta, n, tile, k, nullptr, nullptr);
}

// E, M: n*R values, pass-major, measured after every outer pass.
int oracle_sweep_series(void* h, double beta, int n, int tile, int k, int64_t* E, int64_t* M) {
    return sweep_passes(*(Oracle*)h, beta, n, tile, k, E, M);
}

int oracle_observables(void* h, int64_t* E, int64_t* M) {
    Oracle& o = *(Oracle*)h;
    for (int r = 0; r < o.R; ++r) observables(o, r, E + r, M + r);
    return 0;
}

// S8c.7: Q_ab = Σ_i s_i^a s_i^b
int oracle_overlap(void* h, int a, int b, int64_t* Q) {
    Oracle& o = *(Oracle*)h;
    if (a < 0 || b < 0 || a >= o.R || b >= o.R) return -1;
    const int8_t* sa = o.s.data() + (uint64_t)a * o.N;
    const int8_t* sb = o.s.data() + (uint64_t)b * o.N;
    int64_t q = 0;
    for (uint64_t i = 0; i < o.N; ++i) q += sa[i] * sb[i];
    *Q = q;
    return 0;
}

int oracle_copy_spins(void* h, int8_t* dst) {
    Oracle& o = *(Oracle*)h;
    std::memcpy(dst, o.s.data(), o.s.size());
    return 0;
}

int oracle_set_spins(void* h, const int8_t* src) {
    Oracle& o = *(Oracle*)h;
    for (uint64_t i = 0; i < o.s.size(); ++i) if (src[i] != 1 && src[i] != -1) return -1;
    std::memcpy(o.s.data(), src, o.s.size());
    return 0;
}

int oracle_get_counter(void* h, uint64_t* t) { *t = ((Oracle*)h)->t; return 0; }
int oracle_set_counter(void* h, uint64_t t) { ((Oracle*)h)->t = t; return 0; }
// mode: 0 = RNG_WORDS (S8c.3), 1 = RNG_PLANES.  Does not touch spins or the counter.
int oracle_set_rng(void* h, int mode) {
    if (mode != RNG_WORDS && mode != RNG_PLANES) return -1;
    ((Oracle*)h)->rng = mode;
    return 0;
}
int oracle_get_rng(void* h) { return ((Oracle*)h)->rng; }
int oracle_set_memo(void* h, int on) { ((Oracle*)h)->use_memo = on ? 1 : 0; return 0; }
// the 32-bit random of (replica r, site i, half-sweep H) under the handle's current mapping
uint32_t oracle_sweep_random(void* h, int r, uint64_t i, uint64_t H) {
    Oracle& o = *(Oracle*)h;
    const uint64_t key = o.shared_sweep ? o.sweep_seed : o.seeds[r];
    return (o.rng == RNG_PLANES) ? sweep_random_planes(o, key, i, H) : sweep_random(o, key, i, H);
}
int oracle_set_tile_order(void* h, int reversed) { ((Oracle*)h)->reverse_tiles = reversed; return 0; }

// S8c.8: FNV-1a-64 over the canonical bytes of replica r (0x01 for +1, 0xFF for -1).
uint64_t oracle_hash(void* h, int r) {
    Oracle& o = *(Oracle*)h;
    const uint8_t* p = (const uint8_t*)(o.s.data() + (uint64_t)r * o.N);
    uint64_t hsh = 0xcbf29ce484222325ull;
    for (uint64_t i = 0; i < o.N; ++i) { hsh ^= p[i]; hsh *= 0x100000001b3ull; }
    return hsh;
}

uint64_t oracle_hash_bytes(const uint8_t* p, uint64_t n) {
    uint64_t hsh = 0xcbf29ce484222325ull;
    for (uint64_t i = 0; i < n; ++i) { hsh ^= p[i]; hsh *= 0x100000001b3ull; }
    return hsh;
}

}  // extern "C"
