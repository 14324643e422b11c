// oracle/heisenberg_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, sequential CPU restatement of the double-checkerboard single-spin Metropolis sweep for
// the classical Heisenberg (O(3)) model, the continuous-spin generalisation the paper names in one
// sentence: "The outlined approach easily generalizes to ... models with continuous spins such as
// the Heisenberg model, where the large efficieny of GPU devices with (single-precision)
// floating-point calculations comes into play".  SURVEY.md §8(f) item 4.
// Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may call it.  It shares no code with
// paper_1006_3865_b200/ and with oracle/ising_oracle.cpp (own Philox, own schedule).
//
// The paper fixes: the model (spins on the unit sphere, nearest-neighbour coupling J = 1, periodic
// hypercubic lattice as P:53-57), the acceptance min[1, exp(-β ΔE)] (eq. (2)), the schedule
// (as for the Ising model), and the precision: SINGLE.  Because one accept/reject
// decision changes the whole later trajectory, the floating-point operations are fixed one by one
// below (readings H1-H8): every operation is an IEEE-754 binary32 operation with
// round-to-nearest-even, fma(a,b,c) is the fused operation with one rounding, nothing is contracted
// or re-associated (build with -ffp-contract=off).  The CUDA side states the same operations with
// __fmaf_rn / __fmul_rn / __fadd_rn / __fsqrt_rn, so the two agree bit for bit.
//
// H1 model, storage   H = -Σ_<ij> s_i·s_j; s[c][i], c = 0,1,2 = x,y,z, float; site index, fine and
//                     coarse colours as S8c.1.
// H2 direction D(wa,wb)  uniform point of the sphere from 40 bits of two 32-bit words (Archimedes: z uniform,
//                     azimuth uniform): z20 = wa >> 12, phi20 = ((wa & 0xfff) << 8) | (wb >> 24)
//                       z   = fma(float(z20), 2^-19, -1)                           (exact, in [-1, 1))
//                       rho = sqrt(fma(-z, z, 1))
//                       q = phi20 >> 17 (octant), t = float(phi20 & 0x1ffff) * 2^-17 (exact); if q odd: t = t - 1
//                       x = t * PI_4;  x2 = x*x;  x3 = x2*x                       (azimuth - Q*pi/2, |x| <= pi/4)
//                       sn = fma(x3, S(x2), x),  S = ((S9*x2 + S7)*x2 + S5)*x2 + S3    by fma, S_n = ±1/n!
//                       cs = fma(x2, C(x2), 1),  C = (((C10*x2 + C8)*x2 + C6)*x2 + C4)*x2 + C2 by fma
//                       Q = ((q + 1) >> 1) & 3:  (c, s) = (cs, sn), (-sn, cs), (-cs, -sn), (sn, -cs)
//                       D = (rho*c, rho*s, z)
//                     (Taylor polynomials: remainders x^11/11! and x^12/12! are below 2e-9 on |x| <= pi/4.)
//                     The remaining 24 bits, wb & 0xffffff, are the uniform number of the acceptance test (H5).
// H3 hot start        s_i = D(wa, wb), (wa, wb) = words (2h, 2h+1), h = i & 1, of Philox(ctr = {i >> 1, 6, 0, 0}, key = seed).
// H4 sweep randoms    one call serves the two sites that are active in a 2x2 block of the xy plane: site (x, y, z) in
//                     half-sweep H = 2t + c(i) takes (wa, wb) = words (2h, 2h+1), h = y & 1, of
//                     Philox(ctr = {g, 5, lo32 H, hi32 H}),  g = (z*(L/2) + (y >> 1))*(L/2) + (x >> 1)
//                     (L even: of the four sites of a block, one per row has the active colour).
// H5 update           proposal s' = D(wa, wb) (uniform, independent of s: symmetric).  Local field
//                     h = ((((s(i-e0) + s(i+e0)) + s(i-e1)) + s(i+e1)) + s(i-e2)) + s(i+e2), per component, in this order.
//                     d = s' - s;  e = d_x*h_x;  e = fma(d_y, h_y, e);  e = fma(d_z, h_z, e)      (ΔE = -e)
//                     accept if e >= 0; else u = float(wb & 0xffffff) * 2^-24 and accept iff u < P(float(β) * e).
// H6 P(a), a < 0      (e^a to about 1e-6 relative)  tt = a * LOG2E; if tt < -64: P = 0; n = rint(tt) (ties to even);
//                     f = tt - n (exact); g = f * LN2; p = 1 + g(1 + g(1/2 + g(1/6 + g(1/24 + g(1/120 + g(1/720 + g/5040))))))
//                     by fma (Horner); P = p * 2^n (exact scaling).
// H7 schedule         S8c.6 verbatim (outer passes, coarse colours, k inner sweeps, fine colours).
// H8 observables      E = -Σ_i Σ_d s_i·s_(i+e_d), M = Σ_i s_i, accumulated in double from the float spins.
//
// Pins (tests/test_heisenberg_oracle.py, `-m "not gpu"`): D against the double-precision closed form;
// P against libm exp; sphere moments; Joyce's exact finite-ring energy (ring of 8; the 2x2 torus = ring
// of 4 with doubled bonds); the high-temperature series in 3D; E of spin spirals (closed form); monotone
// energy in a β = ∞ quench (pins the field against E); schedule invariants.  No function is unpinned.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC heisenberg_oracle.cpp -o liboracle_heisenberg.so

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// Philox4x32-10 (Salmon et al., SC'11), S8c.2 — written out again here on purpose.
void philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

constexpr uint32_t TAG_HSWEEP = 5u, TAG_HINIT = 6u;

// H2.  Constants: the floats nearest to the stated real numbers.
const float PI_4 = (float)0.78539816339744830962;
const float S3 = (float)(-1.0 / 6.0), S5 = (float)(1.0 / 120.0), S7 = (float)(-1.0 / 5040.0), S9 = (float)(1.0 / 362880.0);
const float C2 = (float)(-1.0 / 2.0), C4 = (float)(1.0 / 24.0), C6 = (float)(-1.0 / 720.0), C8 = (float)(1.0 / 40320.0),
            C10 = (float)(-1.0 / 3628800.0);

void direction(uint32_t wa, uint32_t wb, float out[3]) {
    const uint32_t z20 = wa >> 12;
    const uint32_t phi20 = ((wa & 0xfffu) << 8) | (wb >> 24);
    const float z = fmaf((float)z20, 0x1p-19f, -1.0f);
    const float rho = sqrtf(fmaf(-z, z, 1.0f));
    const uint32_t q = phi20 >> 17;
    float t = (float)(phi20 & 0x1ffffu) * 0x1p-17f;
    if (q & 1u) t = t - 1.0f;
    const float x = t * PI_4;
    const float x2 = x * x;
    const float x3 = x2 * x;
    float ps = fmaf(x2, S9, S7);
    ps = fmaf(x2, ps, S5);
    ps = fmaf(x2, ps, S3);
    const float sn = fmaf(x3, ps, x);
    float pc = fmaf(x2, C10, C8);
    pc = fmaf(x2, pc, C6);
    pc = fmaf(x2, pc, C4);
    pc = fmaf(x2, pc, C2);
    const float cs = fmaf(x2, pc, 1.0f);
    float c, s;
    switch (((q + 1u) >> 1) & 3u) {
        case 0: c = cs; s = sn; break;
        case 1: c = -sn; s = cs; break;
        case 2: c = -cs; s = -sn; break;
        default: c = sn; s = -cs; break;
    }
    out[0] = rho * c;
    out[1] = rho * s;
    out[2] = z;
}

// H6.
const float LOG2E = (float)1.4426950408889634074, LN2 = (float)0.69314718055994530942;
const float E2 = (float)(1.0 / 2.0), E3 = (float)(1.0 / 6.0), E4 = (float)(1.0 / 24.0), E5 = (float)(1.0 / 120.0),
            E6 = (float)(1.0 / 720.0), E7 = (float)(1.0 / 5040.0);

float accept_probability(float a) {   // a < 0
    const float tt = a * LOG2E;
    if (tt < -64.0f) return 0.0f;
    const float n = rintf(tt);
    const float f = tt - n;
    const float g = f * LN2;
    float p = fmaf(g, E7, E6);
    p = fmaf(g, p, E5);
    p = fmaf(g, p, E4);
    p = fmaf(g, p, E3);
    p = fmaf(g, p, E2);
    p = fmaf(g, p, 1.0f);
    p = fmaf(g, p, 1.0f);
    const uint32_t bits = (uint32_t)((int)n + 127) << 23;
    float scale;
    std::memcpy(&scale, &bits, 4);
    return p * scale;
}

struct Heis {
    int dim, L;
    uint64_t N;
    uint64_t seed;
    uint64_t t = 0;
    int reverse_tiles = 0;
    std::vector<float> s;   // s[c*N + i]
    uint64_t accepted = 0, attempted = 0;
};

inline void coords(const Heis* h, uint64_t i, int xyz[3]) {
    xyz[0] = (int)(i % h->L);
    xyz[1] = h->dim > 1 ? (int)((i / h->L) % h->L) : 0;
    xyz[2] = h->dim > 2 ? (int)(i / ((uint64_t)h->L * h->L)) : 0;
}

inline uint64_t neighbour(const Heis* h, uint64_t i, int d, int sign) {
    int xyz[3];
    coords(h, i, xyz);
    uint64_t stride = 1;
    for (int a = 0; a < d; ++a) stride *= (uint64_t)h->L;
    const int v = xyz[d];
    const int w = (v + sign + h->L) % h->L;
    return i + (uint64_t)((int64_t)(w - v) * (int64_t)stride);
}

// H5: one Metropolis update of site i in half-sweep H.
void update(Heis* h, uint64_t i, uint64_t H, float betaf) {
    int xyz[3];
    coords(h, i, xyz);
    const uint64_t half_L = (uint64_t)(h->L / 2);
    const uint64_t g = ((uint64_t)xyz[2] * half_L + (uint64_t)(xyz[1] >> 1)) * half_L + (uint64_t)(xyz[0] >> 1);
    const int hw = xyz[1] & 1;
    const uint32_t ctr[4] = {(uint32_t)g, TAG_HSWEEP, (uint32_t)H, (uint32_t)(H >> 32)};
    const uint32_t key[2] = {(uint32_t)h->seed, (uint32_t)(h->seed >> 32)};
    uint32_t w[4];
    philox(ctr, key, w);
    const uint32_t wa = w[2 * hw], wb = w[2 * hw + 1];
    float sp[3];
    direction(wa, wb, sp);
    const uint64_t N = h->N;
    float hf[3];
    for (int c = 0; c < 3; ++c) {
        float acc = h->s[c * N + neighbour(h, i, 0, -1)] + h->s[c * N + neighbour(h, i, 0, +1)];
        for (int d = 1; d < h->dim; ++d) {
            acc = acc + h->s[c * N + neighbour(h, i, d, -1)];
            acc = acc + h->s[c * N + neighbour(h, i, d, +1)];
        }
        hf[c] = acc;
    }
    const float dx = sp[0] - h->s[i], dy = sp[1] - h->s[N + i], dz = sp[2] - h->s[2 * N + i];
    float e = dx * hf[0];
    e = fmaf(dy, hf[1], e);
    e = fmaf(dz, hf[2], e);
    bool acc = e >= 0.0f;
    if (!acc) {
        const float u = (float)(wb & 0xffffffu) * 0x1p-24f;
        acc = u < accept_probability(betaf * e);
    }
    h->attempted++;
    if (acc) {
        h->accepted++;
        h->s[i] = sp[0]; h->s[N + i] = sp[1]; h->s[2 * N + i] = sp[2];
    }
}

}  // namespace

extern "C" {

void horacle_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox(ctr, key, out); }
void horacle_direction(uint32_t w0, uint32_t w1, float* out) { direction(w0, w1, out); }
float horacle_accept_probability(float a) { return accept_probability(a); }

void* horacle_create(int dim, int L, uint64_t seed) {
    if (dim < 1 || dim > 3 || L < 2 || (L & 1)) return nullptr;
    Heis* h = new Heis;
    h->dim = dim; h->L = L; h->seed = seed;
    h->N = 1;
    for (int d = 0; d < dim; ++d) h->N *= (uint64_t)L;
    h->s.resize(3 * h->N);
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    for (uint64_t i = 0; i < h->N; ++i) {   // H3
        const uint32_t ctr[4] = {(uint32_t)(i >> 1), TAG_HINIT, 0u, 0u};
        uint32_t w[4];
        philox(ctr, key, w);
        float v[3];
        direction(w[2 * (i & 1)], w[2 * (i & 1) + 1], v);
        for (int c = 0; c < 3; ++c) h->s[c * h->N + i] = v[c];
    }
    return h;
}

void horacle_destroy(void* p) { delete (Heis*)p; }

// H7 = S8c.6: for pass: for C in {0,1}: for tiles of coarse colour C: for j < k: for c in {0,1}: sites of colour c.
int horacle_sweep(void* p, double beta, int n, int T, int k) {
    Heis* h = (Heis*)p;
    if (!h || n < 0 || k < 1 || !(beta >= 0.0) || !std::isfinite(beta)) return -1;
    if (T == 0) T = h->L;
    if (T < 2 || (T & 1) || h->L % T) return -1;
    const int B = h->L / T;
    if (B != 1 && (B & 1)) return -1;
    const float betaf = (float)beta;
    const int dim = h->dim;
    const int Bz = dim > 2 ? B : 1, By = dim > 1 ? B : 1;
    const int Tz = dim > 2 ? T : 1, Ty = dim > 1 ? T : 1;
    const int64_t ntiles = (int64_t)B * By * Bz;
    for (int pass = 0; pass < n; ++pass) {
        for (int C = 0; C < 2; ++C) {
            for (int64_t q = 0; q < ntiles; ++q) {
                const int64_t tile = h->reverse_tiles ? ntiles - 1 - q : q;
                const int tx = (int)(tile % B), ty = (int)((tile / B) % By), tz = (int)(tile / ((int64_t)B * By));
                if (((tx + ty + tz) & 1) != C) continue;
                for (int j = 0; j < k; ++j) {
                    const uint64_t t = h->t + (uint64_t)pass * k + j;
                    for (int c = 0; c < 2; ++c)
                        for (int lz = 0; lz < Tz; ++lz)
                            for (int ly = 0; ly < Ty; ++ly)
                                for (int lx = 0; lx < T; ++lx) {
                                    const int x = tx * T + lx, y = ty * T + ly, z = tz * T + lz;
                                    if (((x + y + z) & 1) != c) continue;
                                    const uint64_t i = (uint64_t)x + (uint64_t)h->L * ((uint64_t)y + (uint64_t)h->L * z);
                                    update(h, i, 2 * t + c, betaf);
                                }
                }
            }
        }
    }
    h->t += (uint64_t)n * k;
    return 0;
}

// H8
int horacle_observables(void* p, double* E, double* M) {
    Heis* h = (Heis*)p;
    if (!h) return -1;
    const uint64_t N = h->N;
    double e = 0.0, m[3] = {0, 0, 0};
    for (uint64_t i = 0; i < N; ++i) {
        for (int d = 0; d < h->dim; ++d) {
            const uint64_t j = neighbour(h, i, d, +1);
            for (int c = 0; c < 3; ++c) e -= (double)h->s[c * N + i] * (double)h->s[c * N + j];
        }
        for (int c = 0; c < 3; ++c) m[c] += (double)h->s[c * N + i];
    }
    if (E) *E = e;
    if (M) { M[0] = m[0]; M[1] = m[1]; M[2] = m[2]; }
    return 0;
}

int horacle_copy_spins(void* p, float* dst) {
    Heis* h = (Heis*)p;
    if (!h || !dst) return -1;
    std::memcpy(dst, h->s.data(), 3 * h->N * sizeof(float));
    return 0;
}

int horacle_set_spins(void* p, const float* src) {
    Heis* h = (Heis*)p;
    if (!h || !src) return -1;
    std::memcpy(h->s.data(), src, 3 * h->N * sizeof(float));
    return 0;
}

uint64_t horacle_get_counter(void* p) { return ((Heis*)p)->t; }
void horacle_set_counter(void* p, uint64_t t) { ((Heis*)p)->t = t; }
void horacle_set_tile_order(void* p, int reverse) { ((Heis*)p)->reverse_tiles = reverse; }
void horacle_acceptance(void* p, uint64_t* accepted, uint64_t* attempted) {
    Heis* h = (Heis*)p;
    *accepted = h->accepted; *attempted = h->attempted;
}

}  // extern "C"
