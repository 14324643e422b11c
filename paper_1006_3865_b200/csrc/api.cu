// api.cu — the C ABI of include/ising.h: argument checking, the host-side acceptance table
// (a2), storage-layout bookkeeping and kernel-path selection.  All compute is in the
// kernels of generic.cu / tile_i8.cu / tile_planes.cu / tile3d_planes.cu / amsc.cu; there is no CPU path.
#include <cmath>
#include <cstdarg>
#include <cstring>
#include <atomic>
#include <mutex>
#include <new>
#include <string>
#include <unordered_map>

#include "kernels.h"

namespace ising {

static thread_local char g_err[512] = "";
static std::atomic<uint64_t> g_launches{0};

Hooks& hooks() {
    static Hooks h;
    return h;
}

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

void count_launch(uint64_t n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

// Every block is released through the hook that was installed when it was allocated (nullptr = cudaFree), whatever
// ising_set_device_hooks has been called with in between: the owner is remembered per pointer.
static std::mutex g_owner_mu;
static std::unordered_map<void*, void (*)(void*)>& owners() {
    static std::unordered_map<void*, void (*)(void*)> m;
    return m;
}

void* dev_alloc(size_t bytes) {
    if (bytes == 0) bytes = 16;
    void* p = nullptr;
    void (*owner)(void*) = nullptr;
    if (hooks().alloc) {
        owner = hooks().dealloc;
        p = hooks().alloc(bytes);
        if (!p) { set_error("device allocation hook returned NULL for %zu bytes", bytes); return nullptr; }
    } else {
        cudaError_t e = cudaMalloc(&p, bytes);
        if (e != cudaSuccess) {
            set_error("cudaMalloc(%zu) failed: %s", bytes, cudaGetErrorString(e));
            return nullptr;
        }
    }
    try {
        std::lock_guard<std::mutex> lock(g_owner_mu);
        owners()[p] = owner;
    } catch (...) {                          // cannot remember the owner: give the block back now rather than leak or mis-free it
        if (owner) owner(p); else cudaFree(p);
        set_error("out of host memory while recording a device allocation");
        return nullptr;
    }
    return p;
}

void dev_free(void* p) {
    if (!p) return;
    void (*owner)(void*) = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_owner_mu);
        auto it = owners().find(p);
        if (it != owners().end()) { owner = it->second; owners().erase(it); }
    }
    if (owner) owner(p);
    else cudaFree(p);
}

static bool is_device_ptr(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

static int have_device() {
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n < 1) {
        cudaGetLastError();
        set_error("no CUDA device: libising_b200 has no CPU path (%s)",
                  e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
        return ISING_ECUDA;
    }
    return 0;
}

// a2 / S8c.4: thr[m] = floor(exp(-β·4m)·2^32) in double, m = 1..dim.
static void threshold_table(double beta, int dim, uint64_t thr[3]) {
    for (int m = 1; m <= 3; ++m)
        thr[m - 1] = (m <= dim) ? (uint64_t)std::floor(std::exp(-beta * 4.0 * (double)m) * 4294967296.0) : 0;
}

static Accept make_accept(double beta, int dim) {
    uint64_t thr[3];
    threshold_table(beta, dim, thr);
    Accept a;
    a.always = 0;
    for (int m = 0; m < 3; ++m) {
        a.thr_is_2p32[m] = (m < dim && thr[m] >= 4294967296ull) ? 1u : 0u;
        a.thr[m] = a.thr_is_2p32[m] ? 0xffffffffu : (uint32_t)thr[m];
        a.cneg[m] = 0;
        if (m >= dim) continue;
        if (thr[m] == 0) a.always += 1;                       // r >= 0 always
        else if (!a.thr_is_2p32[m]) a.cneg[m] = (uint32_t)(4294967296ull - thr[m]);
    }
    return a;
}

static bool tile_valid(const ising_ctx* h, int T) {
    if (T < 2 || (T & 1) || h->L % T) return false;
    const int B = h->L / T;
    return B == 1 || (B % 2 == 0);
}

// ---- storage bookkeeping --------------------------------------------------------------
static int to_canon_scratch_now(ising_ctx* h) {   // tiles -> d_canon, store state unchanged
    switch (h->store) {
        case Store::TileI8: return launch_tile_i8_to_canon(h, h->store_tile, h->d_tiles, h->d_canon);
        case Store::PlaneI8: return launch_planes_to_canon(h, h->store_tile, false, h->d_tiles, h->d_canon);
        case Store::PlaneBits: return launch_planes_to_canon(h, h->store_tile, true, h->d_tiles, h->d_canon);
        case Store::Plane3I8: return launch_3d_to_canon(h, false, h->d_tiles, h->d_canon);
        case Store::Plane3Bits: return launch_3d_to_canon(h, true, h->d_tiles, h->d_canon);
        case Store::Amsc: return launch_amsc_to_canon(h, h->d_tiles, h->d_canon);
        default: return 0;
    }
}

// ... unless d_canon already holds the current state (read-only calls in a row convert once: ising_copy_spins,
// ising_overlap, ising_copy_spins_bits; every writer of the tile records bumps state_version)
static int to_canon_scratch(ising_ctx* h) {
    if (h->store == Store::Canon) return 0;
    if (h->sweeping) {                        // measuring between the passes of one call: the records change pass by pass
        h->canon_version = 0;
        return to_canon_scratch_now(h);
    }
    if (h->canon_version == h->state_version) return 0;
    const int rc = to_canon_scratch_now(h);
    h->canon_version = rc ? 0 : h->state_version;
    return rc;
}

static int ensure_canon(ising_ctx* h) {
    if (h->store == Store::Canon) return 0;
    const int rc = to_canon_scratch(h);
    if (rc) return rc;
    h->store = Store::Canon;
    h->store_tile = 0;
    return 0;
}

// Bring the spins into tile records of `kind` for tile edge T (re-laid out through the canonical array).
static int ensure_store(ising_ctx* h, Store kind, int T) {
    if (h->store == kind && h->store_tile == T) return 0;
    int rc = ensure_canon(h);
    if (rc) return rc;
    const bool is3 = kind == Store::Plane3I8 || kind == Store::Plane3Bits;
    const size_t need = kind == Store::Amsc ? amsc_spin_bytes(h)
                        : kind == Store::TileI8 ? tile_i8_bytes(h, T)
                        : is3 ? tile3d_bytes(h, kind == Store::Plane3Bits)
                              : tile_planes_bytes(h, T, kind == Store::PlaneBits);
    if (need > h->tiles_bytes) {
        ISING_CUDA_OK(cudaStreamSynchronize(hooks().stream));
        dev_free(h->d_tiles);
        h->tiles_bytes = 0;
        h->d_tiles = dev_alloc(need);
        if (!h->d_tiles) return ISING_ENOMEM;
        h->tiles_bytes = need;
    }
    rc = kind == Store::Amsc ? launch_canon_to_amsc(h, h->d_canon, h->d_tiles)
         : kind == Store::TileI8 ? launch_canon_to_tile_i8(h, T, h->d_canon, h->d_tiles)
         : is3 ? launch_canon_to_3d(h, kind == Store::Plane3Bits, h->d_canon, h->d_tiles)
               : launch_canon_to_planes(h, T, kind == Store::PlaneBits, h->d_canon, h->d_tiles);
    if (rc) return rc;
    h->store = kind;
    h->store_tile = T;
    h->canon_version = h->state_version;         // d_canon still holds this very state
    return 0;
}

// a10 wherever the spins currently live: directly on 2D plane records, else on the canonical array.
static int observables_now(ising_ctx* h, long long* d_E, long long* d_M) {
    const bool planes2d = (h->store == Store::PlaneI8 || h->store == Store::PlaneBits) && h->L / h->store_tile >= 2 &&
                          (!h->has_J || h->Jtiles_tile == h->store_tile);
    if (planes2d) return launch_observables_planes(h, h->store_tile, h->store == Store::PlaneBits, d_E, d_M);
    const bool planes3d = (h->store == Store::Plane3I8 || h->store == Store::Plane3Bits) && (!h->has_J || h->Jtiles_tile == h->store_tile);
    if (planes3d) return launch_observables3d(h, h->store == Store::Plane3Bits, d_E, d_M);
    int rc = (h->store == Store::Canon) ? 0 : to_canon_scratch(h);
    if (rc) return rc;
    return launch_observables_canon(h, h->d_canon, d_E, d_M);
}

static const int8_t* canon_view(ising_ctx* h, int* rc) {
    *rc = (h->store == Store::Canon) ? 0 : to_canon_scratch(h);
    return h->d_canon;
}

static int copy_out(void* dst, const void* d_src, size_t bytes, bool* synced) {
    cudaStream_t st = hooks().stream;
    const bool dev = is_device_ptr(dst);
    ISING_CUDA_OK(cudaMemcpyAsync(dst, d_src, bytes, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st));
    ISING_CUDA_OK(cudaStreamSynchronize(st));
    if (synced) *synced = true;
    return 0;
}

}  // namespace ising

using namespace ising;

extern "C" {

const char* ising_last_error(void) { return g_err; }
uint64_t ising_kernel_launches(void) { return g_launches.load(); }

int ising_set_device_hooks(void* (*alloc)(size_t), void (*dealloc)(void*), void* cuda_stream) {
    if ((alloc == nullptr) != (dealloc == nullptr)) {
        set_error("ising_set_device_hooks: alloc and dealloc must both be set or both be NULL");
        return ISING_EINVAL;
    }
    hooks().alloc = alloc;
    hooks().dealloc = dealloc;
    hooks().stream = (cudaStream_t)cuda_stream;
    return 0;
}

int ising_thresholds(double beta, int dim, uint64_t* out) {
    if (!out || (dim != 2 && dim != 3) || !(beta >= 0.0) || !std::isfinite(beta)) {
        set_error("ising_thresholds: need dim in {2,3}, finite beta >= 0, out != NULL");
        return ISING_EINVAL;
    }
    threshold_table(beta, dim, out);
    return 0;
}

void ising_destroy(ising_handle h) {
    if (!h) return;
    cudaStreamSynchronize(hooks().stream);
    dev_free(h->d_J);
    if (h->d_sweep_seeds != h->d_seeds) dev_free(h->d_sweep_seeds);
    dev_free(h->d_seeds);
    dev_free(h->d_canon);
    dev_free(h->d_tiles);
    dev_free(h->d_Jtiles);
    dev_free(h->d_amsc_J);
    dev_free(h->d_xedge);
    dev_free(h->d_gacc);
    dev_free(h->d_obs);
    dev_free(h->d_pair);
    dev_free(h->d_flag);
    delete h;
}

static ising_handle create_impl(int dim, int L, const int8_t* J, const uint64_t* seeds, int R, bool multi, uint64_t sweep_seed) {
    if ((dim != 2 && dim != 3) || L < 2 || (L & 1) || R < 1 || !seeds) {
        set_error("ising_create: need dim in {2,3}, even L >= 2, n_replicas >= 1, seeds != NULL "
                  "(got dim=%d L=%d R=%d)", dim, L, R);
        return nullptr;
    }
    uint64_t N = 1;
    for (int d = 0; d < dim; ++d) N *= (uint64_t)L;
    if (N > (1ull << 32)) {
        set_error("ising_create: N = L^dim = %llu exceeds 2^32", (unsigned long long)N);
        return nullptr;
    }
    if (have_device()) return nullptr;
    ising_ctx* h = new (std::nothrow) ising_ctx;
    if (!h) return nullptr;
    h->dim = dim; h->L = L; h->R = R; h->N = N;
    try {
        h->seeds.assign(seeds, seeds + R);
    } catch (...) {
        delete h;
        set_error("ising_create: out of host memory");
        return nullptr;
    }
    h->J_per_replica = multi; h->shared_sweep = multi; h->sweep_seed = sweep_seed;
    if (multi) h->rng = ISING_RNG_WORDS;     // one random word per site serves every realisation (ising.h)
    cudaStream_t st = hooks().stream;
    auto fail = [&](void) -> ising_handle { ising_destroy(h); return nullptr; };
    h->d_seeds = (uint64_t*)dev_alloc(sizeof(uint64_t) * R);
    h->d_canon = (int8_t*)dev_alloc((size_t)R * N);
    h->d_obs = (long long*)dev_alloc(sizeof(long long) * (2 * (size_t)R + 2));
    h->d_flag = (int*)dev_alloc(sizeof(int));
    if (!h->d_seeds || !h->d_canon || !h->d_obs || !h->d_flag) return fail();
    if (cudaMemcpyAsync(h->d_seeds, h->seeds.data(), sizeof(uint64_t) * R, cudaMemcpyHostToDevice, st) != cudaSuccess) {
        set_error("ising_create: seed upload failed: %s", cudaGetErrorString(cudaGetLastError()));
        return fail();
    }
    h->d_sweep_seeds = h->d_seeds;
    if (multi) {                                       // R copies of the shared sweep key (R17)
        h->d_sweep_seeds = (uint64_t*)dev_alloc(sizeof(uint64_t) * R);
        if (!h->d_sweep_seeds) return fail();
        std::vector<uint64_t> ks;
        try { ks.assign((size_t)R, sweep_seed); } catch (...) { set_error("ising_create_multi: out of host memory"); return fail(); }
        if (cudaMemcpyAsync(h->d_sweep_seeds, ks.data(), sizeof(uint64_t) * R, cudaMemcpyHostToDevice, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess) {
            set_error("ising_create_multi: seed upload failed: %s", cudaGetErrorString(cudaGetLastError()));
            return fail();
        }
    }
    if (J) {
        const size_t jb = (size_t)dim * N * (multi ? (size_t)R : 1);
        h->d_J = (int8_t*)dev_alloc(jb);
        if (!h->d_J) return fail();
        const bool dev = is_device_ptr(J);
        if (cudaMemcpyAsync(h->d_J, J, jb, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st) != cudaSuccess) {
            set_error("ising_create: coupling upload failed: %s", cudaGetErrorString(cudaGetLastError()));
            return fail();
        }
        int bad = 0;
        if (launch_validate_pm1(h->d_J, jb, h->d_flag, &bad)) return fail();
        if (bad) {
            set_error("ising_create: couplings must be +1 or -1");
            return fail();
        }
        h->has_J = true;
    }
    if (launch_hot_start(h)) return fail();
    if (cudaStreamSynchronize(st) != cudaSuccess) {   // seeds vector may go away; surface errors here
        set_error("ising_create: %s", cudaGetErrorString(cudaGetLastError()));
        return fail();
    }
    return h;
}

ising_handle ising_create_batch(int dim, int L, const int8_t* J, const uint64_t* seeds, int R) {
    return create_impl(dim, L, J, seeds, R, false, 0);
}

ising_handle ising_create_multi(int dim, int L, const int8_t* couplings, const uint64_t* init_seeds, int R, uint64_t sweep_seed) {
    if (!couplings) {
        set_error("ising_create_multi: couplings must not be NULL (R*dim*N values)");
        return nullptr;
    }
    return create_impl(dim, L, couplings, init_seeds, R, true, sweep_seed);
}

ising_handle ising_create(int dim, int L, const int8_t* J, uint64_t seed) {
    return ising_create_batch(dim, L, J, &seed, 1);
}

}  // extern "C"

// ---- sweeps ---------------------------------------------------------------------------
// One ising_sweep / ising_sweep_series call.  Kernel families are tried in the order of kPaths: each entry either does not
// apply (kSkip: the next one is asked), or runs the whole call (kDone), or fails (a negative ISING_E* code).
namespace {

struct SweepCall {
    ising_ctx* h;
    Accept acc;
    int n, T, k;
    long long *d_E, *d_M;          // series outputs on the device (or nullptr)
    bool want_series, bits, thr_fits;
    cudaStream_t st;
    int Tc2, Tc3;                  // coarse tile edge of a masked double checkerboard on the 2D / 3D register tiling, or 0
};
constexpr int kSkip = 1, kDone = 0;

// last_path strings live for the life of the process: "<family>_<i8|bits>"
const char* path_name(const char* family, bool bits) {
    static std::mutex mu;
    static std::unordered_map<std::string, std::string>* names = new std::unordered_map<std::string, std::string>();
    try {
        std::lock_guard<std::mutex> lock(mu);
        std::string key = std::string(family) + (bits ? "_bits" : "_i8");
        return names->emplace(key, key).first->second.c_str();
    } catch (...) {
        return family;
    }
}

// coupling records (a9) in the form of the tile records in use: built once per (kind, tile edge)
int ensure_couplings(ising_ctx* h, bool three_d, int T) {
    if (!h->has_J || (h->Jtiles_tile == T && h->Jtiles_kind == (three_d ? 3 : 2))) return 0;
    const size_t need = three_d ? coupling_record3d_bytes(h) : coupling_record_bytes(h);
    if (need > h->Jtiles_bytes) {
        cudaStreamSynchronize(hooks().stream);
        dev_free(h->d_Jtiles); h->d_Jtiles = nullptr; h->Jtiles_bytes = 0; h->Jtiles_tile = 0;
        h->d_Jtiles = dev_alloc(need);
        if (!h->d_Jtiles) return ISING_ENOMEM;
        h->Jtiles_bytes = need;
    }
    h->Jtiles_tile = 0;
    const int rc = three_d ? launch_convert_couplings3d(h, h->d_Jtiles) : launch_convert_couplings(h, T, h->d_Jtiles);
    if (rc) return rc;
    h->Jtiles_tile = T; h->Jtiles_kind = three_d ? 3 : 2;
    return 0;
}

int ensure_scratch(void** p, size_t* have, size_t need) {
    if (need <= *have) return 0;
    cudaStreamSynchronize(hooks().stream);
    dev_free(*p); *p = nullptr; *have = 0;
    *p = dev_alloc(need);
    if (!*p) return ISING_ENOMEM;
    *have = need;
    return 0;
}

// n passes, one launcher call per pass, E and M measured on the records after each pass if a series is wanted
template <class Launch>
int per_pass(const SweepCall& c, Launch launch) {
    ising_ctx* h = c.h;
    int rc = 0;
    for (int pass = 0; pass < c.n && !rc; ++pass) {
        rc = launch(h->t + (uint64_t)pass * (uint64_t)c.k);
        if (!rc && c.want_series)
            rc = observables_now(h, c.d_E ? c.d_E + (size_t)pass * h->R : nullptr, c.d_M ? c.d_M + (size_t)pass * h->R : nullptr);
    }
    return rc;
}

bool planes_rng(const SweepCall& c) { return !c.h->force_generic && c.h->rng == ISING_RNG_PLANES; }
bool onchip_ok(const ising_ctx* h) { return !h->no_resident && !h->no_onchip; }

// f1: asynchronous multi-spin coding, 32 realisations per word, one random number per site
int path_amsc(SweepCall& c) {
    ising_ctx* h = c.h;
    if (h->force_generic || !amsc_supported(h, c.T)) return kSkip;
    h->last_path = "amsc";
    int rc = 0;
    if (!h->d_amsc_J) {
        h->d_amsc_J = dev_alloc(amsc_bond_bytes(h));
        if (!h->d_amsc_J) return ISING_ENOMEM;
        rc = launch_amsc_pack_J(h, h->d_amsc_J);
        if (rc) { dev_free(h->d_amsc_J); h->d_amsc_J = nullptr; return rc; }      // never sweep on half-packed bonds
    }
    rc = ensure_store(h, Store::Amsc, 0);
    if (rc) return rc;
    return per_pass(c, [&](uint64_t t0) { return launch_amsc_pass(h, c.acc, c.T, c.k, t0, h->d_amsc_J); });
}

// a8, config 1: the 64 x 64 plain checkerboard, the whole run in one launch, E / M measured in the kernel
int path_plain64(SweepCall& c) {
    ising_ctx* h = c.h;
    if (!planes_rng(c) || !plain64_supported(h, c.T)) return kSkip;
    h->last_path = path_name("plain64_planes", c.bits);
    int rc = ensure_store(h, c.bits ? Store::PlaneBits : Store::PlaneI8, c.T);
    if (!rc) rc = ensure_couplings(h, false, c.T);
    if (!rc && c.n > 0) rc = launch_plain64(h, c.acc, c.bits, c.n, c.k, h->t, c.d_E, c.d_M);
    return rc;
}

// a8 beyond L = 64 (tile == L) and the double checkerboard of coarse tiles other than the register tiles (the paper's
// T = 2 ... 16; 128, 256, ...) as masked half-sweeps, 2D: cluster-resident if the lattice is small, else a launch
// per half-sweep.  The register tiling Tp is invisible in the result.
int path_plain2d(SweepCall& c) {
    ising_ctx* h = c.h;
    if (!planes_rng(c) || h->dim != 2 || c.n <= 0 || !(c.T == h->L || c.Tc2)) return kSkip;
    int Tp = 0;
    if (onchip_ok(h)) Tp = resident_planes_supported(h, 32) ? 32 : (resident_planes_supported(h, 64) ? 64 : 0);
    const bool resident = Tp != 0;
    if (!Tp) Tp = tile_planes_supported(h, 64) ? 64 : (tile_planes_supported(h, 32) ? 32 : 0);
    if (!Tp) return kSkip;
    // k_grid_plain (below) wants the 32 x 32 register tiling: at 64 x 64 its unspecialised compare spills under the 72 registers of
    // 28 warps per SM
    // (measured: with every tile exchanging its boundary after every half-sweep the on-chip form wins up to
    // 2^24 sites — 1.3 ... 2.3 x — and loses to the launch per half-sweep from 2^26 on, where that one is HBM-bound at 70 %)
    const bool grid_ok = !resident && !c.want_series && onchip_ok(h) && (uint64_t)c.n * (uint64_t)c.k * (c.Tc2 ? 2u : 1u) >= 4u &&
                         (uint64_t)h->R * h->N <= (1ull << 24);
    static const int plain_T = getenv("ISING_GRID_PLAIN_T") ? atoi(getenv("ISING_GRID_PLAIN_T")) : 32;       // tuning aid
    if (grid_ok && tile_planes_supported(h, plain_T) && grid_planes_supported(h, plain_T)) Tp = plain_T;
    else if (!resident && (h->store == Store::PlaneI8 || h->store == Store::PlaneBits) && (h->store_tile == 32 || h->store_tile == 64) &&
             tile_planes_supported(h, h->store_tile))
        Tp = h->store_tile;          // short calls and series between long ones: keep the register tiling the records are in
    int rc = ensure_store(h, c.bits ? Store::PlaneBits : Store::PlaneI8, Tp);
    if (!rc) rc = ensure_couplings(h, false, Tp);
    if (rc) return rc;
    if (resident) {
        if (launch_resident_planes(h, c.acc, Tp, c.bits, c.n, c.k, h->t, c.d_E, c.d_M, true, c.Tc2) == 0) {
            h->last_path = path_name(c.Tc2 ? "resident_masked" : "resident_plain", c.bits);
            return kDone;
        }
        cudaGetLastError();          // the cluster did not fit: a launch per half-sweep
    }
    // beyond the cluster, while the lattice fits the shared memory of the GPU: every half-sweep of the call in one cooperative
    // launch (k_grid_plain); a call of a few half-sweeps does not pay for loading and storing the lattice once
    if (grid_ok && grid_planes_supported(h, Tp)) {
        rc = ensure_scratch(&h->d_xedge, &h->xedge_bytes, grid_plain_xedge_bytes(h, Tp));
        if (rc) return rc;
        const int g = launch_grid_plain(h, c.acc, Tp, c.bits, c.n, c.k, h->t, c.Tc2, h->d_xedge);
        if (g == 0) { h->last_path = path_name(c.Tc2 ? "grid_masked" : "grid_plain", c.bits); return kDone; }
        if (g != 1) return g;
    }
    h->last_path = path_name(c.Tc2 ? "tile_masked" : "tile_plain", c.bits);
    return per_pass(c, [&](uint64_t t0) { return launch_tile_planes_plain(h, c.acc, Tp, c.bits, 1, c.k, t0, c.Tc2); });
}

// the same in 3D: 8^3 register tiles, cluster-resident up to L = 64, else a launch per half-sweep
int path_plain3d(SweepCall& c) {
    ising_ctx* h = c.h;
    if (!planes_rng(c) || h->dim != 3 || c.n <= 0 || !(c.T == h->L || c.Tc3) || !tile3d_supported(h, 8)) return kSkip;
    int rc = ensure_store(h, c.bits ? Store::Plane3Bits : Store::Plane3I8, 8);
    if (!rc) rc = ensure_couplings(h, true, 8);
    if (rc) return rc;
    if (onchip_ok(h) && resident3d_supported(h, 8)) {
        if (launch_resident3d(h, c.acc, c.bits, c.n, c.k, h->t, c.d_E, c.d_M, true, c.Tc3) == 0) {
            h->last_path = path_name(c.Tc3 ? "resident3d_masked" : "resident3d_plain", c.bits);
            return kDone;
        }
        cudaGetLastError();
    }
    h->last_path = path_name(c.Tc3 ? "tile3d_masked" : "tile3d_plain", c.bits);
    return per_pass(c, [&](uint64_t t0) { return launch_tile3d_plain(h, c.acc, c.bits, 1, c.k, t0, c.Tc3); });
}

// a1-a7 on the 2D register tiles 32 / 64 (planes mapping): one launch per call where that pays — cluster-resident (small
// lattices), grid-resident (lattices that fit on chip), data-flow (HBM-resident, k = 1) — else a launch per coarse colour
int path_tiled2d(SweepCall& c) {
    ising_ctx* h = c.h;
    if (!planes_rng(c) || !tile_planes_supported(h, c.T)) return kSkip;
    const int T = c.T, n = c.n, k = c.k;
    int rc = ensure_store(h, c.bits ? Store::PlaneBits : Store::PlaneI8, T);
    if (!rc) rc = ensure_couplings(h, false, T);
    if (rc) return rc;
    // run-time specialisation pays for its ~1 s of compilation only on big calls (AUTO: >= 2^27 attempted flips)
    const bool use_jit = h->jit_mode == ISING_JIT_ON || (h->jit_mode == ISING_JIT_AUTO && (double)n * k * (double)h->N * h->R >= 134217728.0);
    h->last_jit = 0;
    if (n >= 2 && onchip_ok(h)) {
        if (resident_planes_supported(h, T)) {
            // small lattices: one thread-block cluster per replica (no specialised form: not when the caller insists on one)
            if (h->jit_mode != ISING_JIT_ON) {
                if (launch_resident_planes(h, c.acc, T, c.bits, n, k, h->t, c.d_E, c.d_M, false, 0) == 0) {
                    h->last_path = path_name("resident_planes", c.bits);
                    return kDone;
                }
                cudaGetLastError();      // the cluster did not fit (shared or partitioned GPU): a launch per colour instead
            }
        } else if (grid_planes_supported(h, T)) {
            // beyond the cluster, still on chip: one cooperative launch on all SMs, boundary words through L2 (k_grid_planes)
            rc = ensure_scratch(&h->d_xedge, &h->xedge_bytes, grid_planes_xedge_bytes(h, T));
            if (!rc && c.want_series) rc = ensure_scratch(&h->d_gacc, &h->gacc_bytes, grid_planes_acc_bytes(h, n));
            if (rc) return rc;
            const int g = launch_grid_planes(h, c.acc, T, c.bits, n, k, h->t, h->d_xedge, h->d_gacc, c.d_E, c.d_M, use_jit, h->jit_mode != ISING_JIT_ON);
            if (g == 0) { h->last_path = path_name("grid_planes", c.bits); return kDone; }
            if (g != 1) cudaGetLastError();      // the cooperative launch was refused (shared or partitioned GPU)
        }
    }
    // HBM-resident lattices, several passes, nothing to measure in between, int8 records at k = 1 (the HBM-bound case): one
    // persistent launch, colours ordered by data flow (k_flow_planes: +2.5 % at L = 16384, +5 % at L = 8192; for k >= 2 the
    // register budget of the persistent loop costs more than the idle launch tails it removes, and bit records gain nothing)
    if (!c.want_series && !h->no_resident && !h->no_flow && ((k == 1 && !c.bits) || h->no_onchip) && flow_planes_supported(h, T, n)) {
        rc = ensure_scratch(&h->d_xedge, &h->xedge_bytes, flow_planes_scratch_bytes(h, T));
        if (rc) return rc;
        if (launch_flow_planes(h, c.acc, T, c.bits, n, k, h->t, h->d_xedge, use_jit) == 0) {
            h->last_path = path_name("flow_planes", c.bits);
            return kDone;
        }
        cudaGetLastError();
    }
    h->last_path = path_name("tile_planes", c.bits);
    return per_pass(c, [&](uint64_t t0) { return launch_tile_planes_pass(h, c.acc, T, c.bits, k, t0, use_jit); });
}

// the same on the 3D 8^3 register tiles
int path_tiled3d(SweepCall& c) {
    ising_ctx* h = c.h;
    if (!planes_rng(c) || !tile3d_supported(h, c.T)) return kSkip;
    const int T = c.T, n = c.n, k = c.k;
    int rc = ensure_store(h, c.bits ? Store::Plane3Bits : Store::Plane3I8, T);
    if (!rc) rc = ensure_couplings(h, true, T);
    if (rc) return rc;
    const bool use_jit = h->jit_mode == ISING_JIT_ON || (h->jit_mode == ISING_JIT_AUTO && (double)n * k * (double)h->N * h->R >= 134217728.0);
    h->last_jit = 0;
    if (n >= 2 && onchip_ok(h)) {
        if (resident3d_supported(h, T)) {
            if (h->jit_mode != ISING_JIT_ON) {
                if (launch_resident3d(h, c.acc, c.bits, n, k, h->t, c.d_E, c.d_M, false, 0) == 0) {
                    h->last_path = path_name("resident3d_planes", c.bits);
                    return kDone;
                }
                cudaGetLastError();
            }
        } else if (grid3d_supported(h, T) && ((use_jit && !h->has_J) || k < 4 || (uint64_t)h->R * h->N / 1024u <= 148u * 20u)) {
            // The run-time build of k_grid3d takes the CTA shape the lattice wants and wins at every k (config 4, k = 16:
            // 3030 against 2720 flips/ns); the pre-compiled one with two jobs of a colour per warp loses 5 % to the
            // per-pass kernels at k >= 4.
            rc = ensure_scratch(&h->d_xedge, &h->xedge_bytes, grid3d_xedge_bytes(h));
            if (!rc && c.want_series) rc = ensure_scratch(&h->d_gacc, &h->gacc_bytes, grid3d_acc_bytes(h, n));
            if (rc) return rc;
            const int g = launch_grid3d(h, c.acc, c.bits, n, k, h->t, h->d_xedge, h->d_gacc, c.d_E, c.d_M, use_jit);
            if (g == 0) { h->last_path = path_name("grid3d_planes", c.bits); return kDone; }
            if (g != 1) cudaGetLastError();
        }
    }
    h->last_path = path_name("tile3d_planes", c.bits);
    return per_pass(c, [&](uint64_t t0) { return launch_tile3d_pass(h, c.acc, c.bits, k, t0, use_jit); });
}

// words mapping, int8 row-major tile records (SURVEY's normative mapping)
int path_tile_i8(SweepCall& c) {
    ising_ctx* h = c.h;
    if (h->force_generic || !c.thr_fits || h->rng != ISING_RNG_WORDS || h->layout != ISING_LAYOUT_I8 || !tile_i8_supported(h, c.T)) return kSkip;
    h->last_path = "tile_i8";
    const int rc = ensure_store(h, Store::TileI8, c.T);
    if (rc) return rc;
    return per_pass(c, [&](uint64_t t0) { return launch_tile_i8_pass(h, c.acc, c.T, c.k, t0); });
}

// everything else: global-memory kernels on the canonical array (correct, not fast; never a CPU path)
int path_generic(SweepCall& c) {
    ising_ctx* h = c.h;
    if (h->layout != ISING_LAYOUT_I8 && !h->force_generic) {
        set_error("ising_sweep: no bit-packed kernel for dim=%d L=%d tile=%d rng=%d", h->dim, h->L, c.T, h->rng);
        return ISING_EUNSUPPORTED;
    }
    h->last_path = "generic";
    const int rc = ensure_canon(h);
    if (rc) return rc;
    return launch_generic_sweep(h, c.acc, c.n, c.T, c.k, c.d_E, c.d_M);
}

typedef int (*SweepPath)(SweepCall&);
const SweepPath kPaths[] = {path_amsc, path_plain64, path_plain2d, path_plain3d, path_tiled2d, path_tiled3d, path_tile_i8, path_generic};

}  // namespace

static int sweep_impl(ising_handle h, double beta, int n, int tile, int k, int64_t* E, int64_t* M) {
    if (!h) { set_error("ising_sweep: NULL handle"); return ISING_EINVAL; }
    const int T = (tile == 0) ? h->L : tile;
    if (!tile_valid(h, T)) {
        set_error("ising_sweep: tile=%d invalid for L=%d (need T even, T | L, L/T even or T == L)", tile, h->L);
        return ISING_EINVAL;
    }
    if (k < 1 || n < 0 || !(beta >= 0.0) || !std::isfinite(beta)) {
        set_error("ising_sweep: need k_inner >= 1, n_sweeps >= 0, finite beta >= 0");
        return ISING_EINVAL;
    }
    SweepCall c;
    c.h = h; c.acc = make_accept(beta, h->dim); c.n = n; c.T = T; c.k = k;
    c.st = hooks().stream;
    c.bits = h->layout == ISING_LAYOUT_BITS;
    c.want_series = (E != nullptr) || (M != nullptr);
    c.d_E = c.d_M = nullptr;
    struct Sweeping {                         // while passes are being launched no cached canonical copy is valid
        ising_ctx* h; bool on;
        ~Sweeping() { h->sweeping = false; if (on) ++h->state_version; }
    } sweeping{h, n > 0};
    h->sweeping = n > 0;
    const size_t cnt = (size_t)n * h->R;
    long long* tmp = nullptr;
    const bool E_dev = E && is_device_ptr(E), M_dev = M && is_device_ptr(M);
    if (c.want_series && cnt) {
        const size_t need = ((E && !E_dev) ? cnt : 0) + ((M && !M_dev) ? cnt : 0);
        if (need) {
            tmp = (long long*)dev_alloc(need * sizeof(long long));
            if (!tmp) return ISING_ENOMEM;
        }
        long long* q = tmp;
        if (E) { c.d_E = E_dev ? (long long*)E : q; if (!E_dev) q += cnt; }
        if (M) { c.d_M = M_dev ? (long long*)M : q; }
    }
    const Accept& acc = c.acc;
    c.thr_fits = !(acc.thr_is_2p32[0] || acc.thr_is_2p32[1] || acc.thr_is_2p32[2]);   // beta = 0 only
    // 0 < beta < ~1.4e-17: thr[1] rounds to 2^32 while thr[2] (thr[3]) is 2^32 - 1.  The multi-spin kernels fold "2^32" into one
    // all-or-nothing mask, so that case (the accept decision differs for r = 0xffffffff only) goes to the generic kernels,
    // which compare every threshold on its own
    bool thr_mixed = false;
    for (int m = 1; m < h->dim; ++m) thr_mixed = thr_mixed || (acc.thr_is_2p32[m] != acc.thr_is_2p32[0]);
    struct ForceGeneric {
        ising_ctx* h; int saved;
        ~ForceGeneric() { h->force_generic = saved; }
    } fg{h, h->force_generic};
    if (thr_mixed) h->force_generic = 1;
    const bool pow2 = T >= 2 && (T & (T - 1)) == 0 && T != h->L;
    c.Tc2 = (pow2 && T != 32 && T != 64) ? T : 0;
    c.Tc3 = (h->dim == 3 && pow2 && T != 8) ? T : 0;
    int rc = kSkip;
    for (SweepPath path : kPaths) {
        rc = path(c);
        if (rc != kSkip) break;
    }
    if (!rc) h->t += (uint64_t)n * (uint64_t)k;
    if (!rc && tmp) {
        long long* q = tmp;
        if (E && !E_dev) { rc = copy_out(E, q, cnt * sizeof(long long), nullptr); q += cnt; }
        if (!rc && M && !M_dev) rc = copy_out(M, q, cnt * sizeof(long long), nullptr);
    }
    if (tmp) { cudaStreamSynchronize(c.st); dev_free(tmp); }
    return rc;
}

extern "C" {

int ising_sweep(ising_handle h, double beta, int n_sweeps, int tile, int k_inner) {
    return sweep_impl(h, beta, n_sweeps, tile, k_inner, nullptr, nullptr);
}

int ising_sweep_series(ising_handle h, double beta, int n_sweeps, int tile, int k_inner, int64_t* E, int64_t* M) {
    return sweep_impl(h, beta, n_sweeps, tile, k_inner, E, M);
}

int ising_observables(ising_handle h, int64_t* E, int64_t* M) {
    if (!h) { set_error("ising_observables: NULL handle"); return ISING_EINVAL; }
    int rc = observables_now(h, h->d_obs, h->d_obs + h->R);
    if (rc) return rc;
    if (E) { rc = copy_out(E, h->d_obs, sizeof(long long) * h->R, nullptr); if (rc) return rc; }
    if (M) { rc = copy_out(M, h->d_obs + h->R, sizeof(long long) * h->R, nullptr); if (rc) return rc; }
    ISING_CUDA_OK(cudaStreamSynchronize(hooks().stream));
    return 0;
}

int ising_overlap(ising_handle h, int a, int b, int64_t* Q) {
    if (!h || !Q || a < 0 || b < 0 || a >= h->R || b >= h->R) {
        set_error("ising_overlap: bad handle, NULL output or replica index out of range");
        return ISING_EINVAL;
    }
    int rc = 0;
    const int8_t* s = canon_view(h, &rc);
    if (rc) return rc;
    long long* d_Q = h->d_obs + 2 * h->R;
    rc = launch_overlap_canon(h, s, a, b, d_Q);
    if (rc) return rc;
    return copy_out(Q, d_Q, sizeof(long long), nullptr);
}

int ising_overlap_all(ising_handle h, int64_t* Q) {
    if (!h || !Q) { set_error("ising_overlap_all: NULL argument"); return ISING_EINVAL; }
    const size_t RR = (size_t)h->R * h->R;
    if (!h->d_pair) {
        h->d_pair = (long long*)dev_alloc(2 * RR * sizeof(long long));
        if (!h->d_pair) return ISING_ENOMEM;
    }
    unsigned long long* d_D = (unsigned long long*)h->d_pair;
    long long* d_Q = h->d_pair + RR;
    int rc;
    const uint64_t tiles_per_rep = h->store_tile ? (h->dim == 2 ? (uint64_t)(h->L / h->store_tile) * (h->L / h->store_tile)
                                                                 : (uint64_t)(h->L / 8) * (h->L / 8) * (h->L / 8)) : 0;
    switch (h->store) {                      // directly on the tile records where their spin bodies are contiguous
        case Store::PlaneI8: case Store::PlaneBits: {
            const uint32_t body = (uint32_t)(h->store == Store::PlaneBits ? h->store_tile * h->store_tile / 8 : h->store_tile * h->store_tile);
            rc = launch_overlap_all(h, h->d_tiles, tiles_per_rep * (body + 64), tiles_per_rep, body + 64, body, 1, d_D, d_Q);
            break;
        }
        case Store::Plane3I8: case Store::Plane3Bits: {
            const bool bits = h->store == Store::Plane3Bits;
            const uint32_t rec = (uint32_t)(tile3d_bytes(h, bits) / ((size_t)h->R * tiles_per_rep));
            rc = launch_overlap_all(h, h->d_tiles, tiles_per_rep * rec, tiles_per_rep, rec, bits ? 64u : 512u, 1, d_D, d_Q);
            break;
        }
        default: {                           // canonical +-1 bytes (0x01 ^ 0xff has 7 bits set); N is a multiple of 4 (L even)
            const int8_t* s = canon_view(h, &rc);
            if (!rc) rc = launch_overlap_all(h, s, h->N, 1, h->N, h->N, 7, d_D, d_Q);
            break;
        }
    }
    if (rc) return rc;
    return copy_out(Q, d_Q, RR * sizeof(long long), nullptr);
}

int ising_copy_spins(ising_handle h, int8_t* dst) {
    if (!h || !dst) { set_error("ising_copy_spins: NULL argument"); return ISING_EINVAL; }
    int rc = 0;
    const int8_t* s = canon_view(h, &rc);
    if (rc) return rc;
    return copy_out(dst, s, (size_t)h->R * h->N, nullptr);
}

int ising_set_spins(ising_handle h, const int8_t* src) {
    if (!h || !src) { set_error("ising_set_spins: NULL argument"); return ISING_EINVAL; }
    cudaStream_t st = hooks().stream;
    const size_t bytes = (size_t)h->R * h->N;
    // While the state lives in tile records, d_canon is scratch: land there, check, and only then switch over.
    // Otherwise d_canon is the state and must survive a rejected input: land in a staging buffer.
    const bool scratch = h->store != Store::Canon;
    int8_t* land = scratch ? h->d_canon : (int8_t*)dev_alloc(bytes);
    if (!land) return ISING_ENOMEM;
    if (scratch) h->canon_version = 0;            // the scratch copy is being overwritten
    const bool dev = is_device_ptr(src);
    cudaError_t e = cudaMemcpyAsync(land, src, bytes, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st);
    int bad = 0;
    int rc = (e == cudaSuccess) ? launch_validate_pm1(land, bytes, h->d_flag, &bad) : ISING_ECUDA;
    if (e != cudaSuccess) set_error("ising_set_spins: copy failed: %s", cudaGetErrorString(e));
    if (!rc && bad) { set_error("ising_set_spins: spins must be +1 or -1"); rc = ISING_EINVAL; }
    if (!rc && !scratch) {
        e = cudaMemcpyAsync(h->d_canon, land, bytes, cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) { set_error("ising_set_spins: %s", cudaGetErrorString(e)); rc = ISING_ECUDA; }
    }
    if (!rc) { h->store = Store::Canon; h->store_tile = 0; ++h->state_version; }
    cudaStreamSynchronize(st);
    if (!scratch) dev_free(land);
    return rc;
}

int ising_copy_spins_bits(ising_handle h, uint32_t* dst) {
    if (!h || !dst) { set_error("ising_copy_spins_bits: NULL argument"); return ISING_EINVAL; }
    if (h->N % 32) { set_error("ising_copy_spins_bits: N = %llu is not a multiple of 32", (unsigned long long)h->N); return ISING_EUNSUPPORTED; }
    int rc = 0;
    const int8_t* s = canon_view(h, &rc);
    if (rc) return rc;
    const uint64_t nwords = (uint64_t)h->R * h->N / 32;
    uint32_t* stage = (uint32_t*)dev_alloc(nwords * 4);
    if (!stage) return ISING_ENOMEM;
    rc = launch_pack_bits(s, stage, nwords);
    if (!rc) rc = copy_out(dst, stage, nwords * 4, nullptr);
    cudaStreamSynchronize(hooks().stream);
    dev_free(stage);
    return rc;
}

int ising_set_spins_bits(ising_handle h, const uint32_t* src) {
    if (!h || !src) { set_error("ising_set_spins_bits: NULL argument"); return ISING_EINVAL; }
    if (h->N % 32) { set_error("ising_set_spins_bits: N = %llu is not a multiple of 32", (unsigned long long)h->N); return ISING_EUNSUPPORTED; }
    cudaStream_t st = hooks().stream;
    const uint64_t nwords = (uint64_t)h->R * h->N / 32;
    uint32_t* stage = (uint32_t*)dev_alloc(nwords * 4);
    if (!stage) return ISING_ENOMEM;
    int rc = 0;
    cudaError_t e = cudaMemcpyAsync(stage, src, nwords * 4, is_device_ptr(src) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { set_error("ising_set_spins_bits: copy failed: %s", cudaGetErrorString(e)); rc = ISING_ECUDA; }
    h->canon_version = 0;
    if (!rc) rc = launch_unpack_bits(stage, h->d_canon, nwords);      // every bit pattern is a valid state
    if (!rc) { h->store = Store::Canon; h->store_tile = 0; ++h->state_version; }
    cudaStreamSynchronize(st);
    dev_free(stage);
    return rc;
}

int ising_set_layout(ising_handle h, int layout) {
    if (!h || (layout != ISING_LAYOUT_I8 && layout != ISING_LAYOUT_BITS)) {
        set_error("ising_set_layout: layout must be ISING_LAYOUT_I8 or ISING_LAYOUT_BITS");
        return ISING_EINVAL;
    }
    if (layout == h->layout) return 0;
    const int rc = ensure_canon(h);
    if (rc) return rc;
    h->layout = layout;
    return 0;
}

int ising_set_rng(ising_handle h, int mode) {
    if (!h || (mode != ISING_RNG_WORDS && mode != ISING_RNG_PLANES)) {
        set_error("ising_set_rng: mode must be ISING_RNG_WORDS or ISING_RNG_PLANES");
        return ISING_EINVAL;
    }
    h->rng = mode;
    return 0;
}

int ising_set_jit(ising_handle h, int mode) {
    if (!h || (mode != ISING_JIT_AUTO && mode != ISING_JIT_OFF && mode != ISING_JIT_ON)) {
        set_error("ising_set_jit: mode must be ISING_JIT_AUTO, ISING_JIT_OFF or ISING_JIT_ON");
        return ISING_EINVAL;
    }
    h->jit_mode = mode;
    return 0;
}

int ising_last_sweep_specialized(ising_handle h) { return h ? h->last_jit : 0; }

int ising_get_counter(ising_handle h, uint64_t* t) {
    if (!h || !t) { set_error("ising_get_counter: NULL argument"); return ISING_EINVAL; }
    *t = h->t;
    return 0;
}

int ising_set_counter(ising_handle h, uint64_t t) {
    if (!h) { set_error("ising_set_counter: NULL handle"); return ISING_EINVAL; }
    h->t = t;
    return 0;
}

int ising_synchronize(ising_handle h) {
    (void)h;
    ISING_CUDA_OK(cudaStreamSynchronize(hooks().stream));
    return 0;
}

const char* ising_sweep_path(ising_handle h) { return h ? h->last_path : "none"; }

int ising_force_path(ising_handle h, int generic_only) {
    if (!h) { set_error("ising_force_path: NULL handle"); return ISING_EINVAL; }
    h->force_generic = generic_only == 1 ? 1 : 0;
    h->no_resident = generic_only == 2 ? 1 : 0;
    h->no_flow = generic_only == 3 ? 1 : 0;
    h->no_onchip = generic_only == 4 ? 1 : 0;
    return 0;
}

}  // extern "C"
