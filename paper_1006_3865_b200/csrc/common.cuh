// common.cuh — handle, error plumbing and launch helpers shared by the .cu files of
// libising_b200.  Product code: nothing here (or anywhere under csrc/) includes oracle/.
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "../../include/ising.h"

namespace ising {

// ---- process-wide hooks (ising_set_device_hooks) -------------------------------------
struct Hooks {
    void* (*alloc)(size_t) = nullptr;
    void (*dealloc)(void*) = nullptr;
    cudaStream_t stream = nullptr;
};
Hooks& hooks();
void set_error(const char* fmt, ...);
void count_launch(uint64_t n = 1);

void* dev_alloc(size_t bytes);   // through the hooks; nullptr on failure (error set)
void dev_free(void* p);

#define ISING_CUDA_OK(expr)                                                              \
    do {                                                                                 \
        cudaError_t e__ = (expr);                                                        \
        if (e__ != cudaSuccess) {                                                        \
            ::ising::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), \
                               __FILE__, __LINE__);                                      \
            return ISING_ECUDA;                                                          \
        }                                                                                \
    } while (0)

// Opt a kernel in to more than 48 KB of dynamic shared memory, once per (kernel, device): the attribute is per
// device, and one process may drive several.
template <auto Kernel>
int set_max_dynamic_smem(int bytes) {
    static std::atomic<uint64_t> done{0};        // one bit per device ordinal (mod 64)
    int dev = 0;
    ISING_CUDA_OK(cudaGetDevice(&dev));
    const uint64_t bit = 1ull << (dev & 63);
    if (done.load(std::memory_order_acquire) & bit) return 0;
    ISING_CUDA_OK(cudaFuncSetAttribute(Kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    done.fetch_or(bit, std::memory_order_release);
    return 0;
}

// How the spins are currently held in HBM.
enum class Store : int {
    Canon = 0,   // int8 ±1, index order, R*N bytes (generic kernels, observables, I/O)
    TileI8 = 1,  // tile records of 0/1 bytes, colour-split rows + edge columns (tile_i8.cu)
    PlaneI8 = 2, // piece-major tile records of 0/1 bytes (tile_planes.cu)
    PlaneBits = 3, // tile records of bit words (tile_planes.cu)
    Plane3I8 = 4,  // 3D 8^3 tile records, 0/1 bytes + bit-packed face copies (tile3d_planes.cu)
    Plane3Bits = 5, // 3D 8^3 tile records, bit words + face copies
    Amsc = 6       // one 32-bit word per site, bit r = realisation r (amsc.cu)
};

// Acceptance constants handed to every sweep kernel (S8c.4/5).
// The device test is   flip  <=>  n_sat + #{m : r >= thr[m]} <= 2*dim,
// which equals "a <= 0, or r < thr[a/2]" because thr[1] >= thr[2] >= thr[3]
// (n_sat = number of satisfied bonds, a = 2*n_sat - 2*dim).
// cneg[m-1] = 2^32 - thr[m] as a 32-bit addend whose carry-out is (r >= thr[m]);
// thresholds equal to 2^32 (beta = 0) never carry (cneg = 0) and thresholds equal to 0
// always count: those are folded into `always` instead (cneg = 0 as well).
struct Accept {
    uint32_t cneg[3];
    uint32_t always;   // number of m in 1..dim with thr[m] == 0
    uint32_t thr[3];   // thr[m] clipped to 32 bits (for kernels that compare directly)
    uint32_t thr_is_2p32[3];
};

}  // namespace ising

struct ising_ctx {
    int dim = 2;
    int L = 0;
    int R = 1;
    uint64_t N = 0;
    bool has_J = false;
    int8_t* d_J = nullptr;          // canonical ±1, dim*N bytes (nullptr if uniform)
    uint64_t* d_seeds = nullptr;    // R Philox keys (hot start; and sweeps unless shared_sweep)
    uint64_t* d_sweep_seeds = nullptr;   // keys of the sweep stream: d_seeds, or R copies of sweep_seed (R17)
    bool J_per_replica = false;     // d_J holds R coupling arrays (multi-realisation batch, R17)
    bool shared_sweep = false;
    uint64_t sweep_seed = 0;
    std::vector<uint64_t> seeds;
    uint64_t t = 0;                 // inner sweeps done (S8c.6)

    int rng = ISING_RNG_PLANES;     // RNG->site mapping (DESIGN.md §3 R6)
    int layout = ISING_LAYOUT_I8;   // requested HBM layout
    ising::Store store = ising::Store::Canon;
    int store_tile = 0;             // T of the tile records when store != Canon
    int8_t* d_canon = nullptr;      // R*N bytes; valid iff store == Canon (else scratch)
    void* d_tiles = nullptr;        // tile-record storage (TileI8 / PlaneI8 / PlaneBits)
    size_t tiles_bytes = 0;
    void* d_amsc_J = nullptr;       // JX, JY word lattices of a multi handle (2*N words), built on first use
    void* d_xedge = nullptr;        // k_grid_planes: boundary-word exchange records (128 B per tile)
    size_t xedge_bytes = 0;
    void* d_gacc = nullptr;         // k_grid_planes: per-pass accumulators of a series call
    size_t gacc_bytes = 0;
    void* d_Jtiles = nullptr;       // couplings in tile-record form for store_tile
    int Jtiles_tile = 0;
    int Jtiles_kind = -1;
    size_t Jtiles_bytes = 0;

    long long* d_obs = nullptr;     // 2*R int64 accumulators (+1 for overlap)
    long long* d_pair = nullptr;    // ising_overlap_all: R*R difference counts + R*R overlaps
    uint64_t state_version = 1;     // bumped by everything that changes the spins
    bool sweeping = false;          // inside ising_sweep / ising_sweep_series
    uint64_t canon_version = 0;     // state_version d_canon was last converted from while the state lives in tile records (0: never)
    int* d_flag = nullptr;          // validation flag
    const char* last_path = "none";
    int force_generic = 0;
    int no_resident = 0;            // ising_force_path(h, 2): per-pass launches even where the cluster-resident kernel applies
    int no_flow = 0;                // ising_force_path(h, 3): a launch per colour also where the persistent data-flow kernel applies
    int no_onchip = 0;              // ising_force_path(h, 4): never the cluster / grid resident kernels (the data-flow kernel may run)
    int jit_mode = 0;               // ISING_JIT_AUTO / OFF / ON (ising_set_jit)
    int last_jit = 0;               // 1 if the last tile launch used a run-time specialised kernel
};
