// kernels.h — host-side launch functions implemented by the .cu files; called by api.cu.
#pragma once
#include "common.cuh"

namespace ising {

// ---- generic.cu: canonical int8 ±1 storage, any even L, any valid tile ---------------
int launch_hot_start(ising_ctx* h);                                   // S8c.3 (a11)
int launch_generic_sweep(ising_ctx* h, const Accept& acc, int n, int T, int k,
                         long long* d_E, long long* d_M);             // a1,a4-a6,a8,a9
int launch_observables_canon(ising_ctx* h, const int8_t* d_spins, long long* d_E,
                             long long* d_M);                         // a10 (R values each)
int launch_overlap_canon(ising_ctx* h, const int8_t* d_spins, int a, int b, long long* d_Q);
int launch_overlap_all(ising_ctx* h, const void* base, uint64_t rep_stride_bytes, uint64_t n_chunks, uint64_t chunk_stride_bytes,
                       uint64_t chunk_bytes, int bits_per_diff, unsigned long long* d_D, long long* d_Q);   // all R*R overlaps, any spin store
int launch_validate_pm1(const int8_t* d, uint64_t n, int* d_flag, int* host_bad);
int launch_pack_bits(const int8_t* d_canon, uint32_t* d_words, uint64_t nwords);     // +-1 bytes -> one bit per site
int launch_unpack_bits(const uint32_t* d_words, int8_t* d_canon, uint64_t nwords);

// ---- tile_i8.cu: 2D tile records of 0/1 bytes, warp-per-tile staged kernel -----------
bool tile_i8_supported(const ising_ctx* h, int T);
size_t tile_i8_bytes(const ising_ctx* h, int T);
int launch_canon_to_tile_i8(ising_ctx* h, int T, const int8_t* d_canon, void* d_tiles);
int launch_tile_i8_to_canon(ising_ctx* h, int T, const void* d_tiles, int8_t* d_canon);
int launch_tile_i8_pass(ising_ctx* h, const Accept& acc, int T, int k, uint64_t t_first);

// ---- tile_planes.cu: 2D multi-spin tile kernel (RNG mapping "planes"), int8 or bit records ----
bool tile_planes_supported(const ising_ctx* h, int T);
size_t tile_planes_bytes(const ising_ctx* h, int T, bool bits);
int launch_canon_to_planes(ising_ctx* h, int T, bool bits, const int8_t* d_canon, void* d_tiles);
int launch_planes_to_canon(ising_ctx* h, int T, bool bits, const void* d_tiles, int8_t* d_canon);
size_t coupling_record_bytes(const ising_ctx* h);
int launch_convert_couplings(ising_ctx* h, int T, void* d_jrec);
bool plain64_supported(const ising_ctx* h, int T);
int launch_plain64(ising_ctx* h, const Accept& acc, bool bits, int n, int k, uint64_t t_first, long long* d_E, long long* d_M);
int launch_observables_planes(ising_ctx* h, int T, bool bits, long long* d_E, long long* d_M);
int launch_tile_planes_pass(ising_ctx* h, const Accept& acc, int T, bool bits, int k, uint64_t t_first, bool use_jit);
int launch_tile_planes_plain(ising_ctx* h, const Accept& acc, int T, bool bits, int n, int k, uint64_t t_first, int Tc);   // a8, large L; Tc: coarse tiles 2..16 or 0
bool resident_planes_supported(const ising_ctx* h, int T);      // small lattices: the whole call in one cluster launch
int launch_resident_planes(ising_ctx* h, const Accept& acc, int T, bool bits, int n, int k, uint64_t t_first,
                           long long* d_E, long long* d_M, bool plain, int Tc);   // d_E / d_M: optional series, n * R values each;
                                                                           // plain: the tile == L schedule, T = register tiling only

bool grid_planes_supported(const ising_ctx* h, int T);          // 512 < L <= ~4096: the whole call in one launch, every tile in registers on all SMs
size_t grid_planes_xedge_bytes(const ising_ctx* h, int T);
size_t grid_plain_xedge_bytes(const ising_ctx* h, int T);      // k_grid_plain: two exchange records per tile
// a8 / coarse tiles on chip on all SMs (k_grid_plain): 0 = done, 1 = does not fit or refused (nothing launched)
int launch_grid_plain(ising_ctx* h, const Accept& acc, int T, bool bits, int n, int k, uint64_t t_first, int Tc, void* d_xedge);
size_t grid_planes_acc_bytes(const ising_ctx* h, int n);
int launch_grid_planes(ising_ctx* h, const Accept& acc, int T, bool bits, int n, int k, uint64_t t_first, void* d_xedge, void* d_acc,
                       long long* d_E, long long* d_M, bool use_jit, bool allow_pc);   // returns 1 (nothing launched) if the lattice does not fit;
                                                                                       // allow_pc: the producer / consumer form where it applies

bool flow_planes_supported(const ising_ctx* h, int T, int n);   // HBM-resident lattices, n >= 2 passes: one persistent launch, colours ordered by data flow
size_t flow_planes_scratch_bytes(const ising_ctx* h, int T);
int launch_flow_planes(ising_ctx* h, const Accept& acc, int T, bool bits, int n, int k, uint64_t t_first, void* d_scratch, bool use_jit);

// ---- tile3d_planes.cu: 3D multi-spin tile kernel, 8x8x8 tiles (RNG mapping "planes") ----------
bool tile3d_supported(const ising_ctx* h, int T);
size_t tile3d_bytes(const ising_ctx* h, bool bits);
int launch_canon_to_3d(ising_ctx* h, bool bits, const int8_t* d_canon, void* d_tiles);
int launch_3d_to_canon(ising_ctx* h, bool bits, const void* d_tiles, int8_t* d_canon);
int launch_tile3d_pass(ising_ctx* h, const Accept& acc, bool bits, int k, uint64_t t_first, bool use_jit);
size_t coupling_record3d_bytes(const ising_ctx* h);
int launch_convert_couplings3d(ising_ctx* h, void* d_jrec);
bool resident3d_supported(const ising_ctx* h, int T);            // L <= 64: the whole call in one cluster launch
int launch_resident3d(ising_ctx* h, const Accept& acc, bool bits, int n, int k, uint64_t t_first, long long* d_E, long long* d_M,
                      bool plain, int Tc);                        // plain: the tile == L schedule; Tc: masked coarse tiles or 0
bool grid3d_supported(const ising_ctx* h, int T);               // L > 64: the whole call in one cooperative launch (k_grid3d)
size_t grid3d_xedge_bytes(const ising_ctx* h);
size_t grid3d_acc_bytes(const ising_ctx* h, int n);
int launch_grid3d(ising_ctx* h, const Accept& acc, bool bits, int n, int k, uint64_t t_first, void* d_xedge, void* d_acc,
                  long long* d_E, long long* d_M, bool use_jit);          // returns 1 (nothing launched) if the lattice does not fit
int launch_tile3d_plain(ising_ctx* h, const Accept& acc, bool bits, int n, int k, uint64_t t_first, int Tc);   // a8 in 3D, L > 64
int launch_observables3d(ising_ctx* h, bool bits, long long* d_E, long long* d_M);   // a10 on 3D tile records

// ---- amsc.cu: asynchronous multi-spin coding, 32 disorder realisations per word lattice, up to 256 per handle, 2D and 3D (R17) ----
bool amsc_supported(const ising_ctx* h, int T);
bool amsc3d_supported(const ising_ctx* h, int T);
size_t amsc_spin_bytes(const ising_ctx* h);
size_t amsc_bond_bytes(const ising_ctx* h);
int launch_amsc_pack_J(ising_ctx* h, void* d_jwords);
int launch_canon_to_amsc(ising_ctx* h, const int8_t* d_canon, void* d_words);
int launch_amsc_to_canon(ising_ctx* h, const void* d_words, int8_t* d_canon);
int launch_amsc_pass(ising_ctx* h, const Accept& acc, int T, int k, uint64_t t_first, const void* d_jwords);

// ---- planes_jit.cu: run-time specialisation of k_tile_planes on the threshold head bits (NVRTC) ----
cudaKernel_t planes_jit_kernel(int T, bool bits, bool hasj, uint32_t hp, int B, int R, int NS);   // NS: tiles per lane
cudaKernel_t planes3d_jit_kernel(bool bits, unsigned long long hp3, int R);   // nullptr: not available
cudaKernel_t grid3d_jit_kernel(bool bits, unsigned long long hp3, int R, int threads, int blocks, bool series);   // k_grid3d specialised on the three threshold heads and the CTA shape
cudaKernel_t flow_jit_kernel(int T, bool bits, bool hasj, uint32_t hp, int B, int R, int NS, bool staged);   // k_flow_planes, specialised like k_tile_planes
cudaKernel_t grid_jit_kernel(int T, bool bits, bool hasj, uint32_t hp, int B, int R, int threads, int blocks, bool park, bool series, int strip);   // k_grid_planes specialised on the threshold heads and the CTA shape
uint64_t planes_jit_compiled();
const char* planes_jit_last_log();

}  // namespace ising
