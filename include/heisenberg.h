/* heisenberg.h — C ABI of the continuous-spin (classical Heisenberg, O(3)) double-checkerboard Metropolis
 * sweep in libising_b200.so: the generalisation the paper names in P:100 ("models with continuous spins such
 * as the Heisenberg model, where the large efficieny of GPU devices with (single-precision) floating-point
 * calculations comes into play"); SURVEY.md §8(f) item 4.  The paper gives no method for it, so every step is a
 * reading, H1-H8 of DESIGN.md §3.7: model H = -Σ_<ij> s_i·s_j on the periodic square / simple cubic lattice
 * (P:53-57), proposal = a fresh uniform direction, acceptance min[1, exp(-β ΔE)] (eq. (2)), schedule =
 * the double checkerboard of P:62-74 exactly as for the Ising model, arithmetic in
 * IEEE binary32 with every operation fixed (fused multiply-adds where stated, nothing re-associated), random
 * numbers from Philox4x32-10 keyed by the seed.  Results are bit-identical to oracle/heisenberg_oracle.cpp.
 *
 * Conventions shared with ising.h: plain pointers and sizes, no exceptions; 0 on success, negative ISING_E*
 * codes on failure with the message in ising_last_error(); device memory and the stream come from
 * ising_set_device_hooks(); kernels are counted by ising_kernel_launches(); there is no CPU path.
 */
#ifndef HEISENBERG_B200_H
#define HEISENBERG_B200_H

#include <stdint.h>

#include "ising.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct heis_ctx* heis_handle; /* opaque, owned by the library */

/* Hot start (H3): s_i = D(wa, wb) with (wa, wb) = words (2h, 2h+1), h = i & 1, of Philox(ctr = {i >> 1, 6, 0, 0},
 * key = seed), D the direction map H2.  dim in {2, 3}; L even, N = L^dim <= 2^32.  Spins live in HBM as three float
 * planes s[c][i], c = x, y, z, i = x + L*(y + L*z).  The shared-memory tile kernels serve L % 4 == 0 with tile in
 * {16, 32, 64} (2D) / {4, 8, 16} (3D) and L/tile even; every other valid combination runs on the generic kernels.
 * Returns NULL on failure. */
heis_handle heis_create(int dim, int L, uint64_t seed);
void heis_destroy(heis_handle h);

/* n_sweeps outer passes of the double checkerboard (H7): per pass the tiles of coarse colour 0, then
 * colour 1; per tile k_inner inner sweeps, each = fine colour 0 then fine colour 1; update H5
 * with the acceptance probability H6 and the random numbers H4 (one Philox call per 2x2 block of the xy plane and
 * half-sweep); beta is rounded to float once.  tile: edge T, even, T | L, L/T even or
 * T == L (0 means L: plain checkerboard).  One pass attempts k_inner*N updates; the handle's counter of inner
 * sweeps advances by n_sweeps*k_inner.  Asynchronous on the hooked stream. */
int heis_sweep(heis_handle h, double beta, int n_sweeps, int tile, int k_inner);

/* H8: E = -Σ_i Σ_d s_i·s_(i+e_d) and M[3] = Σ_i s_i, accumulated in double from the float spins (the order of
 * the sum is not fixed: equal to the oracle's up to double rounding).  E, M: caller-owned, host or device;
 * either may be NULL.  Synchronises. */
int heis_observables(heis_handle h, double* E, double* M);

/* heis_sweep with E and M after every outer pass: E[n_sweeps] and M[3 * n_sweeps] (pass-major: Mx, My, Mz of pass p
 * at M + 3p), caller-owned, host or device, either may be NULL.  Nothing is copied or synchronised between the passes
 * (the sums are accumulated on the device); synchronises at the end. */
int heis_sweep_series(heis_handle h, double beta, int n_sweeps, int tile, int k_inner, double* E, double* M);

/* dst / src: 3*N floats, component-major (x plane, y plane, z plane), host or device.  Synchronise.
 * heis_set_spins does not normalise or check the lengths. */
int heis_copy_spins(heis_handle h, float* dst);
int heis_set_spins(heis_handle h, const float* src);

/* The counter t of inner sweeps done (selects the random numbers of the next sweep, H4). */
int heis_get_counter(heis_handle h, uint64_t* t);
int heis_set_counter(heis_handle h, uint64_t t);

/* Which kernel family served the last heis_sweep: "heis_tile" (tile staged in shared memory for the k inner
 * sweeps), "heis_generic" (one launch per half-sweep on the live array) or "none".  heis_force_generic(h, 1)
 * routes every later sweep through the generic kernels (tests). */
const char* heis_sweep_path(heis_handle h);
int heis_force_generic(heis_handle h, int on);

#ifdef __cplusplus
}
#endif
#endif
