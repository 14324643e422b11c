// no_alloc.cu — ising_overlap_all_static (include/ising.h): all pairwise overlaps Q_ab = sum_i s_i^a s_i^b (S8c.7; BASELINE
// config 5: "pairwise overlap q") for callers that may not allocate device memory: code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc.  A variant of k_overlap_all (generic.cu): the same XOR + popcount
// pass and the same R x R table of difference counts, but the table does not come from the handle's allocation: it lives in a
// file-scope __device__ array of a fixed, modest size that every GPU which loads the library holds until the process exits.
//
// The entry point calls no cudaMalloc / cudaFree and no allocating library routine, takes no handle, and only enqueues work:
// inputs and outputs are the caller's device buffers.  Every call shares the one array (it keeps the last call's contents,
// so each call clears the part it uses first): calls that overlap on the GPU (two streams, two host threads) race.
#include <algorithm>
#include <mutex>

#include "common.cuh"

namespace ising {

namespace {

constexpr int kThreads = 256;
constexpr int kPairChunk = 8;
constexpr int kMaxR = ISING_STATIC_MAX_REPLICAS;

// 64 x 64 x 8 bytes = 32 KiB per GPU.  In host code this name is a host-side stand-in, not a device address: kernels are
// given the pointer cudaGetSymbolAddress returns (static_scratch below), never the name.
static __device__ __align__(256) unsigned long long g_pair_counts[kMaxR * kMaxR];

// D[a * R + b], b > a: popc summed over the words of replicas a and b (7 set bits per differing +-1 byte).  Block row a
// (blockIdx.y) compares replica a with the replicas b > a, eight at a time; spins: [R][N] bytes read as N / 4 words.
__global__ void __launch_bounds__(kThreads) k_overlap_all_static(const uint32_t* __restrict__ spins, uint64_t rep_words, int R,
                                                                 unsigned long long* __restrict__ D) {
    const int a = blockIdx.y;
    __shared__ unsigned long long sh[kThreads / 32][kPairChunk];
    for (int b0 = a + 1; b0 < R; b0 += kPairChunk) {
        unsigned long long acc[kPairChunk];
#pragma unroll
        for (int j = 0; j < kPairChunk; ++j) acc[j] = 0;
        for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < rep_words; i += (uint64_t)gridDim.x * blockDim.x) {
            const uint32_t wa = __ldg(spins + (uint64_t)a * rep_words + i);
#pragma unroll
            for (int j = 0; j < kPairChunk; ++j)
                if (b0 + j < R) acc[j] += (unsigned)__popc(wa ^ __ldg(spins + (uint64_t)(b0 + j) * rep_words + i));
        }
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
        for (int j = 0; j < kPairChunk; ++j) {
            unsigned long long v = acc[j];
            for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
            if (lane == 0) sh[w][j] = v;
        }
        __syncthreads();
        if (threadIdx.x < kPairChunk && b0 + (int)threadIdx.x < R) {
            unsigned long long v = 0;
            for (int ww = 0; ww < kThreads / 32; ++ww) v += sh[ww][threadIdx.x];
            atomicAdd(D + (size_t)a * R + (b0 + threadIdx.x), v);
        }
        __syncthreads();
    }
}

// Q_ab = N - 2 #differing sites; 0x01 ^ 0xff has 7 bits set
__global__ void k_overlap_finish_static(const unsigned long long* __restrict__ D, long long* __restrict__ Q, int R, long long nsites) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= R * R) return;
    const int a = i / R, b = i - a * R;
    if (a == b) { Q[i] = nsites; return; }
    const unsigned long long d = a < b ? D[(size_t)a * R + b] : D[(size_t)b * R + a];
    Q[i] = nsites - 2ll * (long long)(d / 7u);
}

// The device address of g_pair_counts on the CURRENT device, resolved once per device (with that device current).
int static_scratch(unsigned long long** out) {
    constexpr int kMaxDevices = 64;
    static std::mutex mu;
    static unsigned long long* addr[kMaxDevices] = {};
    int dev = 0;
    ISING_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) { set_error("ising_overlap_all_static: device ordinal %d out of range", dev); return ISING_EUNSUPPORTED; }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        unsigned long long* p = nullptr;
        ISING_CUDA_OK(cudaGetSymbolAddress((void**)&p, g_pair_counts));
        addr[dev] = p;
    }
    *out = addr[dev];
    return 0;
}

}  // namespace

}  // namespace ising

extern "C" int ising_overlap_all_static(const int8_t* d_spins, int n_replicas, uint64_t n_sites, int64_t* d_Q, void* cuda_stream) {
    using namespace ising;
    if (!d_spins || !d_Q) { set_error("ising_overlap_all_static: NULL pointer"); return ISING_EINVAL; }
    if (n_replicas < 1 || n_replicas > kMaxR) {
        set_error("ising_overlap_all_static: %d replicas, the static scratch holds at most ISING_STATIC_MAX_REPLICAS = %d "
                  "(use ising_overlap_all on a handle for more)", n_replicas, kMaxR);
        return ISING_EINVAL;
    }
    if (n_sites == 0 || (n_sites & 3u) || n_sites > (1ull << 40) || ((uintptr_t)d_spins & 3u) || ((uintptr_t)d_Q & 7u)) {
        set_error("ising_overlap_all_static: n_sites must be a positive multiple of 4 (at most 2^40), d_spins 4-byte and d_Q 8-byte aligned");
        return ISING_EINVAL;
    }
    unsigned long long* d_D = nullptr;
    if (int rc = static_scratch(&d_D)) return rc;
    cudaStream_t st = cuda_stream ? (cudaStream_t)cuda_stream : hooks().stream;
    const int R = n_replicas;
    const uint64_t rep_words = n_sites / 4;
    // the array keeps the last call's counts: clear the R x R words this call accumulates into
    ISING_CUDA_OK(cudaMemsetAsync(d_D, 0, sizeof(unsigned long long) * (size_t)R * R, st));
    if (R > 1) {
        unsigned gx = (unsigned)std::min<uint64_t>((rep_words + kThreads - 1) / kThreads, 148u * 8u);
        k_overlap_all_static<<<dim3(gx, (unsigned)(R - 1)), kThreads, 0, st>>>((const uint32_t*)d_spins, rep_words, R, d_D);
        count_launch();
    }
    k_overlap_finish_static<<<(R * R + 255) / 256, 256, 0, st>>>(d_D, (long long*)d_Q, R, (long long)n_sites);
    count_launch();
    ISING_CUDA_OK(cudaGetLastError());
    return 0;
}
