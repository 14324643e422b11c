// planes_jit.cu — run-time specialisation of the 2D multi-spin tile kernel on the head bits of the
// acceptance thresholds.
//
// Every site is compared with one threshold only (thr[1] if exactly one bond is unsatisfied, thr[2] if none).
// If the 12 head bits of thr[1] and thr[2] are compile-time constants, that per-site choice folds into the
// LOP3 immediates of the bit-serial compare: 2 LOP3 per plane instead of 4 (−12 % of the instructions of a
// block update; +10 % flips/ns at k = 1, +17 % at k = 16).  The thresholds depend on beta, so the kernel
// k_tile_planes<T, BITS, HASJ, HP> of tile_planes_device.cuh — the same hand-written source the library is built
// from — is compiled for sm_100a by NVRTC the first time a (T, BITS, HASJ, HP) combination is needed and cached
// for the life of the process.  libnvrtc is loaded with dlopen: when it is missing, or anything fails, the
// caller falls back to the pre-compiled kernel with run-time threshold operands (same results, slower).
#include <dlfcn.h>
#include <stdlib.h>

#include <map>
#include <mutex>
#include <string>
#include <tuple>
#include <vector>

#include "kernels.h"

namespace ising {

namespace {

// The device sources, concatenated by build.py: philox.cuh + planes_common.cuh + tile_planes_device.cuh (2D) and
// philox.cuh + planes_common.cuh + tile3d_planes_device.cuh (3D).
const char* const kJitSource =
#include "jit_source.inc"
    ;
const char* const kJitSource3d =
#include "jit_source3d.inc"
    ;

typedef int nvrtcResult_t;
typedef struct _nvrtcProgram* nvrtcProgram_t;

struct Nvrtc {
    void* lib = nullptr;
    nvrtcResult_t (*CreateProgram)(nvrtcProgram_t*, const char*, const char*, int, const char* const*, const char* const*) = nullptr;
    nvrtcResult_t (*DestroyProgram)(nvrtcProgram_t*) = nullptr;
    nvrtcResult_t (*AddNameExpression)(nvrtcProgram_t, const char*) = nullptr;
    nvrtcResult_t (*CompileProgram)(nvrtcProgram_t, int, const char* const*) = nullptr;
    nvrtcResult_t (*GetLoweredName)(nvrtcProgram_t, const char*, const char**) = nullptr;
    nvrtcResult_t (*GetCUBINSize)(nvrtcProgram_t, size_t*) = nullptr;
    nvrtcResult_t (*GetCUBIN)(nvrtcProgram_t, char*) = nullptr;
    nvrtcResult_t (*GetProgramLogSize)(nvrtcProgram_t, size_t*) = nullptr;
    nvrtcResult_t (*GetProgramLog)(nvrtcProgram_t, char*) = nullptr;
    bool ok = false;

    Nvrtc() {
        if (getenv("ISING_NO_NVRTC")) return;          // testing aid: behave as if libnvrtc were not installed
        const char* names[] = {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so"};
        for (const char* n : names) {
            lib = dlopen(n, RTLD_NOW | RTLD_LOCAL);
            if (lib) break;
        }
        if (!lib) return;
#define ISING_SYM(f) f = reinterpret_cast<decltype(f)>(dlsym(lib, "nvrtc" #f)); if (!f) return
        ISING_SYM(CreateProgram); ISING_SYM(DestroyProgram); ISING_SYM(AddNameExpression); ISING_SYM(CompileProgram);
        ISING_SYM(GetLoweredName); ISING_SYM(GetCUBINSize); ISING_SYM(GetCUBIN); ISING_SYM(GetProgramLogSize); ISING_SYM(GetProgramLog);
#undef ISING_SYM
        ok = true;
    }
};

// The cache is bounded (a temperature scan or a parallel-tempering run meets a new pair of threshold heads at every beta):
// beyond 64 entries (ISING_JIT_CACHE overrides, for tests) the least recently used kernel is dropped and its cubin unloaded (after a synchronisation of
// the library's stream, so that no launch of it is still in flight).  Failed compilations are remembered as nullptr entries
// and age out the same way.
constexpr size_t kJitCacheMaxDefault = 64;
static size_t jit_cache_max() {
    static const size_t v = getenv("ISING_JIT_CACHE") ? (size_t)atoi(getenv("ISING_JIT_CACHE")) : kJitCacheMaxDefault;   // testing aid
    return v < 1 ? 1 : v;
}

struct JitEntry {
    cudaKernel_t kernel = nullptr;               // nullptr = tried and failed
    cudaLibrary_t lib = nullptr;
    uint64_t last_use = 0;
};

struct JitState {
    std::mutex mu;
    std::map<std::string, JitEntry> cache;       // name expression + macros -> kernel
    std::string last_log;
    uint64_t compiled = 0, clock = 0, evicted = 0;
};

JitState& state() {
    static JitState s;
    return s;
}

cudaKernel_t compile_one(const char* source, const std::string& expr, const std::vector<std::string>& defs, std::string& log,
                         cudaLibrary_t* lib_out) {
    static Nvrtc rt;
    if (!rt.ok) { log = "libnvrtc not available"; return nullptr; }
    nvrtcProgram_t prog = nullptr;
    if (rt.CreateProgram(&prog, source, "ising_jit.cu", 0, nullptr, nullptr) != 0) { log = "nvrtcCreateProgram failed"; return nullptr; }
    cudaKernel_t kernel = nullptr;
    do {
        if (rt.AddNameExpression(prog, expr.c_str()) != 0) { log = "nvrtcAddNameExpression failed"; break; }
        std::vector<const char*> opts = {"--gpu-architecture=sm_100a", "--std=c++17", "--generate-line-info"};
        for (const std::string& d : defs) opts.push_back(d.c_str());
        const nvrtcResult_t rc = rt.CompileProgram(prog, (int)opts.size(), opts.data());
        size_t n = 0;
        if (rt.GetProgramLogSize(prog, &n) == 0 && n > 1) { log.resize(n); rt.GetProgramLog(prog, &log[0]); }
        if (rc != 0) break;
        const char* lowered = nullptr;
        if (rt.GetLoweredName(prog, expr.c_str(), &lowered) != 0 || !lowered) { log += " nvrtcGetLoweredName failed"; break; }
        size_t sz = 0;
        if (rt.GetCUBINSize(prog, &sz) != 0 || sz == 0) { log += " no cubin"; break; }
        std::vector<char> cubin(sz);
        if (rt.GetCUBIN(prog, cubin.data()) != 0) { log += " nvrtcGetCUBIN failed"; break; }
        cudaLibrary_t lib = nullptr;
        if (cudaLibraryLoadData(&lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0) != cudaSuccess) {
            log += std::string(" cudaLibraryLoadData: ") + cudaGetErrorString(cudaGetLastError());
            break;
        }
        if (cudaLibraryGetKernel(&kernel, lib, lowered) != cudaSuccess) {
            log += std::string(" cudaLibraryGetKernel: ") + cudaGetErrorString(cudaGetLastError());
            kernel = nullptr;
            cudaLibraryUnload(lib);
            break;
        }
        *lib_out = lib;
    } while (false);
    rt.DestroyProgram(&prog);
    return kernel;
}

cudaKernel_t cached(const char* source, const std::string& expr, const std::vector<std::string>& defs) {
    try {                                        // std::string / std::map may throw: nothing may cross the C ABI
        JitState& s = state();
        std::lock_guard<std::mutex> lock(s.mu);
        std::string key = expr;
        for (const std::string& d : defs) key += " " + d;
        auto it = s.cache.find(key);
        if (it != s.cache.end()) {
            it->second.last_use = ++s.clock;
            return it->second.kernel;
        }
        if (s.cache.size() >= jit_cache_max()) {
            auto lru = s.cache.begin();
            for (auto jt = s.cache.begin(); jt != s.cache.end(); ++jt)
                if (jt->second.last_use < lru->second.last_use) lru = jt;
            if (lru->second.lib) {
                cudaStreamSynchronize(hooks().stream);
                cudaLibraryUnload(lru->second.lib);
            }
            s.cache.erase(lru);
            ++s.evicted;
        }
        std::string log;
        JitEntry e;
        e.kernel = compile_one(source, expr, defs, log, &e.lib);
        e.last_use = ++s.clock;
        if (e.kernel) ++s.compiled; else s.last_log = log;
        s.cache[key] = e;
        return e.kernel;
    } catch (...) {
        return nullptr;                          // the caller falls back to the pre-compiled kernel
    }
}

}  // namespace

// The 2D kernel specialised for (T, BITS, HASJ, HP) and the geometry (B tiles per side, R replicas), compiled on
// first use; nullptr if it cannot be had.
cudaKernel_t planes_jit_kernel(int T, bool bits, bool hasj, uint32_t hp, int B, int R, int NS) {
    char expr[160];
    snprintf(expr, sizeof expr, "ising::jit::k_tile_planes<%d, %s, %s, %uu, %d>", T, bits ? "true" : "false", hasj ? "true" : "false", hp, NS);
    return cached(kJitSource, expr, {"-DISING_JIT_B=" + std::to_string(B) + "u", "-DISING_JIT_R=" + std::to_string(R) + "u"});
}

cudaKernel_t flow_jit_kernel(int T, bool bits, bool hasj, uint32_t hp, int B, int R, int NS, bool staged) {
    char expr[160];
    snprintf(expr, sizeof expr, "ising::jit::k_flow_planes%s<%d, %s, %s, %uu, %d>", staged ? "_staged" : "", T, bits ? "true" : "false",
             hasj ? "true" : "false", hp, NS);
    return cached(kJitSource, expr, {"-DISING_JIT_B=" + std::to_string(B) + "u", "-DISING_JIT_R=" + std::to_string(R) + "u"});
}

// The grid-resident 2D kernel (grid_planes_device.cuh) specialised for (T, BITS, HASJ, HP), the geometry, the CTA shape and
// whether the jobs' constants are parked in shared memory.
cudaKernel_t grid_jit_kernel(int T, bool bits, bool hasj, uint32_t hp, int B, int R, int threads, int blocks, bool park, bool series, int strip) {
    char expr[160];
    snprintf(expr, sizeof expr, "ising::jit::k_grid_planes<%d, %s, %s, %uu>", T, bits ? "true" : "false", hasj ? "true" : "false", hp);
    return cached(kJitSource, expr, {"-DISING_JIT_B=" + std::to_string(B) + "u", "-DISING_JIT_R=" + std::to_string(R) + "u",
                                     "-DISING_G2_THREADS=" + std::to_string(threads), "-DISING_G2_BLOCKS=" + std::to_string(blocks),
                                     park ? "-DISING_G2_PARK=1" : "-DISING_G2_PARK=0", series ? "-DISING_G2_SERIES=1" : "-DISING_G2_SERIES=0", "-DISING_G2_STRIP=" + std::to_string(strip)});
}

// The 3D kernel specialised for (BITS, HP3 = the three threshold heads).
cudaKernel_t planes3d_jit_kernel(bool bits, unsigned long long hp3, int R) {
    char expr[160];
    snprintf(expr, sizeof expr, "ising::jit::k_tile3d_planes<%s, %lluull>", bits ? "true" : "false", hp3);
    return cached(kJitSource3d, expr, {R == 1 ? "-DISING_JIT_R=1" : "-DISING_JIT_R=0"});
}

cudaKernel_t grid3d_jit_kernel(bool bits, unsigned long long hp3, int R, int threads, int blocks, bool series) {
    char expr[160];
    snprintf(expr, sizeof expr, "ising::jit::k_grid3d<%s, false, %lluull>", bits ? "true" : "false", hp3);
    return cached(kJitSource3d, expr, {R == 1 ? "-DISING_JIT_R=1" : "-DISING_JIT_R=0", "-DISING_G3_THREADS=" + std::to_string(threads),
                                       "-DISING_G3_BLOCKS=" + std::to_string(blocks), series ? "-DISING_G3_SERIES=1" : "-DISING_G3_SERIES=0"});
}

uint64_t planes_jit_compiled() { return state().compiled; }
const char* planes_jit_last_log() { return state().last_log.c_str(); }

}  // namespace ising
