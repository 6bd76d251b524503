// noalloc.cu -- sph_scan_u32_noalloc: an exclusive prefix sum (the scan behind the neighbour-cache offsets of Alg. 5,
// PAPER.md:1124-1130, and the stream compaction of PAPER.md:1007-1009) that ALLOCATES NOTHING, for callers that cannot
// call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
//
// It is a variant of scan.cu's single-pass decoupled look-back kernel whose scratch memory -- one 64-bit status word
// per tile of 2048 items and the tile ticket counter -- lives in a file-scope `static __device__` array instead of
// buffers taken from the context's allocator. Consequences, all stated in include/sph_b200.h:
//   * a fixed maximum size: kNoAllocMaxItems = 2^24 items (8192 tiles; the array is 65 792 bytes, held by every GPU
//     that loads the library until the process exits); larger sizes are rejected with SPH_ERR_CAP;
//   * every call on a device shares that one array, which keeps the previous call's contents: the entry point clears
//     the words it uses (cudaMemsetAsync, stream-ordered) before the kernel; calls that OVERLAP on the GPU (different
//     streams without ordering between them) race on it;
//   * in host code the array's name is a host-side stand-in, not a device address: the address is taken once per
//     device, with that device current, by cudaGetSymbolAddress, and that pointer is what the kernel receives.
// No cudaMalloc, cudaFree or allocating library routine is called here; no existing code path is changed.
#include <stdarg.h>

#include <mutex>

#include "common.cuh"

namespace sph {

constexpr int kNaThreads = 256, kNaItems = 8, kNaTile = kNaThreads * kNaItems;      // 2048 items per tile
constexpr int64_t kNoAllocMaxItems = (int64_t)1 << 24;
constexpr int kNaMaxTiles = (int)(kNoAllocMaxItems / kNaTile);                       // 8192
constexpr uint64_t kNaFlagAgg = 1ull << 62, kNaFlagIncl = 2ull << 62, kNaValMask = (1ull << 62) - 1ull;

// scratch: words [0, kNaMaxTiles) = look-back status of each tile, word kNaMaxTiles = the tile ticket counter (+ pad)
static __device__ __align__(256) unsigned long long g_noalloc_scratch[kNaMaxTiles + 32];

// in: n u32 counts; out: n + 1 exclusive prefix sums as u64 (out[n] = total). Same scheme as scan.cu: k_scan.
__global__ void __launch_bounds__(kNaThreads) k_scan_noalloc(const uint32_t* __restrict__ in, uint64_t* __restrict__ out,
                                                             int64_t n, volatile unsigned long long* status,
                                                             unsigned int* counter) {
    __shared__ uint64_t wsum[kNaThreads / 32];
    __shared__ uint64_t s_excl;
    __shared__ uint32_t s_tile;
    const unsigned tid = threadIdx.x, lane = lane_id(), w = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(counter, 1u);       // dynamic tile id: predecessors are always already running
    __syncthreads();
    const uint32_t tile = s_tile;
    const int64_t base = (int64_t)tile * kNaTile + (int64_t)tid * kNaItems;

    uint32_t v[kNaItems];
    uint64_t tsum = 0;
#pragma unroll
    for (int i = 0; i < kNaItems; ++i) {
        v[i] = (base + i < n) ? in[base + i] : 0u;
        tsum += v[i];
    }
    uint64_t inc = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint64_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (unsigned)o) inc += t;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    uint64_t wbase = 0, agg = 0;
#pragma unroll
    for (unsigned j = 0; j < kNaThreads / 32; ++j) {
        if (j < w) wbase += wsum[j];
        agg += wsum[j];
    }
    if (w == 0) {
        // look-back by one warp, 32 predecessors per round trip; all lanes up to the nearest inclusive prefix must have
        // published before their values are summed
        volatile unsigned long long* my = status + tile;
        if (lane == 0) *my = (tile == 0 ? kNaFlagIncl : kNaFlagAgg) | agg;
        uint64_t excl = 0;
        if (tile > 0) {
            int64_t t = (int64_t)tile - 1;
            for (;;) {
                const int64_t idx = t - (int64_t)lane;
                uint64_t sv = kNaFlagIncl;                                   // before tile 0: inclusive prefix 0
                if (idx >= 0) sv = status[idx];
                const unsigned flag = (unsigned)(sv >> 62);
                const unsigned not_ready = __ballot_sync(0xffffffffu, flag == 0u);
                const unsigned incl = __ballot_sync(0xffffffffu, flag == 2u);
                const unsigned first = incl ? (unsigned)__ffs(incl) - 1u : 31u;
                const unsigned need = (first == 31u) ? 0xffffffffu : ((2u << first) - 1u);
                if (not_ready & need) continue;                              // poll again
                uint64_t val = (lane <= first) ? (sv & kNaValMask) : 0ull;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(0xffffffffu, val, o);
                excl += val;
                if (incl) break;
                t -= 32;
            }
            if (lane == 0) *my = kNaFlagIncl | (excl + agg);
        }
        if (lane == 0) s_excl = excl;
    }
    __syncthreads();
    uint64_t run = s_excl + wbase + inc - tsum;
#pragma unroll
    for (int i = 0; i < kNaItems; ++i) {
        if (base + i < n) out[base + i] = run;
        run += v[i];
    }
    if (base <= n - 1 && n - 1 < base + kNaItems) out[n] = run;              // the tile holding item n - 1 writes the total
}

// the scratch array's device address on each device, taken once per device with that device current
constexpr int kNaMaxDevices = 64;
static std::mutex g_na_mutex;
static unsigned long long* g_na_ptr[kNaMaxDevices] = {nullptr};
static thread_local char g_na_err[256] = {0};

static int na_fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_na_err, sizeof(g_na_err), fmt, ap);
    va_end(ap);
    return code;
}

}  // namespace sph

using namespace sph;

extern "C" {

int64_t sph_scan_noalloc_max_items(void) { return kNoAllocMaxItems; }

const char* sph_noalloc_last_error(void) { return g_na_err; }

int sph_scan_u32_noalloc(const uint32_t* in_dev, uint64_t* out_dev, int64_t n, void* cuda_stream) {
    g_na_err[0] = 0;
    if (!in_dev || !out_dev || n < 1)
        return na_fail(SPH_ERR_ARG, "sph_scan_u32_noalloc: null pointer or n < 1 (n = %lld)", (long long)n);
    if (n > kNoAllocMaxItems)
        return na_fail(SPH_ERR_CAP, "sph_scan_u32_noalloc: n = %lld exceeds the fixed maximum of %lld items (static scratch)",
                       (long long)n, (long long)kNoAllocMaxItems);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kNaMaxDevices) {
        cudaGetLastError();
        return na_fail(SPH_ERR_DEVICE, "sph_scan_u32_noalloc: no usable current CUDA device (device %d)", dev);
    }
    unsigned long long* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_na_mutex);
        if (!g_na_ptr[dev]) {
            // set-up, once per device, with that device current: the array's device address (in host code the name
            // g_noalloc_scratch is a stand-in, not an address a kernel can use)
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
            if (e != cudaSuccess || !p) {
                cudaGetLastError();
                return na_fail(SPH_ERR_DEVICE, "sph_scan_u32_noalloc: cudaGetSymbolAddress failed: %s (device %d)",
                               cudaGetErrorString(e), dev);
            }
            g_na_ptr[dev] = static_cast<unsigned long long*>(p);
        }
        scratch = g_na_ptr[dev];
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int64_t tiles = (n + kNaTile - 1) / kNaTile;
    // the array keeps the last call's contents: the status words of this call's tiles and the ticket counter start at zero
    e = cudaMemsetAsync(scratch, 0, (size_t)tiles * sizeof(unsigned long long), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(scratch + kNaMaxTiles, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return na_fail(SPH_ERR_DEVICE, "sph_scan_u32_noalloc: cudaMemsetAsync failed: %s", cudaGetErrorString(e));
    }
    k_scan_noalloc<<<(unsigned)tiles, kNaThreads, 0, st>>>(in_dev, out_dev, n, scratch,
                                                          reinterpret_cast<unsigned int*>(scratch + kNaMaxTiles));
    e = cudaGetLastError();
    if (e != cudaSuccess)
        return na_fail(SPH_ERR_DEVICE, "sph_scan_u32_noalloc: launch failed: %s", cudaGetErrorString(e));
    return SPH_OK;
}

}  // extern "C"
