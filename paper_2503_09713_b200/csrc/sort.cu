// sort.cu -- a2: stable LSD radix sort of (key u64, val u32), onesweep style: one upfront histogram of all
// eight 8-bit digits, then ONE pass per digit that reads each (key,val) once and writes it once; tile prefixes
// are resolved with a decoupled look-back over single-word (flag|count) status entries; ranking inside a tile
// uses a warp-level ballot multisplit. Replaces the paper's bitonic sort, which it
// says dominates the tree build. HBM-bound: 8 B + 8 x 24 B = 200 B per particle.
#include <stdlib.h>

#include <utility>

#include "common.cuh"

namespace sph {

constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;
constexpr int kPasses = 8;
constexpr int kPrefixPass = 3;                   // prefix mode sorts on digits 3..7 = bits 24..63 (40 bits)
constexpr int kPrefixShift = kPrefixPass * 8;
constexpr int kSortThreads = 512;
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kItems = 10;                       // keys per thread
constexpr int kTile = kSortThreads * kItems;     // 5120 keys per tile, 2 CTAs = 32 warps per SM (8 keys per thread at 3 CTAs
                                                 // per SM: 0.99 instead of 0.93 ms at C2; 12 keys spill at 64 registers)
constexpr int kLookBatch = 4;
__device__ __forceinline__ uint32_t pad(uint32_t j) { return j + (j >> 5); }
constexpr uint32_t kFlagAgg = 1u << 30, kFlagIncl = 2u << 30, kValMask = (1u << 30) - 1u;

// ---- kernel 1: histograms of all 8 digits in one read of the keys ----
// A warp takes 32 consecutive keys at a time. The input is the previous step's order, i.e. nearly sorted: the upper
// digits of neighbouring keys are equal, so equal digits come in runs. Each run is added by its head lane alone
// (one shuffle and one ballot per digit); random digits simply give 32 heads. (One shared-memory atomic per key and
// digit serialises on the equal digits; MATCH.ANY per key and digit made this kernel MIO-bound at 8 % of the HBM
// rate.)
__global__ void __launch_bounds__(256) k_sort_hist(const uint64_t* __restrict__ key, int64_t N,
                                                   uint32_t* __restrict__ ghist, int p0) {
    __shared__ uint32_t sh[kPasses][kRadix];
    for (int i = threadIdx.x; i < kPasses * kRadix; i += blockDim.x) (&sh[0][0])[i] = 0;
    __syncthreads();
    const unsigned lane = lane_id();
    constexpr int kU = 4;                                      // keys in flight per thread
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t n_round = (N + 31) / 32 * 32;
    for (int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < n_round; i0 += kU * stride) {
        uint64_t kk[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const int64_t i = i0 + u * stride;
            kk[u] = (i < N) ? key[i] : 0ull;
        }
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const int64_t i = i0 + u * stride;                 // warp-uniform up to the lane offset
            if (i - lane >= N) break;
            const unsigned nvalid = (unsigned)min((int64_t)32, N - (i - lane));
            const bool valid = lane < nvalid;
#pragma unroll
            for (int p = 0; p < kPasses; ++p) {
                if (p < p0) continue;                            // digits below the first pass are not sorted on
                const unsigned d = (unsigned)(kk[u] >> (p * kRadixBits)) & (kRadix - 1);
                const unsigned dprev = __shfl_up_sync(0xffffffffu, d, 1);
                const bool head = valid && (lane == 0u || d != dprev);
                const unsigned heads = __ballot_sync(0xffffffffu, head);
                if (head) {
                    const unsigned rest = (lane == 31u) ? 0u : (heads >> (lane + 1u));
                    const unsigned next = rest ? lane + (unsigned)__ffs(rest) : nvalid;   // next head, or the end
                    atomicAdd(&sh[p][d], next - lane);
                }
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kPasses * kRadix; i += blockDim.x) {
        uint32_t v = (&sh[0][0])[i];
        if (v) atomicAdd(&ghist[i], v);
    }
}

// ---- kernel 2: exclusive scan of each digit histogram -> global digit bases ----
__global__ void __launch_bounds__(kRadix) k_sort_bases(uint32_t* __restrict__ ghist, DevScalars* sc) {
    if (threadIdx.x == 0) { sc->tie_max = 0u; sc->tie_max32 = 0u; sc->sort_redo = 0u; }
    __shared__ uint32_t wsum[kRadix / 32];
    const unsigned d = threadIdx.x, lane = lane_id(), w = d >> 5;
    for (int p = 0; p < kPasses; ++p) {
        uint32_t v = ghist[p * kRadix + d], inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= (unsigned)o) inc += t;
        }
        if (lane == 31) wsum[w] = inc;
        __syncthreads();
        uint32_t base = 0;
        for (unsigned j = 0; j < w; ++j) base += wsum[j];
        ghist[p * kRadix + d] = base + inc - v;
        __syncthreads();
    }
}

// ---- kernel 3: one onesweep pass ----
struct SortSmem {
    uint64_t keys[kTile + kTile / 32];       // indexed through pad(): slots a power of two apart (digits of a
    uint32_t vals[kTile + kTile / 32];       // regular lattice) would otherwise all fall into one bank
    uint32_t whist[kSortWarps][kRadix];
    uint32_t gofs[kRadix];
    uint32_t wsum[kRadix / 32];
    uint32_t tile;
};

__global__ void __launch_bounds__(kSortThreads, 2) k_onesweep(const uint64_t* __restrict__ kin,
                                                            const uint32_t* __restrict__ vin,
                                                            uint64_t* __restrict__ kout, uint32_t* __restrict__ vout,
                                                            int64_t N, int shift, const uint32_t* __restrict__ gbase,
                                                            volatile uint32_t* status, uint32_t* counter) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem& s = *reinterpret_cast<SortSmem*>(smem_raw);
    const unsigned tid = threadIdx.x, lane = lane_id(), w = tid >> 5;

    if (tid == 0) s.tile = atomicAdd(counter, 1u);   // dynamic tile id: predecessors are always already running
    for (int i = tid; i < kSortWarps * kRadix; i += kSortThreads) (&s.whist[0][0])[i] = 0;
    __syncthreads();
    const uint32_t tile = s.tile;
    const int64_t base = (int64_t)tile * kTile;
    const int tile_n = (int)min((int64_t)kTile, N - base);

    // load (warp-striped) and rank inside the warp with match_any multisplit
    uint64_t k[kItems];
    uint32_t rank[kItems];
    const int64_t wbase = base + (int64_t)w * (32 * kItems) + lane;
#pragma unroll
    for (int i = 0; i < kItems; ++i) {
        int64_t idx = wbase + i * 32;
        k[i] = (idx < N) ? kin[idx] : ~0ull;
    }
    const unsigned lt = lanemask_lt();
    // all match masks first, then the serial counter updates
    unsigned mm[kItems];
#pragma unroll
    for (int i = 0; i < kItems; ++i) {
        const bool valid = (wbase + i * 32) < N;
        const unsigned act = __ballot_sync(0xffffffffu, valid);
        const unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
        // lanes with the same digit: eight ballots, one per digit bit (MATCH.ANY was the kernel's largest stall)
        unsigned m = valid ? act : 0u;
#pragma unroll
        for (int b = 0; b < kRadixBits; ++b) {
            const bool bit = ((d >> b) & 1u) != 0u;
            const unsigned bal = __ballot_sync(0xffffffffu, bit);
            m &= bit ? bal : ~bal;
        }
        mm[i] = m;
    }
#pragma unroll
    for (int i = 0; i < kItems; ++i) {
        const bool valid = (wbase + i * 32) < N;
        const unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
        const unsigned m = mm[i];
        uint32_t prev = 0;
        if (valid) prev = s.whist[w][d];
        __syncwarp();
        if (valid && lane == (unsigned)(__ffs(m) - 1)) s.whist[w][d] = prev + __popc(m);
        __syncwarp();
        rank[i] = prev + __popc(m & lt);
    }
    __syncthreads();

    // per digit (thread d): exclusive scan over the warps, tile count, look-back, tile-local digit start
    const unsigned d = tid;
    uint32_t run = 0, inc = 0;
    volatile uint32_t* my = status + (size_t)tile * kRadix + d;
    if (tid < kRadix) {
#pragma unroll
        for (int ww = 0; ww < kSortWarps; ++ww) {
            uint32_t t = s.whist[ww][d];
            s.whist[ww][d] = run;
            run += t;
        }
        *my = (tile == 0 ? kFlagIncl : kFlagAgg) | run;
        // tile-local exclusive scan of the 256 digit counts
        inc = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= (unsigned)o) inc += t;
        }
        if (lane == 31) s.wsum[w] = inc;
    }
    __syncthreads();
    if (tid < kRadix) {
        uint32_t dstart = inc - run;
        for (unsigned j = 0; j < w; ++j) dstart += s.wsum[j];
        // decoupled look-back
        uint32_t excl = 0;
        if (tile > 0) {
            // four predecessors per round trip (independent loads), consumed in order up to the first one that has
            // not published yet or carries an inclusive prefix
            int64_t t = (int64_t)tile - 1;
            for (bool done = false; !done;) {
                uint32_t v[kLookBatch];
#pragma unroll
                for (int j = 0; j < kLookBatch; ++j) {
                    uint32_t vv = 2u << 30;           // before tile 0: inclusive prefix 0
                    if (t - j >= 0) vv = status[(size_t)(t - j) * kRadix + d];
                    v[j] = vv;
                }
#pragma unroll
                for (int j = 0; j < kLookBatch; ++j) {
                    const uint32_t flag = v[j] & ~kValMask;
                    if (flag == 0) break;             // not published yet: poll again from this tile
                    excl += v[j] & kValMask;
                    --t;
                    if (flag == kFlagIncl) { done = true; break; }
                }
            }
            *my = kFlagIncl | (excl + run);
        }
        s.gofs[d] = gbase[d] + excl - dstart;
#pragma unroll
        for (int ww = 0; ww < kSortWarps; ++ww) s.whist[ww][d] += dstart;
    }
    __syncthreads();

    // scatter into shared memory in tile-sorted order
#pragma unroll
    for (int i = 0; i < kItems; ++i) {
        int64_t idx = wbase + i * 32;
        if (idx < N) {
            unsigned d = (unsigned)(k[i] >> shift) & (kRadix - 1);
            uint32_t slot = s.whist[w][d] + rank[i];
            s.keys[pad(slot)] = k[i];
            s.vals[pad(slot)] = vin[idx];
        }
    }
    __syncthreads();

    // coalesced runs out to global memory
    for (int j = tid; j < tile_n; j += kSortThreads) {
        uint64_t kk = s.keys[pad((uint32_t)j)];
        unsigned d = (unsigned)(kk >> shift) & (kRadix - 1);
        uint32_t pos = s.gofs[d] + (uint32_t)j;
        kout[pos] = kk;
        vout[pos] = s.vals[pad((uint32_t)j)];
    }
}

// ---- kernel 4: tie repair / census for the prefix mode ----
// In prefix mode only the digits above bit `shift` are sorted on (stable LSD passes), which leaves keys that share
// those bits in their previous order. The thread at the head of each run of equal prefixes insertion-sorts the run
// by the full key (stable, so equal keys keep their previous order): the result is exactly the stable sort by the
// full key. Runs are rare and short when the prefix resolves the particles (40 of 63 bits: cells of 2^-13.3 of the
// box per axis); the longest run is recorded so that the host falls back to all eight passes when it is not.
// A run longer than max_run is not repaired (the insertion sort is quadratic and runs on one thread): the kernel
// raises sc->sort_redo instead, the tree kernels of this build then do nothing, and the host sorts again with all
// eight passes (api.cu). Prefix mode is only chosen after a sort whose longest run was <= 64, so this needs a sudden
// collapse of many particles into one 2^-13 cell between two steps.
// Two prefix lengths: 40 bits (shift 24, five passes) and 32 bits (shift 32, four passes: cells of 2^-10.7 of the box
// per axis, enough wherever the particle spacing is a few times that). The census is taken for both: at shift 24 the
// kernel also measures the runs of equal 32-bit prefixes (bounded walks; repairs inside 40-bit runs leave the top 40
// bits of every position unchanged, so this may read while other threads repair), at shift 32 its runs are those.
__global__ void __launch_bounds__(256) k_sort_repair(int64_t N, uint64_t* __restrict__ key, uint32_t* __restrict__ val,
                                                     int shift, int64_t max_run, DevScalars* sc) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    if (shift < 32) {
        const uint64_t p32 = key[i] >> 32;
        if (i == 0 || (key[i - 1] >> 32) != p32) {
            int64_t e = i + 1;
            while (e < N && e - i <= 65 && (key[e] >> 32) == p32) ++e;
            if (e - i >= 2) atomicMax(&sc->tie_max32, (unsigned int)(e - i));
        }
    }
    const uint64_t p = key[i] >> shift;
    if (i > 0 && (key[i - 1] >> shift) == p) return;          // not the head of a run
    int64_t e = i + 1;
    while (e < N && e - i <= max_run && (key[e] >> shift) == p) ++e;
    if (e - i < 2) return;
    atomicMax(shift < 32 ? &sc->tie_max : &sc->tie_max32, (unsigned int)min(e - i, (int64_t)0x7fffffff));
    if (e - i > max_run) { sc->sort_redo = 1u; return; }
    for (int64_t a = i + 1; a < e; ++a) {
        const uint64_t kk = key[a];
        const uint32_t vv = val[a];
        int64_t b = a - 1;
        while (b >= i && key[b] > kk) { key[b + 1] = key[b]; val[b + 1] = val[b]; --b; }
        key[b + 1] = kk;
        val[b + 1] = vv;
    }
}

int sort_scratch_bytes(int64_t N, int64_t* tiles, size_t* status_bytes) {
    *tiles = (N + kTile - 1) / kTile;
    *status_bytes = (size_t)kPasses * (size_t)(*tiles) * kRadix * sizeof(uint32_t);
    return SPH_OK;
}

constexpr int64_t kRepairMaxRun = 2048;          // longest run of equal prefixes the repair kernel sorts (4 M key moves at worst)

int launch_sort(sph_ctx* c) {
    // function attributes are per device: set on every launch (cheap) rather than once per process
    SPH_CUDA(c, cudaFuncSetAttribute(k_onesweep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem)));
    const int64_t N = c->N, tiles = c->sort_tiles;
    const size_t status_per_pass = (size_t)tiles * kRadix;
    SPH_CUDA(c, cudaMemsetAsync(c->sort_hist, 0, kPasses * kRadix * sizeof(uint32_t), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(c->sort_status, 0, kPasses * status_per_pass * sizeof(uint32_t), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(c->sort_counters, 0, kPasses * sizeof(uint32_t), c->stream));
    unsigned hb = (unsigned)min((int64_t)148 * 8, (N + 255) / 256);
    // Prefix mode: sort on the top 40 or 32 bits only (five or four passes) and repair the rare runs of equal prefixes;
    // chosen by the host from the longest runs seen in the previous sort (api.cu), all eight passes otherwise.
    // morton_bits = 10: the code sits in bits 62..33, four passes (bits 32..63) sort it completely, no repair
    const bool short_codes = c->p.morton_bits == 10;
    const int p0 = short_codes ? 4 : c->sort_p0;
    c->last_sort_passes = kPasses - p0;
    k_sort_hist<<<hb, 256, 0, c->stream>>>(c->key, N, c->sort_hist, p0);
    k_sort_bases<<<1, kRadix, 0, c->stream>>>(c->sort_hist, c->d_sc);
    c->launches += 2;
    uint64_t *kin = c->key, *kout = c->key_alt;
    uint32_t *vin = c->val, *vout = c->val_alt;
    for (int p = p0; p < kPasses; ++p) {
        k_onesweep<<<(unsigned)tiles, kSortThreads, sizeof(SortSmem), c->stream>>>(
            kin, vin, kout, vout, N, p * kRadixBits, c->sort_hist + p * kRadix,
            c->sort_status + p * status_per_pass, c->sort_counters + p);
        c->launches++;
        uint64_t* tk = kin; kin = kout; kout = tk;
        uint32_t* tv = vin; vin = vout; vout = tv;
    }
    if ((kPasses - p0) & 1) {   // odd number of passes: the result is in the other pair of buffers
        std::swap(c->key, c->key_alt);
        std::swap(c->val, c->val_alt);
    }
    if (!short_codes) {
        // in an eight-pass sort the kernel only takes the census of equal prefixes (every run is already in order);
        // SPH_REPAIR_MAX (tests) lowers the bound so that the redo path can be reached with small inputs
        const char* env = getenv("SPH_REPAIR_MAX");
        const int64_t max_run = (p0 == 0) ? (int64_t)1 << 40 : (env ? (int64_t)atoll(env) : kRepairMaxRun);
        k_sort_repair<<<div_up(N, 256), 256, 0, c->stream>>>(N, c->key, c->val, p0 == 4 ? 32 : kPrefixShift, max_run, c->d_sc);
        c->launches++;
    }
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
