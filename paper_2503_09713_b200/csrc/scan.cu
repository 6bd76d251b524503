// scan.cu -- single-pass exclusive prefix sum with decoupled look-back (the paper's scan of choice,
// PAPER.md:1007-1009; used for the neighbour-cache offsets of Alg. 5, and for leaf-group ids).
// in: n u32 counts; out: n+1 prefix sums (out[n] = total). HBM-bound: 4 B read + sizeof(OutT) written per item.
#include "common.cuh"

namespace sph {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanThreads * kScanItems;   // 2048
constexpr uint64_t kSFlagAgg = 1ull << 62, kSFlagIncl = 2ull << 62, kSValMask = (1ull << 62) - 1ull;

template <typename OutT>
__global__ void __launch_bounds__(kScanThreads) k_scan(const uint32_t* __restrict__ in, OutT* __restrict__ out, int64_t n,
                                                       volatile uint64_t* status, uint32_t* counter,
                                                       unsigned long long* total_out, uint32_t* fill, DevScalars* sc) {
    __shared__ uint64_t wsum[kScanThreads / 32];
    __shared__ uint64_t s_excl;
    __shared__ uint32_t s_tile;
    const unsigned tid = threadIdx.x, lane = lane_id(), w = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(counter, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const int64_t base = (int64_t)tile * kScanTile + (int64_t)tid * kScanItems;

    uint32_t v[kScanItems];
    uint64_t tsum = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        v[i] = (base + i < n) ? in[base + i] : 0u;
        tsum += v[i];
    }
    uint64_t inc = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint64_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (unsigned)o) inc += t;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    uint64_t wbase = 0, agg = 0;
#pragma unroll
    for (unsigned j = 0; j < kScanThreads / 32; ++j) {
        if (j < w) wbase += wsum[j];
        agg += wsum[j];
    }
    if (w == 0) {
        // look-back by one warp: 32 predecessors per round trip; the lanes up to the nearest inclusive prefix must all
        // have published before their values are summed
        volatile uint64_t* my = status + tile;
        if (lane == 0) *my = (tile == 0 ? kSFlagIncl : kSFlagAgg) | agg;
        uint64_t excl = 0;
        if (tile > 0) {
            int64_t t = (int64_t)tile - 1;
            for (;;) {
                const int64_t idx = t - (int64_t)lane;
                uint64_t sv = 2ull << 62;                                   // before tile 0: inclusive prefix 0
                if (idx >= 0) sv = status[idx];
                const unsigned flag = (unsigned)(sv >> 62);
                const unsigned not_ready = __ballot_sync(0xffffffffu, flag == 0u);
                const unsigned incl = __ballot_sync(0xffffffffu, flag == 2u);
                const unsigned first = incl ? (unsigned)__ffs(incl) - 1u : 31u;
                const unsigned need = (first == 31u) ? 0xffffffffu : ((2u << first) - 1u);
                if (not_ready & need) continue;                             // poll again
                uint64_t val = (lane <= first) ? (sv & kSValMask) : 0ull;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(0xffffffffu, val, o);
                excl += val;
                if (incl) break;
                t -= 32;
            }
            if (lane == 0) *my = kSFlagIncl | (excl + agg);
        }
        if (lane == 0) s_excl = excl;
    }
    __syncthreads();
    uint64_t run = s_excl + wbase + inc - tsum;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (base + i < n) {
            out[base + i] = (OutT)run;
            if (fill && v[i]) fill[run] = (uint32_t)(base + i);      // stream compaction of the flagged positions
        }
        run += v[i];
    }
    // the tile holding item n-1 also writes the total
    if (base <= n - 1 && n - 1 < base + kScanItems) {
        out[n] = (OutT)run;
        if (total_out) *total_out = run;
        if (fill) { fill[run] = (uint32_t)n; sc->n_groups = (unsigned int)run; }
    }
}

int scan_scratch_tiles(int64_t N) { return (int)((N + 1 + kScanTile - 1) / kScanTile) + 1; }

template <typename OutT>
static int scan_impl(sph_ctx* c, const uint32_t* in, OutT* out, int64_t n, unsigned long long* total_out,
                     uint32_t* fill = nullptr) {
    if (n <= 0) return SPH_OK;
    int64_t tiles = (n + kScanTile - 1) / kScanTile;
    SPH_CUDA(c, cudaMemsetAsync(c->scan_status, 0, (size_t)tiles * sizeof(uint64_t), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(c->scan_counter, 0, sizeof(uint32_t), c->stream));
    k_scan<OutT><<<(unsigned)tiles, kScanThreads, 0, c->stream>>>(in, out, n, c->scan_status, c->scan_counter, total_out, fill, c->d_sc);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int launch_scan_u32_u64(sph_ctx* c, const uint32_t* in, uint64_t* out, int64_t n, unsigned long long* total_out) {
    return scan_impl<uint64_t>(c, in, (uint64_t*)out, n, total_out);
}
// leaf groups: exclusive scan of the group-start flags (0 / 1) and, in the same pass, grp_lo[g] = first slot of group g,
// grp_lo[n_groups] = n and the group count (tree.cu)
int launch_scan_groups(sph_ctx* c, const uint32_t* gflag, uint32_t* gscan, uint32_t* grp_lo, int64_t n) {
    return scan_impl<uint32_t>(c, gflag, gscan, n, nullptr, grp_lo);
}
__global__ void k_store_u32(const unsigned long long* src, unsigned int* dst) { *dst = (unsigned int)*src; }
int launch_scan_u32_u32(sph_ctx* c, const uint32_t* in, uint32_t* out, int64_t n, unsigned int* total_out) {
    // total goes through a u64 scratch word at the end of scan_status
    unsigned long long* tmp = (unsigned long long*)(c->scan_status + (c->scan_tiles - 1));
    SPH_TRY(scan_impl<uint32_t>(c, in, out, n, total_out ? tmp : nullptr));
    if (total_out) {
        k_store_u32<<<1, 1, 0, c->stream>>>(tmp, total_out);
        c->launches++;
    }
    return SPH_OK;
}

}  // namespace sph
