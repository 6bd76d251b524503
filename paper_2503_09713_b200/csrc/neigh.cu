// neigh.cu -- a4: warp-cooperative, stack-based tree traversal per leaf group writing the neighbour cache
// (Alg. 4; Alg. 5 count -> scan -> fill PAPER.md:1114-1148; two-stage idea PAPER.md:1164-1166;
// criteria of App. E, with the cache tolerance chi, reading A2).
//
// One warp per leaf group (<= 32 Morton-contiguous particles; lane = query particle). Stage 1: the warp pops up
// to 32 nodes at a time from a shared-memory stack, each lane tests one node's box, enlarged by
// R_kern chi max(hmax_group, hmax_node), against the group's box under the periodic minimum image (group-group
// criterion); passing nodes with <= 32 particles become candidate buckets, larger ones push both
// children. Stage 2: candidate buckets are staged in shared memory and every lane tests its own particle against
// them with the exact object-object criterion d^2 < (R_kern chi max(h_a,h_b))^2. The arithmetic
// of that test is written without FMA contraction so that the decision is bit-identical to a plain IEEE
// evaluation.
#include "common.cuh"

namespace sph {

constexpr int kTravWarps = 8;            // warps per block
constexpr int kStackCap = 512;           // stack entries per warp
constexpr int kStackSlack = 192;         // above kStackCap - kStackSlack the warp pops one node at a time (pure DFS)
constexpr int kBucketCap = 64;           // candidate buckets buffered before stage 2 runs
constexpr uint32_t kLeafBit = 0x80000000u;

struct TravBox {
    double L[3], halfL[3];
    int periodic[3];
    double gg_pad;                       // absolute slack added to the conservative box test
};

struct TravWarpSmem {
    uint32_t stack[kStackCap];
    uint32_t blo[kBucketCap], bhi[kBucketCap];
    double cx[32], cy[32], cz[32], ch[32];
};

// separation of two intervals [alo,ahi], [blo,bhi] along one axis (0 if they overlap), minimum over periodic images
__device__ __forceinline__ double axis_gap(double alo, double ahi, double blo, double bhi, double L, int periodic) {
    double g = fmax(fmax(blo - ahi, alo - bhi), 0.0);
    if (periodic) {
        g = fmin(g, fmax(blo + L - ahi, 0.0));
        g = fmin(g, fmax(alo - bhi + L, 0.0));
    }
    return g;
}

__device__ __forceinline__ double min_image(double d, double L, double halfL, int periodic) {
    if (periodic) {
        if (d > halfL) d = __dsub_rn(d, L);
        else if (d < -halfL) d = __dadd_rn(d, L);
    }
    return d;
}

template <bool FILL>
__global__ void __launch_bounds__(kTravWarps * 32) k_traverse(
    int64_t N, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
    const double* __restrict__ h, const NodeRec* __restrict__ nodes, const uint32_t* __restrict__ grp_lo,
    const DevScalars* sc_in, TravBox tb, double rk_chi, uint32_t* __restrict__ cnt,
    const uint64_t* __restrict__ offs, uint32_t* __restrict__ nbr, uint32_t* work_counter, DevScalars* sc_out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TravWarpSmem& s = reinterpret_cast<TravWarpSmem*>(smem_raw)[threadIdx.x >> 5];
    const unsigned lane = lane_id();
    const unsigned lt = lanemask_lt();
    const uint32_t n_groups = sc_in->n_groups;
    unsigned mn = 0xffffffffu, mx = 0u;

    for (;;) {
        uint32_t g = 0;
        if (lane == 0) g = atomicAdd(work_counter, 1u);     // dynamic work distribution (skewed list lengths)
        g = __shfl_sync(0xffffffffu, g, 0);
        if (g >= n_groups) break;
        const uint32_t glo = grp_lo[g], nq = grp_lo[g + 1] - glo;
        const bool qv = lane < nq;
        const uint32_t a = glo + (qv ? lane : 0);
        const double xq = x[a], yq = y[a], zq = z[a], hq = h[a];
        // group box and max h (lanes beyond nq replicate lane 0)
        const double gxl = warp_min(xq), gxh = warp_max(xq), gyl = warp_min(yq), gyh = warp_max(yq);
        const double gzl = warp_min(zq), gzh = warp_max(zq), ghm = warp_max(hq);
        uint32_t n_found = 0;
        uint64_t wofs = 0;
        if (FILL) wofs = offs[a];

        int sp = 0, nb = 0;
        if (lane == 0) s.stack[0] = (N == 1) ? kLeafBit : 0u;
        sp = 1;
        __syncwarp();

        auto stage2 = [&]() {
            for (int b = 0; b < nb; ++b) {
                const uint32_t blo = s.blo[b], bn = s.bhi[b] - blo + 1;
                __syncwarp();
                if (lane < bn) {
                    s.cx[lane] = x[blo + lane]; s.cy[lane] = y[blo + lane];
                    s.cz[lane] = z[blo + lane]; s.ch[lane] = h[blo + lane];
                }
                __syncwarp();
                if (qv) {
                    for (uint32_t cidx = 0; cidx < bn; ++cidx) {
                        double dx = min_image(__dsub_rn(xq, s.cx[cidx]), tb.L[0], tb.halfL[0], tb.periodic[0]);
                        double dy = min_image(__dsub_rn(yq, s.cy[cidx]), tb.L[1], tb.halfL[1], tb.periodic[1]);
                        double dz = min_image(__dsub_rn(zq, s.cz[cidx]), tb.L[2], tb.halfL[2], tb.periodic[2]);
                        double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
                        double rc = __dmul_rn(rk_chi, fmax(hq, s.ch[cidx]));
                        if (d2 < __dmul_rn(rc, rc)) {
                            if (FILL) nbr[wofs + n_found] = blo + cidx;
                            ++n_found;
                        }
                    }
                }
            }
            nb = 0;
        };

        while (sp > 0) {
            int npop = min(sp, 32);
            if (sp > kStackCap - kStackSlack) npop = 1;
            bool have = (int)lane < npop;
            uint32_t e = have ? s.stack[sp - 1 - lane] : 0u;
            sp -= npop;
            __syncwarp();
            bool pass = false, small = false;
            uint32_t rlo = 0, rhi = 0, split = 0;
            if (have) {
                double blo[3], bhi[3], bhm;
                if (e & kLeafBit) {
                    rlo = rhi = e & ~kLeafBit;
                    blo[0] = bhi[0] = x[rlo]; blo[1] = bhi[1] = y[rlo]; blo[2] = bhi[2] = z[rlo];
                    bhm = h[rlo];
                    small = true;
                } else {
                    const double2* p = reinterpret_cast<const double2*>(nodes + e);
                    double2 v0 = __ldg(p), v1 = __ldg(p + 1), v2 = __ldg(p + 2), v3 = __ldg(p + 3);
                    blo[0] = v0.x; blo[1] = v0.y; blo[2] = v1.x; bhi[0] = v1.y; bhi[1] = v2.x; bhi[2] = v2.y;
                    bhm = v3.x;
                    long long ints = __double_as_longlong(v3.y);
                    int32_t other = (int32_t)(ints & 0xffffffffll);
                    split = (uint32_t)(ints >> 32);
                    rlo = min(e, (uint32_t)other);
                    rhi = max(e, (uint32_t)other);
                    small = (rhi - rlo + 1) <= (uint32_t)kGroup;
                }
                // group-group criterion, conservative under rounding (tiny pad)
                double ext = rk_chi * fmax(ghm, bhm) * (1.0 + 1e-9) + tb.gg_pad;
                pass = axis_gap(gxl, gxh, blo[0], bhi[0], tb.L[0], tb.periodic[0]) <= ext &&
                       axis_gap(gyl, gyh, blo[1], bhi[1], tb.L[1], tb.periodic[1]) <= ext &&
                       axis_gap(gzl, gzh, blo[2], bhi[2], tb.L[2], tb.periodic[2]) <= ext;
            }
            const bool push = pass && !small, emit = pass && small;
            const unsigned pm = __ballot_sync(0xffffffffu, push), em = __ballot_sync(0xffffffffu, emit);
            if (push) {
                int at = sp + 2 * __popc(pm & lt);
                s.stack[at] = (rhi == split + 1) ? (kLeafBit | (split + 1)) : (split + 1);
                s.stack[at + 1] = (rlo == split) ? (kLeafBit | split) : split;
            }
            sp += 2 * __popc(pm);
            if (emit) {
                int at = nb + __popc(em & lt);
                s.blo[at] = rlo;
                s.bhi[at] = rhi;
            }
            nb += __popc(em);
            __syncwarp();
            if (nb > kBucketCap - 32) stage2();
        }
        __syncwarp();
        stage2();

        if (!FILL) {
            if (qv) {
                cnt[a] = n_found;
                mn = min(mn, n_found);
                mx = max(mx, n_found);
            }
        }
    }
    if (!FILL) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
            mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        }
        if (lane == 0 && mx >= mn) {
            atomicMin(&sc_out->nbr_min, mn);
            atomicMax(&sc_out->nbr_max, mx);
        }
    }
}

__global__ void k_trav_reset(uint32_t* work_counter, DevScalars* sc, int reset_minmax) {
    *work_counter = 0u;
    if (reset_minmax) { sc->nbr_min = 0xffffffffu; sc->nbr_max = 0u; }
}

int launch_traverse(sph_ctx* c, bool fill) {
    static bool attr_set = false;
    const int smem = (int)sizeof(TravWarpSmem) * kTravWarps;
    if (!attr_set) {
        SPH_CUDA(c, cudaFuncSetAttribute(k_traverse<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        SPH_CUDA(c, cudaFuncSetAttribute(k_traverse<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        attr_set = true;
    }
    TravBox tb;
    double Lmax = 0.0;
    for (int k = 0; k < 3; ++k) {
        tb.L[k] = c->box.hi[k] - c->box.lo[k];
        tb.halfL[k] = 0.5 * tb.L[k];
        tb.periodic[k] = c->box.periodic[k];
        Lmax = fmax(Lmax, tb.L[k]);
    }
    tb.gg_pad = 1e-14 * Lmax;
    const double rk_chi = kRkern * c->p.chi;
    uint32_t* wc = c->sort_counters + 8;   // spare counter word
    k_trav_reset<<<1, 1, 0, c->stream>>>(wc, c->d_sc, fill ? 0 : 1);
    // persistent grid: enough warps to fill the machine, work handed out through an atomic counter
    int64_t warps_needed = (c->N + 31) / 32;   // upper bound on useful warps is the group count <= N
    unsigned blocks = (unsigned)min((int64_t)148 * 6, (warps_needed + kTravWarps - 1) / kTravWarps);
    if (blocks == 0) blocks = 1;
    if (fill)
        k_traverse<true><<<blocks, kTravWarps * 32, smem, c->stream>>>(c->N, c->cur.x, c->cur.y, c->cur.z, c->cur.h,
                                                                       c->nodes, c->grp_lo, c->d_sc, tb, rk_chi, c->cnt,
                                                                       c->offs, c->nbr, wc, c->d_sc);
    else
        k_traverse<false><<<blocks, kTravWarps * 32, smem, c->stream>>>(c->N, c->cur.x, c->cur.y, c->cur.z, c->cur.h,
                                                                        c->nodes, c->grp_lo, c->d_sc, tb, rk_chi, c->cnt,
                                                                        c->offs, c->nbr, wc, c->d_sc);
    c->launches += 2;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
