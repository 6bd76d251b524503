// tree.cu -- a3: Karras binary radix tree over the sorted Morton keys (Table B2
// PAPER.md:899-907; delta operator Eq. B2, with Karras' index tie-break for equal keys, DESIGN.md
// reading O3), a3b: bottom-up tight AABB + max-h per node with atomic visit flags (north_star (3)),
// and the leaf groups: maximal nodes holding <= 32 particles (the paper's ~10-particle reduced leaves,
// PAPER.md:382, obtained here without a second tree definition).
#include "common.cuh"

namespace sph {

// indices are 32-bit: N < 2^30 (sph_init_ex), and i + lmax * d stays within (-2^30, 2^31 - 2]
__device__ __forceinline__ int delta_aug(const uint64_t* __restrict__ key, int N, uint64_t ki, int i, int j) {
    if ((unsigned)j >= (unsigned)N) return -1;
    uint64_t kj = __ldg(key + j);
    if (ki != kj) return __clzll((long long)(ki ^ kj));
    return 64 + __clz(i ^ j);
}

// ---- Alg. 1: removal mask over the sorted codes. Lines 1-5: duplicates; lines 6-22: one
// reduction pass (every thread reads the mask of the previous pass: a synchronous pass, reading A17).
// delta = common-prefix length of the code words (Eq. B2), -1 for a neighbour that does not exist.
__global__ void __launch_bounds__(256) k_leaf_mask_init(int64_t N, const uint64_t* __restrict__ key, uint32_t* __restrict__ xi) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) xi[i] = (i == 0 || key[i] != key[i - 1]) ? 1u : 0u;
}
__global__ void __launch_bounds__(256) k_leaf_reduce_pass(int64_t N, const uint64_t* __restrict__ key,
                                                          const uint32_t* __restrict__ xin, uint32_t* __restrict__ xout) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    if (!xin[i]) { xout[i] = 0u; return; }
    int64_t im1 = i - 1;
    while (im1 >= 0 && !xin[im1]) --im1;
    int64_t im2 = im1 - 1;
    while (im2 >= 0 && !xin[im2]) --im2;
    int64_t ip1 = i + 1;
    while (ip1 < N && !xin[ip1]) ++ip1;
    const uint64_t ki = key[i];
    const int d0 = (ip1 < N) ? __clzll((long long)(ki ^ key[ip1])) : -1;
    const int dm1 = (im1 >= 0) ? __clzll((long long)(key[im1] ^ ki)) : -1;
    const int dm2 = (im2 >= 0) ? __clzll((long long)(key[im2] ^ key[im1])) : -1;
    xout[i] = (d0 < dm1 && dm2 < dm1) ? 0u : 1u;     // second leaf of a two-leaf parent: removed
}
// kept codes and their index map by the scan of the mask (stream compaction)
__global__ void __launch_bounds__(256) k_leaf_export(int64_t N, const uint64_t* __restrict__ key, const uint32_t* __restrict__ xi,
                                                     const uint32_t* __restrict__ lscan, uint64_t* codes, uint32_t* ids) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    if (xi[i]) {
        if (codes) codes[lscan[i]] = key[i];
        if (ids) ids[lscan[i]] = (uint32_t)i;
    }
    if (i == N - 1 && ids) ids[lscan[N]] = (uint32_t)N;
}

// one thread per internal node i in [0, N-2]
// lscan (may be null): exclusive scan of the Alg. 1 mask; the slots lo..hi lie in one reduced leaf iff no code is kept
// in (lo, hi], i.e. lscan[hi + 1] == lscan[lo + 1]
__global__ void __launch_bounds__(256) k_karras(int64_t N64, const uint64_t* __restrict__ key, NodeRec* __restrict__ nodes,
                                                int32_t* __restrict__ parent, uint32_t* __restrict__ gflag, int gmax,
                                                const uint32_t* __restrict__ lscan, const DevScalars* __restrict__ sc) {
    if (sc->sort_redo) return;   // keys are not in order (sort.cu: k_sort_repair gave up): no groups, nothing downstream runs
    const int N = (int)N64;
    const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x);
    if (i >= N - 1) return;
    const uint64_t ki = key[i];
    const int dn = delta_aug(key, N, ki, i, i + 1), dp = delta_aug(key, N, ki, i, i - 1);
    const int d = (dn - dp) > 0 ? 1 : -1;
    const int dmin = (d > 0) ? dp : dn;
    int lmax = 2;
    while (delta_aug(key, N, ki, i, i + lmax * d) > dmin) lmax <<= 1;
    int l = 0;
    for (int t = lmax >> 1; t >= 1; t >>= 1)
        if (delta_aug(key, N, ki, i, i + (l + t) * d) > dmin) l += t;
    const int j = i + l * d;
    const int dnode = delta_aug(key, N, ki, i, j);
    int s = 0, t = l;
    do {
        t = (t + 1) >> 1;
        if (delta_aug(key, N, ki, i, i + (s + t) * d) > dnode) s += t;
    } while (t > 1);
    const int gamma = i + s * d + (d < 0 ? -1 : 0);
    const int lo = min(i, j), hi = max(i, j);
    nodes[i].other = (int32_t)j;
    nodes[i].split = (int32_t)gamma;
    parent[(lo == gamma) ? (N - 1 + gamma) : gamma] = (int32_t)i;
    parent[(hi == gamma + 1) ? (N - 1 + gamma + 1) : (gamma + 1)] = (int32_t)i;
    if (i == 0) parent[0] = -1;
    // leaf groups: the maximal nodes that hold <= gmax (sph_params.group_max <= kGroup) particles and, in the Alg. 1
    // variant, lie inside one reduced leaf: children that qualify of a node that does not
    auto groupable = [&](int a, int b) { return b - a + 1 <= gmax && (!lscan || lscan[b + 1] == lscan[a + 1]); };
    if (groupable(lo, hi)) {
        if (i == 0) gflag[0] = 1u;   // the whole tree is one group
    } else {
        if (groupable(lo, gamma)) gflag[lo] = 1u;          // left child covers [lo, gamma]
        if (groupable(gamma + 1, hi)) gflag[gamma + 1] = 1u;   // right child covers [gamma + 1, hi]
    }
}

// a3b: bottom-up boxes. A thread carrying a finished child box up the tree announces itself at the parent with an
// atomic flag; the second arrival merges both children and goes on. Sibling records are read with L2 loads (ld.cg)
// issued after the flag atomic has returned, so only the release side (record written -> fence -> flag) needs a fence.
// Group-level boxes, kernel 1 of 2: one warp per leaf group (<= 32 consecutive leaves = one complete subtree).
// Lane j holds leaf glo + j and looks after internal node glo + j if that node lies inside the subtree. The subtree
// is evaluated bottom-up in rounds inside the warp: a node whose children are ready (a leaf always is) fetches their
// boxes with shuffles and merges them. The bottom five levels of the tree thus need no flags, fences or dependent
// L2 round trips, and the records are written once, coalesced.
__global__ void __launch_bounds__(256) k_aabb_groups(int64_t N, const double* __restrict__ x, const double* __restrict__ y,
                                                     const double* __restrict__ z, const double* __restrict__ h,
                                                     NodeRec* nodes, const uint32_t* __restrict__ grp_lo,
                                                     const DevScalars* sc) {
    const unsigned lane = lane_id();
    const uint32_t n_groups = sc->n_groups;
    const uint32_t warps_total = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t g = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; g < n_groups; g += warps_total) {
        const uint32_t glo = grp_lo[g], n = grp_lo[g + 1] - glo;
        if (n < 2u) continue;                                 // a single leaf has no internal node
        const uint32_t a = glo + (lane < n ? lane : 0u);
        const double lx = x[a], ly = y[a], lz = z[a], lh = h[a];
        const int64_t i = (int64_t)glo + lane;
        bool mine = false, lleaf = false, rleaf = false;
        int srcL = 0, srcR = 0;
        if (lane < n && i < N - 1) {
            const int32_t other = nodes[i].other, split = nodes[i].split;
            const int64_t lo = min(i, (int64_t)other), hi = max(i, (int64_t)other);
            mine = lo >= (int64_t)glo && hi < (int64_t)glo + n;
            lleaf = (lo == split); rleaf = (hi == split + 1);
            srcL = mine ? (int)(split - (int64_t)glo) : 0;
            srcR = mine ? srcL + 1 : 0;
        }
        // my node: lo xyz, hi xyz, hmax. Leaf children first (one exchange of the leaves' positions), then rounds over
        // the internal children only: a child whose node is complete hands its box over by shuffles. min / max by
        // compare-and-select (no NaNs here; fmin / fmax expand to NaN-safe sequences); they are exact, so the order in
        // which the two children are merged does not matter.
        auto mn = [](double a, double b) { return a < b ? a : b; };
        auto mx = [](double a, double b) { return a > b ? a : b; };
        const double inf = __longlong_as_double(0x7ff0000000000000ll);
        double b0 = inf, b1 = inf, b2 = inf, b3 = -inf, b4 = -inf, b5 = -inf, b6 = 0.0;
        {
            const double Llx = __shfl_sync(0xffffffffu, lx, srcL), Lly = __shfl_sync(0xffffffffu, ly, srcL);
            const double Llz = __shfl_sync(0xffffffffu, lz, srcL), Llh = __shfl_sync(0xffffffffu, lh, srcL);
            const double Rlx = __shfl_sync(0xffffffffu, lx, srcR), Rly = __shfl_sync(0xffffffffu, ly, srcR);
            const double Rlz = __shfl_sync(0xffffffffu, lz, srcR), Rlh = __shfl_sync(0xffffffffu, lh, srcR);
            if (mine && lleaf) { b0 = Llx; b1 = Lly; b2 = Llz; b3 = Llx; b4 = Lly; b5 = Llz; b6 = Llh; }
            if (mine && rleaf) {
                b0 = mn(b0, Rlx); b1 = mn(b1, Rly); b2 = mn(b2, Rlz); b3 = mx(b3, Rlx); b4 = mx(b4, Rly); b5 = mx(b5, Rlz);
                b6 = mx(b6, Rlh);
            }
        }
        bool needL = mine && !lleaf, needR = mine && !rleaf;
        for (;;) {
            const unsigned dm = __ballot_sync(0xffffffffu, !needL && !needR);      // complete nodes (and idle lanes)
            if (dm == 0xffffffffu) break;
            const bool okL = needL && ((dm >> srcL) & 1u), okR = needR && ((dm >> srcR) & 1u);
            const double L0 = __shfl_sync(0xffffffffu, b0, srcL), L1 = __shfl_sync(0xffffffffu, b1, srcL);
            const double L2 = __shfl_sync(0xffffffffu, b2, srcL), L3 = __shfl_sync(0xffffffffu, b3, srcL);
            const double L4 = __shfl_sync(0xffffffffu, b4, srcL), L5 = __shfl_sync(0xffffffffu, b5, srcL);
            const double L6 = __shfl_sync(0xffffffffu, b6, srcL);
            const double R0 = __shfl_sync(0xffffffffu, b0, srcR), R1 = __shfl_sync(0xffffffffu, b1, srcR);
            const double R2 = __shfl_sync(0xffffffffu, b2, srcR), R3 = __shfl_sync(0xffffffffu, b3, srcR);
            const double R4 = __shfl_sync(0xffffffffu, b4, srcR), R5 = __shfl_sync(0xffffffffu, b5, srcR);
            const double R6 = __shfl_sync(0xffffffffu, b6, srcR);
            if (okL) {
                b0 = mn(b0, L0); b1 = mn(b1, L1); b2 = mn(b2, L2); b3 = mx(b3, L3); b4 = mx(b4, L4); b5 = mx(b5, L5);
                b6 = mx(b6, L6);
                needL = false;
            }
            if (okR) {
                b0 = mn(b0, R0); b1 = mn(b1, R1); b2 = mn(b2, R2); b3 = mx(b3, R3); b4 = mx(b4, R4); b5 = mx(b5, R5);
                b6 = mx(b6, R6);
                needR = false;
            }
        }
        if (mine) {
            double* q = reinterpret_cast<double*>(nodes + i);
            q[0] = b0; q[1] = b1; q[2] = b2; q[3] = b3; q[4] = b4; q[5] = b5; q[6] = b6;
        }
    }
}

// Group-level boxes, kernel 2 of 2: one thread per group carries the group's box (its root node's record, written
// by kernel 1, or the single leaf) up the tree. A thread announces itself at the parent with an atomic flag; the
// second arrival merges both children and goes on. Sibling records are read with L2 loads (ld.cg) issued after the
// flag atomic has returned, so only the release side (record written -> fence -> flag) needs a fence.
__global__ void __launch_bounds__(256) k_aabb_climb(int64_t N, const double* __restrict__ x, const double* __restrict__ y,
                                                    const double* __restrict__ z, const double* __restrict__ h,
                                                    NodeRec* nodes, const int32_t* __restrict__ parent, uint32_t* visit,
                                                    const uint32_t* __restrict__ grp_lo, const DevScalars* sc) {
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= sc->n_groups) return;
    const uint32_t glo = grp_lo[g], n = grp_lo[g + 1] - glo;
    double lo[3], hi[3], hm;
    int32_t cur;
    bool cur_leaf = (n == 1u);
    if (cur_leaf) {
        cur = (int32_t)glo;
        lo[0] = hi[0] = x[glo]; lo[1] = hi[1] = y[glo]; lo[2] = hi[2] = z[glo];
        hm = h[glo];
    } else {
        // the group's root: the internal node whose range is the whole group (its index is one end of the range)
        cur = (nodes[glo].other == (int32_t)(glo + n - 1u)) ? (int32_t)glo : (int32_t)(glo + n - 1u);
        const double* p = reinterpret_cast<const double*>(nodes + cur);
        lo[0] = p[0]; lo[1] = p[1]; lo[2] = p[2]; hi[0] = p[3]; hi[1] = p[4]; hi[2] = p[5]; hm = p[6];
    }
    int32_t node = cur_leaf ? parent[N - 1 + cur] : parent[cur];
    bool wrote = false;                                        // records of kernel 1 are already visible
    while (node >= 0) {
        if (wrote) __threadfence();                            // my record is visible before I announce myself
        if (atomicAdd(&visit[node], 1u) == 0u) return;         // first arrival: the sibling's thread will carry on
        asm volatile("" ::: "memory");                         // keep the sibling loads below the atomic
        const int32_t oth = nodes[node].other, split = nodes[node].split;
        const int32_t nlo = min(node, oth), nhi = max(node, oth);
        const bool lleaf = (nlo == split), rleaf = (nhi == split + 1);
        const bool i_am_left = (cur == split) && (cur_leaf == lleaf);
        const int32_t sib = i_am_left ? split + 1 : split;
        const bool sib_leaf = i_am_left ? rleaf : lleaf;
        double slo[3], shi[3], shm;
        if (sib_leaf) {
            slo[0] = shi[0] = x[sib]; slo[1] = shi[1] = y[sib]; slo[2] = shi[2] = z[sib];
            shm = h[sib];
        } else {
            const double* p = reinterpret_cast<const double*>(nodes + sib);   // through L2: written by another SM
#pragma unroll
            for (int k = 0; k < 3; ++k) { slo[k] = __ldcg(p + k); shi[k] = __ldcg(p + 3 + k); }
            shm = __ldcg(p + 6);
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) { lo[k] = fmin(lo[k], slo[k]); hi[k] = fmax(hi[k], shi[k]); }
        hm = fmax(hm, shm);
        double* q = reinterpret_cast<double*>(nodes + node);
#pragma unroll
        for (int k = 0; k < 3; ++k) { __stcg(q + k, lo[k]); __stcg(q + 3 + k, hi[k]); }
        __stcg(q + 6, hm);
        wrote = true;
        cur = node;
        cur_leaf = false;
        node = parent[node];
    }
}

__global__ void k_single_group(uint32_t* gflag) { gflag[0] = 1u; }

int launch_tree(sph_ctx* c) {
    const int64_t N = c->N;
    SPH_CUDA(c, cudaMemsetAsync(c->gflag, 0, (size_t)N * sizeof(uint32_t), c->stream));
    const uint32_t* lscan = nullptr;
    if (c->p.leaf_reduction >= 1) {
        // Alg. 1: duplicate mask, n_red = leaf_reduction - 1 passes, scan (leaf ids)
        uint32_t *a = c->xi_a, *b = c->xi_b;
        k_leaf_mask_init<<<div_up(N, 256), 256, 0, c->stream>>>(N, c->key, a);
        c->launches++;
        for (int pass = 1; pass < c->p.leaf_reduction; ++pass) {
            k_leaf_reduce_pass<<<div_up(N, 256), 256, 0, c->stream>>>(N, c->key, a, b);
            c->launches++;
            uint32_t* t = a; a = b; b = t;
        }
        c->xi_final = a;
        SPH_TRY(launch_scan_u32_u32(c, a, c->lscan, N, nullptr));
        lscan = c->lscan;
    }
    if (N >= 2) {
        k_karras<<<div_up(N - 1, 256), 256, 0, c->stream>>>(N, c->key, c->nodes, c->parent, c->gflag, c->p.group_max, lscan, c->d_sc);
        c->launches++;
    } else {
        k_single_group<<<1, 1, 0, c->stream>>>(c->gflag);
        c->launches++;
    }
    SPH_TRY(launch_scan_groups(c, c->gflag, c->gscan, c->grp_lo, N));      // scan + grp_lo + group count in one pass
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int launch_leaf_export(sph_ctx* c, uint64_t* codes, uint32_t* ids) {
    k_leaf_export<<<div_up(c->N, 256), 256, 0, c->stream>>>(c->N, c->key, c->xi_final, c->lscan, codes, ids);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int launch_aabb(sph_ctx* c) {
    const int64_t N = c->N;
    if (N < 2) return SPH_OK;
    SPH_CUDA(c, cudaMemsetAsync(c->visit, 0, (size_t)(N - 1) * sizeof(uint32_t), c->stream));
    // the group count of this tree is only known on the device: the climb grid is sized by its upper bound N
    k_aabb_groups<<<148 * 16, 256, 0, c->stream>>>(N, c->cur.x, c->cur.y, c->cur.z, c->cur.h, c->nodes, c->grp_lo, c->d_sc);
    k_aabb_climb<<<div_up(N, 256), 256, 0, c->stream>>>(N, c->cur.x, c->cur.y, c->cur.z, c->cur.h, c->nodes, c->parent, c->visit,
                                                         c->grp_lo, c->d_sc);
    c->launches++;
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
