// tree.cu -- a3: Karras binary radix tree over the sorted Morton keys (Table B2
// PAPER.md:899-907; delta operator Eq. B2, with Karras' index tie-break for equal keys, DESIGN.md
// reading O3), a3b: bottom-up tight AABB + max-h per node with atomic visit flags (north_star (3)),
// and the leaf groups: maximal nodes holding <= 32 particles (the paper's ~10-particle reduced leaves,
// PAPER.md:382, obtained here without a second tree definition).
#include "common.cuh"

namespace sph {

__device__ __forceinline__ int delta_aug(const uint64_t* __restrict__ key, int64_t N, uint64_t ki, int64_t i, int64_t j) {
    if (j < 0 || j >= N) return -1;
    uint64_t kj = __ldg(key + j);
    if (ki != kj) return __clzll((long long)(ki ^ kj));
    return 64 + __clz((int)((uint32_t)i ^ (uint32_t)j));
}

// one thread per internal node i in [0, N-2]
__global__ void __launch_bounds__(256) k_karras(int64_t N, const uint64_t* __restrict__ key, NodeRec* __restrict__ nodes,
                                                int32_t* __restrict__ parent, uint32_t* __restrict__ gflag) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N - 1) return;
    const uint64_t ki = key[i];
    const int dn = delta_aug(key, N, ki, i, i + 1), dp = delta_aug(key, N, ki, i, i - 1);
    const int64_t d = (dn - dp) > 0 ? 1 : -1;
    const int dmin = (d > 0) ? dp : dn;
    int64_t lmax = 2;
    while (delta_aug(key, N, ki, i, i + lmax * d) > dmin) lmax <<= 1;
    int64_t l = 0;
    for (int64_t t = lmax >> 1; t >= 1; t >>= 1)
        if (delta_aug(key, N, ki, i, i + (l + t) * d) > dmin) l += t;
    const int64_t j = i + l * d;
    const int dnode = delta_aug(key, N, ki, i, j);
    int64_t s = 0, t = l;
    do {
        t = (t + 1) >> 1;
        if (delta_aug(key, N, ki, i, i + (s + t) * d) > dnode) s += t;
    } while (t > 1);
    const int64_t gamma = i + s * d + (d < 0 ? -1 : 0);
    const int64_t lo = min(i, j), hi = max(i, j);
    nodes[i].other = (int32_t)j;
    nodes[i].split = (int32_t)gamma;
    parent[(lo == gamma) ? (N - 1 + gamma) : gamma] = (int32_t)i;
    parent[(hi == gamma + 1) ? (N - 1 + gamma + 1) : (gamma + 1)] = (int32_t)i;
    if (i == 0) parent[0] = -1;
    // leaf groups: children of nodes with more than kGroup particles that themselves hold <= kGroup
    if (hi - lo + 1 <= kGroup) {
        if (i == 0) gflag[0] = 1u;   // the whole tree is one group
    } else {
        if (gamma - lo + 1 <= kGroup) gflag[lo] = 1u;        // left child covers [lo, gamma]
        if (hi - gamma <= kGroup) gflag[gamma + 1] = 1u;     // right child covers [gamma + 1, hi]
    }
}

__global__ void __launch_bounds__(256) k_group_fill(int64_t N, const uint32_t* __restrict__ gflag,
                                                    const uint32_t* __restrict__ gscan, uint32_t* __restrict__ grp_lo,
                                                    DevScalars* sc) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    if (gflag[i]) grp_lo[gscan[i]] = (uint32_t)i;
    if (i == N - 1) {
        uint32_t ng = gscan[N];
        grp_lo[ng] = (uint32_t)N;
        sc->n_groups = ng;
    }
}

// bottom-up boxes: one thread per leaf; the second thread to reach a node merges its children and goes on.
// A node whose two children are both leaves needs no flag: the left leaf's thread merges the pair directly and the
// right leaf's thread retires at once (about half of all leaves, so half of the bottom-level atomics and fences).
// Sibling records are read with L2 loads (ld.cg) issued after the flag atomic has returned, so only the release
// side (record written -> fence -> flag) needs a fence.
__global__ void __launch_bounds__(256) k_aabb(int64_t N, const double* __restrict__ x, const double* __restrict__ y,
                                              const double* __restrict__ z, const double* __restrict__ h,
                                              NodeRec* nodes, const int32_t* __restrict__ parent, uint32_t* visit) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    double lo[3] = {x[i], y[i], z[i]}, hi[3] = {lo[0], lo[1], lo[2]}, hm = h[i];
    int32_t cur = (int32_t)i;
    bool cur_leaf = true;
    int32_t node = parent[N - 1 + i];
    while (node >= 0) {
        const int32_t other = nodes[node].other, split = nodes[node].split;
        const int32_t nlo = min(node, other), nhi = max(node, other);
        const bool lleaf = (nlo == split), rleaf = (nhi == split + 1);
        const bool i_am_left = (cur == split) && (cur_leaf == lleaf);
        const int32_t sib = i_am_left ? split + 1 : split;
        const bool sib_leaf = i_am_left ? rleaf : lleaf;
        if (cur_leaf && sib_leaf) {
            if (!i_am_left) return;                       // the left leaf's thread handles the pair
        } else {
            __threadfence();                              // my record is visible before I announce myself
            if (atomicAdd(&visit[node], 1u) == 0u) return;    // first arrival: the sibling's thread will carry on
            asm volatile("" ::: "memory");                // keep the sibling loads below the atomic in program order
        }
        double slo[3], shi[3], shm;
        if (sib_leaf) {
            slo[0] = shi[0] = x[sib]; slo[1] = shi[1] = y[sib]; slo[2] = shi[2] = z[sib];
            shm = h[sib];
        } else {
            const double* p = reinterpret_cast<const double*>(nodes + sib);   // read through L2: written by another SM
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
        cur = node;
        cur_leaf = false;
        node = parent[node];
    }
}

__global__ void k_single_group(uint32_t* gflag) { gflag[0] = 1u; }

int launch_tree(sph_ctx* c) {
    const int64_t N = c->N;
    SPH_CUDA(c, cudaMemsetAsync(c->gflag, 0, (size_t)N * sizeof(uint32_t), c->stream));
    if (N >= 2) {
        k_karras<<<div_up(N - 1, 256), 256, 0, c->stream>>>(N, c->key, c->nodes, c->parent, c->gflag);
        c->launches++;
    } else {
        k_single_group<<<1, 1, 0, c->stream>>>(c->gflag);
        c->launches++;
    }
    SPH_TRY(launch_scan_u32_u32(c, c->gflag, c->gscan, N, nullptr));
    k_group_fill<<<div_up(N, 256), 256, 0, c->stream>>>(N, c->gflag, c->gscan, c->grp_lo, c->d_sc);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int launch_aabb(sph_ctx* c) {
    const int64_t N = c->N;
    if (N < 2) return SPH_OK;
    SPH_CUDA(c, cudaMemsetAsync(c->visit, 0, (size_t)(N - 1) * sizeof(uint32_t), c->stream));
    k_aabb<<<div_up(N, 256), 256, 0, c->stream>>>(N, c->cur.x, c->cur.y, c->cur.z, c->cur.h, c->nodes, c->parent, c->visit);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
