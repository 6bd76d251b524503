// neigh.cu -- a4: warp-cooperative, stack-based tree traversal per leaf group writing the neighbour cache
// (Alg. 4; Alg. 5; two-stage idea PAPER.md:1164-1166; criteria of App. E,
// PAPER.md:1217-1229, with the cache tolerance chi, reading A2).
//
// One warp per leaf group (<= 32 Morton-contiguous particles; lane = query particle), ONE pass. A warp takes kShare
// consecutive groups at a time and walks the tree once for their common box, collecting the bucket nodes within
// reach; each group then only re-tests those buckets against its own box (stage 1 is mostly the thinly populated
// top of the tree, and consecutive groups share it).
//   Stage 1: the warp pops up to 32 nodes at a time from a shared-memory stack; each lane tests one node's box,
//     enlarged by R_kern chi max(hmax_group, hmax_node), against the group's box under the periodic minimum image
//     (group-group criterion). Passing nodes with <= 32 particles become candidate buckets (slot
//     ranges), larger ones push both children.
//   Stage 2: each bucket is staged in shared memory (positions and the precomputed cutoff square of every
//     candidate) and every lane tests its own particle against it with the exact object-object criterion
//     d^2 < (R_kern chi max(h_a,h_b))^2, written without FMA contraction so that the decision is
//     bit-identical to a plain IEEE evaluation. (R_kern chi h)^2 is precomputed per particle: rounding, scaling
//     by a positive constant and squaring are monotone, so max() commutes with them exactly. Buckets whose union
//     box with the group spans at most L/2 on every periodic axis cannot wrap and take a loop without the
//     minimum-image selects (the decision is exact).
//     Fast path (a4): the exact test is only needed for pairs close to the cutoff. Each group works in
//     coordinates relative to the centre of its box, scaled by a power of two so that its reach is O(1), and rounded
//     to fp32; the test runs in packed fp32 (two candidates per FADD2 / FMUL2 / FFMA2), with an error bound derived
//     from the 2^-24 roundings of the relative coordinates. A bucket in which some lane saw |d^2 - cutoff^2| inside
//     that bound is tested again with the plain IEEE fp64 expressions (from global memory): every decision that is
//     kept is provably the fp64 one, so the sets stay bit-exact.
//   Output (the cache): the group's candidate array (the sorted slots of the candidates that passed
//     the prefilter, in traversal order) and, per particle, the ascending list of 16-bit indices into that
//     candidate array. Hits are buffered in shared memory, candidate slots in a per-warp global scratch row, and
//     both are written out coalesced once the group is complete; space comes from two bump allocators (count ->
//     allocate -> fill per group; the host re-runs the pass with larger pools if one overflowed). A group whose
//     lists outgrow the shared-memory rows spills them to a per-warp scratch in global memory; beyond that (lists
//     longer than kSpillCap + the row capacity, more than kScrCap candidates) it allocates from its exact counts and walks a
//     second time writing directly.
#include <stdlib.h>

#include "common.cuh"

namespace sph {

constexpr int kTravWarps = 8;            // warps per block
constexpr int kStackCap = 512;           // stack entries per warp
constexpr int kStackSlack = 192;         // above kStackCap - kStackSlack the warp pops one node at a time (pure DFS)
constexpr int kPendCap = 64;             // candidate buckets buffered before stage 2 runs
constexpr int kHitCapR2 = 112, kHitCapR3 = 224;   // buffered hits per lane: kernels of radius 2; M5 / M6
constexpr int kTravWarpsR3 = 5;          // warps per block with the larger rows
constexpr int kHitSlack = 32;            // room for one more bucket beyond kHitCap (overflow is checked per bucket)
static_assert((kHitCapR2 + kHitSlack + 8) % 8 == 0 && (kHitCapR3 + kHitSlack + 8) % 8 == 0, "hit rows are copied as 16-byte words");
constexpr int kShare = 4;               // consecutive groups that share one tree walk
constexpr int kUbCap = 192;             // bucket nodes collected by the shared walk
constexpr int kSpillCap = 512;            // hits per lane that can spill from the shared-memory row to the warp's global scratch
constexpr int kScrCap = 2048;            // candidate slots buffered per group (global scratch row of the warp)
constexpr uint32_t kLeafBit = 0x80000000u;
constexpr uint32_t kWrapBit = 0x80000000u;

struct TravBox {
    double L[3], halfL[3];
    int periodic[3];
    double gg_pad;                       // absolute slack added to the conservative box test
    uint32_t gmax;                       // nodes with <= gmax particles are buckets (sph_params.group_max)
    double kappa;                        // ((1 + kShellEps) / chi)^2 (at most 1): inner threshold / cache threshold
    float kappa_f;
    const uint32_t* lscan;               // Alg. 1 variant (else null): scan of the removal mask; a bucket must also lie
                                         // inside one reduced leaf: lscan[hi + 1] == lscan[lo + 1]
};

// HC = hit-row capacity in entries (lists of a group's particles are buffered here): 112 for the kernels of radius 2
// (about 81 neighbours at h_fact 1.2), 224 for M5 / M6 (about 157), which then run five warps per CTA
template <int HC>
struct TravWarpSmemT {
    static constexpr int kCap = HC, kStride = HC + kHitSlack + 8;   // in u16; rows 16-byte aligned (copied out as uint4)
    uint32_t stack[kStackCap];
    uint32_t plo[kPendCap + 1], pn[kPendCap + 1];   // pending buckets: first slot | wrap bit, particle count (+ a sentinel)
    float2 pkb[kPendCap + 1];                 // per pending bucket, from its reach and the group's (bucket_bounds): the prefilter's
                                              // slack K and the fast path's uncertainty band B, in the group's scaled units
    float4 cand[kGroup + 4];                  // staged candidates (compacted), in pairs: {x0, x1, y0, y1}, {z0, z1, r0, r1}:
                                              // scaled fp32 coordinates relative to the group's centre, r = cutoff^2
    uint32_t cslotb[kGroup];                  // their sorted slots (exact path)
    uint32_t ub[kUbCap];                      // bucket nodes within reach of the kShare groups' common box
    __align__(16) uint16_t hits[32 * kStride];
};

struct TravOut {
    uint32_t* cnt;
    uint32_t* cnt_in;
    uint64_t* lstart;
    uint16_t* lists;
    uint64_t list_cap;
    uint32_t* cslot;
    uint64_t cslot_cap;
    uint32_t* scratch;       // kScrCap entries per warp of the grid
    uint16_t* hit_scratch;   // 32 x kSpillCap entries per warp of the grid: spilled parts of the hit rows
    GroupRec* ginfo;
    uint64_t ginfo_cap;
};

// min / max by compare-and-select: operands here are never NaN, and fmin()/fmax() expand to a NaN-safe sequence of
// about six instructions on sm_100
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
// max(a, 0) by the sign bit (integer pipe; `a > 0 ? a : 0` compiles to a NaN-quieting fp64 max of six instructions)
__device__ __forceinline__ double clamp0(double a) { return __double2hiint(a) >= 0 ? a : 0.0; }

// separation of two intervals [alo,ahi], [blo,bhi] along one axis (0 if they overlap), minimum over periodic images
__device__ __forceinline__ double axis_gap(double alo, double ahi, double blo, double bhi, double L, int periodic) {
    double g = clamp0(dmax(blo - ahi, alo - bhi));
    if (periodic) {
        g = dmin(g, clamp0(blo + L - ahi));
        g = dmin(g, clamp0(alo - bhi + L));
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

// per-lane / per-group traversal state
struct GroupCtx {
    double xq, yq, zq, rc2q;
    double gxl, gxh, gyl, gyh, gzl, gzh, ghm;
    double rc2g;          // (R_kern chi hmax_group)^2, for the per-candidate prefilter
    uint32_t nhit;        // per lane: hits so far (exact)
    uint32_t nin;         // per lane: inner hits so far (exact)
    uint32_t wpos;        // per lane: inner entries in the lane's row (DIRECT: inner entries written)
    uint32_t cpos;        // per lane: shell entries in the lane's row, from the top (DIRECT: shell entries written)
    uint32_t nspill;      // per lane, buffered mode: inner hits of this group already spilled to the warp's global scratch
    uint32_t cspill;      // per lane, buffered mode: shell hits already spilled (they fill the scratch row from its top)
    uint16_t* lcend;      // DIRECT: this lane's first shell entry in global memory (right after its inner entries)
    float kin_a;          // per lane: kappa * ra2, the inner threshold of the query in scaled fp32
    bool hard_overflow;   // warp-uniform: a row could not spill any more (the group is walked a second time)
    uint16_t* hspill;     // warp-uniform: the warp's hit scratch (row p = hspill + p * kSpillCap belongs to lane p)
    uint32_t ncs;         // warp-uniform: candidates (prefilter survivors) so far
    uint16_t* lptr;       // DIRECT: this lane's list in global memory
    uint32_t* cptr;       // candidate slots: the warp's scratch row, or (DIRECT) the group's array in global memory
    bool can_write;       // DIRECT: allocation succeeded
    bool anywrap;         // warp-uniform: some bucket of this group may wrap around a periodic axis
    // fp32 fast path (warp-uniform unless marked): coordinates relative to (cx, cy, cz), scaled by sc (a power of two)
    bool use32;
    double cx, cy, cz, sc, ksc;   // ksc = R_kern chi sc
    float ax, ay, az, ra2, rca;   // per lane: scaled relative position, cutoff^2 and cutoff (rounded up) of the query
    float ex, ey, ez;             // scaled half extents of the group's box, rounded up
    float twoA, rcg, rc2g_f;      // 2 max(ex, ey, ez); scaled reach of the group (rounded up) and its square
};

// d2 < a || d2 < b as two predicate-combining compares (the compiler otherwise builds a NaN-safe fp64 max)
__device__ __forceinline__ bool lt_either(double d2, double a, double b) {
    int r;
    asm("{\n\t.reg .pred p;\n\tsetp.lt.f64 p, %1, %2;\n\tsetp.lt.or.f64 p, %1, %3, p;\n\tselp.s32 %0, 1, 0, p;\n\t}"
        : "=r"(r) : "d"(d2), "d"(a), "d"(b));
    return r != 0;
}

// packed fp32 pairs (sm_100: FADD2 / FMUL2 / FFMA2, two candidates per instruction)
__device__ __forceinline__ unsigned long long pk2(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(unsigned long long v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long sub2(unsigned long long a, unsigned long long b) {
    unsigned long long r;
    asm("sub.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ unsigned long long mul2(unsigned long long a, unsigned long long b) {
    unsigned long long r;
    asm("mul.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// A particle's list has two segments: the INNER entries, d < R_kern (1 + kShellEps) max(h_a, h_b) at
// build time, and the SHELL entries beyond (cached for the chi tolerance; they can only matter to a later kernel if some
// h grew by more than kShellEps). The lane's row in shared memory fills from both ends: inner entries upwards from the
// row start (ascending candidate index), shell entries downwards from the row top.
template <bool DIRECT>
__device__ __forceinline__ void record_inner(GroupCtx& G, uint32_t& wp, uint32_t local) {
    if (DIRECT) {
        if (G.can_write) G.lptr[G.wpos] = (uint16_t)local;
        ++G.wpos;
    } else {
        // wp = 32-bit shared-memory address of the lane's next free entry; the row keeps kHitSlack entries free at the
        // start of a bucket, so no capacity check is needed inside it
        // no "memory" clobber: the hit rows alias nothing that is read inside a bucket's test loop, and the loads of
        // the next candidates must be free to move above this store (stage2 closes the loop with a compiler barrier)
        asm volatile("st.shared.u16 [%0], %1;" :: "r"(wp), "h"((unsigned short)local));
        wp += 2u;
    }
}
template <bool DIRECT>
__device__ __forceinline__ void record_shell(GroupCtx& G, uint32_t& wq, uint32_t local) {
    if (DIRECT) {
        if (G.can_write) G.lcend[G.cpos] = (uint16_t)local;
        ++G.cpos;
    } else {
        wq -= 2u;
        asm volatile("st.shared.u16 [%0], %1;" :: "r"(wq), "h"((unsigned short)local));
    }
}

// fast path: inner if vin <= band, else shell if v < 0; predicated stores and pointer updates, no branches
template <bool DIRECT>
__device__ __forceinline__ void record_fast(GroupCtx& G, uint32_t& wp, uint32_t& wq, float vin, float v, float band,
                                            uint32_t local) {
    if (DIRECT) {
        if (vin <= band) record_inner<true>(G, wp, local);
        else if (v < 0.f) record_shell<true>(G, wq, local);
    } else {
        asm volatile(
            "{\n\t.reg .pred pi, ps;\n\t"
            "setp.le.f32 pi, %2, %3;\n\t"
            "setp.lt.and.f32 ps, %4, 0f00000000, !pi;\n\t"
            "@pi st.shared.u16 [%0], %5;\n\t"
            "@pi add.u32 %0, %0, 2;\n\t"
            "@ps add.u32 %1, %1, -2;\n\t"
            "@ps st.shared.u16 [%1], %5;\n\t}"
            : "+r"(wp), "+r"(wq) : "f"(vin), "f"(band), "f"(v), "h"((unsigned short)local));
    }
}

// Error bound of the fp32 fast path, in the group's scaled units. Relative coordinates r = x - centre (min-imaged for
// buckets that may wrap) are exact to 2^-53 |r| in fp64 and are rounded once to fp32: |fl(r) - r| <= 2^-24 |r|. With
// |r_a| <= A (half extent of the group's box) and |r_b| <= A + 3.01 rcm + 6 E for every candidate that passed the
// prefilter below, each difference d_k = fl(r_a,k - r_b,k) has |d_k - true| <= E := 1.3e-7 (2 A + 3.1 rcm) (2^-23 =
// 1.19e-7), hence |d2_f - d2| <= 2 sqrt(3) E d + 3 E^2 + 3.01 2^-24 d2, the thresholds carry 2^-24 (query) and 3 2^-24
// (candidate: (float)(R chi h s) squared) relative, and
// for every test of a bucket  |v_f - v| <= B/4,  B := E (14 rcm' + 12 E) + 2.5e-6 rcm'^2,  v = d2 - max(cutoff^2),
// rcm' = the larger of the GROUP's and the bucket's reach, which bounds every query lane's (true hit: d <= rcm'; true miss: d2 - err(d) is increasing in
// d beyond rcm', or E > rcm' / sqrt(3) and 12 E^2 covers it). So |v_f| > B implies sign(v_f) = sign(v), and sign(v) is
// the fp64 decision because that differs from the real-number one only within 1e-15 relative of the cutoff.
template <bool DIRECT, class S>
__device__ __forceinline__ void stage2(S& s, GroupCtx& G, int npend, unsigned lane, unsigned lt,
                                       const double* __restrict__ x, const double* __restrict__ y,
                                       const double* __restrict__ z, const double* __restrict__ h,
                                       const TravBox& tb, double rk_chi) {
    const uint32_t rowbase = (uint32_t)__cvta_generic_to_shared(&s.hits[lane * S::kStride]);
    const uint32_t rowtop = rowbase + 2u * (uint32_t)(S::kCap + kHitSlack);
    uint32_t wp = rowbase + 2u * G.wpos;          // 32-bit shared-memory addresses: next free inner entry,
    uint32_t wq = rowtop - 2u * G.cpos;           // lowest shell entry
    const unsigned long long nkap2 = pk2(-tb.kappa_f, -tb.kappa_f);
    const unsigned long long ax2 = pk2(G.ax, G.ax), ay2 = pk2(G.ay, G.ay), az2 = pk2(G.az, G.az);
    // software pipeline: the next bucket's candidate (one per lane) is in flight while this one is tested
    double px = 0.0, py = 0.0, pz = 0.0, ph = 0.0;
    if (lane == 0) { s.plo[npend] = 0u; s.pn[npend] = 0u; }      // sentinel: the prefetch past the last bucket loads nothing
    __syncwarp();
    {
        const uint32_t blo = s.plo[0] & ~kWrapBit;
        if (lane < s.pn[0]) { px = x[blo + lane]; py = y[blo + lane]; pz = z[blo + lane]; ph = h[blo + lane]; }
    }
    for (int b = 0; b < npend; ++b) {
        const uint32_t plo = s.plo[b], bn = s.pn[b];
        const uint32_t blo = plo & ~kWrapBit;
        const bool wrap = (plo & kWrapBit) != 0u;
        G.anywrap |= wrap;
        const double cx = px, cy = py, cz = pz, ch = ph;
        {
            const uint32_t nlo = s.plo[b + 1] & ~kWrapBit;
            if (lane < s.pn[b + 1]) { px = x[nlo + lane]; py = y[nlo + lane]; pz = z[nlo + lane]; ph = h[nlo + lane]; }
        }
        // per-candidate prefilter (one lane per candidate): squared distance from the candidate to the group's box
        // against the larger of its own and the group's cutoff, conservative under rounding
        bool keep = lane < bn;
        float fx = 0.f, fy = 0.f, fz = 0.f, fr = 0.f, band = 0.f;
        if (G.use32) {
            double rx = cx - G.cx, ry = cy - G.cy, rz = cz - G.cz;
            if (wrap) {   // nearest periodic image of the candidate relative to the group's centre (unique: see launch)
                rx = min_image(rx, tb.L[0], tb.halfL[0], tb.periodic[0]);
                ry = min_image(ry, tb.L[1], tb.halfL[1], tb.periodic[1]);
                rz = min_image(rz, tb.L[2], tb.halfL[2], tb.periodic[2]);
            }
            fx = (float)(rx * G.sc); fy = (float)(ry * G.sc); fz = (float)(rz * G.sc);
            fr = (float)(ch * G.ksc);                    // scaled cutoff radius, then its square: 3 roundings of 2^-24
            fr *= fr;
            const float2 kb = s.pkb[b];                  // K = 16 E (rcm + E), B = E (14 rcm + 12 E) + 2.5e-6 rcm^2
            const float gx = fmaxf(fabsf(fx) - G.ex, 0.f), gy = fmaxf(fabsf(fy) - G.ey, 0.f), gz = fmaxf(fabsf(fz) - G.ez, 0.f);
            keep = keep && (gx * gx + gy * gy + gz * gz <= fmaxf(fr, G.rc2g_f) * 1.0001f + kb.x);
            band = kb.y;
        } else if (keep && !wrap) {   // plain fp64 version (groups too large for the scaled frame); wrapping buckets keep all
            const double rc = __dmul_rn(rk_chi, ch);
            const double rc2 = __dmul_rn(rc, rc);
            const double gx = clamp0(dmax(G.gxl - cx, cx - G.gxh));
            const double gy = clamp0(dmax(G.gyl - cy, cy - G.gyh));
            const double gz = clamp0(dmax(G.gzl - cz, cz - G.gzh));
            keep = gx * gx + gy * gy + gz * gz <= dmax(rc2, G.rc2g) * (1.0 + 1e-9);
        }
        const unsigned km = __ballot_sync(0xffffffffu, keep);
        const uint32_t nk = (uint32_t)__popc(km), pos = (uint32_t)__popc(km & lt);
        __syncwarp();                                   // readers of the previous bucket are done
        float* const cf = reinterpret_cast<float*>(s.cand);
        if (keep) {
            float* q = cf + (pos >> 1) * 8 + (pos & 1u);   // pair pos / 2, element pos & 1
            q[0] = fx; q[2] = fy; q[4] = fz; q[6] = fr;
            s.cslotb[pos] = blo + lane;
            if (DIRECT ? G.can_write : (G.ncs + pos < (uint32_t)kScrCap)) G.cptr[G.ncs + pos] = blo + lane;
        }
        if (lane < 4u) {                                // four candidates nobody can hit behind the last one
            const uint32_t pp = nk + lane;
            float* q = cf + (pp >> 1) * 8 + (pp & 1u);
            q[0] = 1e18f; q[2] = 1e18f; q[4] = 1e18f; q[6] = 0.f;
        }
        __syncwarp();
        const uint32_t w0 = wp, q0 = wq;
        const uint32_t wpos0 = G.wpos, cpos0 = G.cpos;       // (DIRECT counts entries written in these)
        bool exact = !G.use32;
        if (G.use32) {
            float amin = 3e38f;
            uint32_t id = G.ncs;
            for (uint32_t j = 0; j < nk; j += 4, id += 4) {
                // four candidates per trip, all loads before the first hit store (the assembler keeps shared-memory
                // loads behind earlier shared-memory stores)
                float4 c[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) c[u] = s.cand[j + u];
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const float4 c0 = c[2 * u], c1 = c[2 * u + 1];
                    const unsigned long long dx = sub2(ax2, pk2(c0.x, c0.y)), dy = sub2(ay2, pk2(c0.z, c0.w));
                    const unsigned long long dz = sub2(az2, pk2(c1.x, c1.y));
                    const unsigned long long d2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
                    // M = the larger cutoff^2 of the pair; v = d2 - M (< 0: hit), vin = d2 - kappa M (<= band: inner)
                    const unsigned long long m2 = pk2(fmaxf(c1.z, G.ra2), fmaxf(c1.w, G.ra2));
                    float v0, v1, i0, i1;
                    upk2(sub2(d2, m2), v0, v1);
                    upk2(fma2(m2, nkap2, d2), i0, i1);
                    amin = fminf(amin, fminf(fabsf(v0), fabsf(v1)));
                    record_fast<DIRECT>(G, wp, wq, i0, v0, band, id + 2 * u);
                    record_fast<DIRECT>(G, wp, wq, i1, v1, band, id + 2 * u + 1);
                }
            }
            asm volatile("" ::: "memory");
            // some test of this bucket too close to its cutoff for fp32: the bucket is decided again in fp64
            exact = __any_sync(0xffffffffu, amin <= band);
            if (exact) { wp = w0; wq = q0; G.wpos = wpos0; G.cpos = cpos0; }
        }
        if (exact) {
            // plain IEEE fp64 test, no FMA contraction: bit-identical to the oracle's decision. One candidate at a
            // time from global memory (warp-uniform addresses); rare on the fast path's workloads
            for (uint32_t j = 0; j < nk; ++j) {
                const uint32_t sl = s.cslotb[j];
                const double rcb = __dmul_rn(rk_chi, h[sl]);
                const double rc2b = __dmul_rn(rcb, rcb);
                double dx = __dsub_rn(G.xq, x[sl]), dy = __dsub_rn(G.yq, y[sl]), dz = __dsub_rn(G.zq, z[sl]);
                if (wrap) {
                    dx = min_image(dx, tb.L[0], tb.halfL[0], tb.periodic[0]);
                    dy = min_image(dy, tb.L[1], tb.halfL[1], tb.periodic[1]);
                    dz = min_image(dz, tb.L[2], tb.halfL[2], tb.periodic[2]);
                }
                const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
                if (lt_either(d2, G.rc2q, rc2b)) {
                    // shell only if surely beyond the inner radius of both (a shell entry wrongly kept inner costs
                    // time, never correctness)
                    if (d2 >= tb.kappa * dmax(G.rc2q, rc2b) * (1.0 + 1e-9)) record_shell<DIRECT>(G, wq, G.ncs + j);
                    else record_inner<DIRECT>(G, wp, G.ncs + j);
                }
            }
            asm volatile("" ::: "memory");
        }
        if (!DIRECT) {
            G.wpos = (wp - rowbase) >> 1;
            G.cpos = (rowtop - wq) >> 1;
            // A row keeps room for one more bucket only while it holds at most HC entries: when some lane is beyond
            // that, every lane moves its row to its part of the warp's global scratch (same two-ended layout; the
            // order of the inner entries is kept: spilled part, then the row); when that is full too the group is
            // counted on and walked a second time writing directly.
            if (__any_sync(0xffffffffu, G.wpos + G.cpos > (uint32_t)S::kCap)) {
                if (!G.hard_overflow &&
                    __all_sync(0xffffffffu, G.nspill + G.wpos + G.cspill + G.cpos <= (uint32_t)kSpillCap)) {
                    // the warp moves one row at a time (coalesced 16-bit stores)
                    __syncwarp();
                    for (uint32_t p = 0; p < 32u; ++p) {
                        const uint32_t wn = __shfl_sync(0xffffffffu, G.wpos, p), ns = __shfl_sync(0xffffffffu, G.nspill, p);
                        const uint32_t cn = __shfl_sync(0xffffffffu, G.cpos, p), cs = __shfl_sync(0xffffffffu, G.cspill, p);
                        uint16_t* dst = G.hspill + (size_t)p * kSpillCap + ns;
                        for (uint32_t k = lane; k < wn; k += 32) dst[k] = s.hits[p * S::kStride + k];
                        uint16_t* dsc = G.hspill + (size_t)p * kSpillCap + (kSpillCap - cs - cn);
                        for (uint32_t k = lane; k < cn; k += 32) dsc[k] = s.hits[p * S::kStride + (S::kCap + kHitSlack - cn) + k];
                    }
                    __syncwarp();
                } else {
                    G.hard_overflow = true;       // the rows' content no longer matters, only the counts
                }
                G.nspill += G.wpos;
                G.cspill += G.cpos;
                G.wpos = 0u;
                G.cpos = 0u;
                wp = rowbase;
                wq = rowtop;
            }
        }
        G.ncs += nk;
    }
    // exact counts so far: inner = spilled + in the row (DIRECT: written), all = inner + shell
    G.nin = (DIRECT ? 0u : G.nspill) + G.wpos;
    G.nhit = G.nin + (DIRECT ? 0u : G.cspill) + G.cpos;
}

// The two error-bound terms of a bucket on the fp32 fast path (derivation above stage2), computed once per bucket by the
// lane that found it: with rcm = the larger reach of the GROUP and the bucket (>= the rcm' of any query lane of the
// group, so the band is the same or wider than the per-lane one: conservative) and E = 1.3e-7 (2 A + 3.1 rcm).
__device__ __forceinline__ float2 bucket_bounds(float prc, const GroupCtx& G) {
    const float rcm = fmaxf(prc, G.rcg);
    const float E = 1.3e-7f * (G.twoA + 3.1f * rcm);
    return make_float2(16.f * E * (rcm + E), E * (14.f * rcm + 12.f * E) + 2.5e-6f * rcm * rcm);
}

// One node against the box / hmax of G: group-group criterion on the squared box-box gap under the
// minimum image, conservative under rounding (tiny pad); `wrap` says whether any (query, candidate) separation can
// exceed L/2 on a periodic axis (exact: rounding is monotone). Entry e = internal node index, or leaf slot | kLeafBit.
struct NodeHit { bool pass, small, wrap; uint32_t rlo, rhi, split; float prc; };
__device__ __forceinline__ NodeHit node_test(uint32_t e, const GroupCtx& G, const double* __restrict__ x,
                                             const double* __restrict__ y, const double* __restrict__ z,
                                             const double* __restrict__ h, const NodeRec* __restrict__ nodes,
                                             const TravBox& tb, double rk_chi) {
    NodeHit r;
    double blo[3], bhi[3], bhm;
    r.split = 0u;
    if (e & kLeafBit) {
        r.rlo = r.rhi = e & ~kLeafBit;
        blo[0] = bhi[0] = x[r.rlo]; blo[1] = bhi[1] = y[r.rlo]; blo[2] = bhi[2] = z[r.rlo];
        bhm = h[r.rlo];
        r.small = true;
    } else {
        const double2* p = reinterpret_cast<const double2*>(nodes + e);
        const double2 v0 = __ldg(p), v1 = __ldg(p + 1), v2 = __ldg(p + 2), v3 = __ldg(p + 3);
        blo[0] = v0.x; blo[1] = v0.y; blo[2] = v1.x; bhi[0] = v1.y; bhi[1] = v2.x; bhi[2] = v2.y;
        bhm = v3.x;
        const long long ints = __double_as_longlong(v3.y);
        const int32_t other = (int32_t)(ints & 0xffffffffll);
        r.split = (uint32_t)(ints >> 32);
        r.rlo = min(e, (uint32_t)other);
        r.rhi = max(e, (uint32_t)other);
        r.small = (r.rhi - r.rlo + 1) <= tb.gmax;
        if (tb.lscan && r.small) r.small = __ldg(tb.lscan + r.rhi + 1) == __ldg(tb.lscan + r.rlo + 1);
    }
    r.prc = (float)(rk_chi * bhm * G.sc) * 1.000001f;   // the node's reach in the group's scaled units, rounded up
    const double ext = rk_chi * dmax(G.ghm, bhm) * (1.0 + 1e-9) + tb.gg_pad;
    const double ggx = axis_gap(G.gxl, G.gxh, blo[0], bhi[0], tb.L[0], tb.periodic[0]);
    const double ggy = axis_gap(G.gyl, G.gyh, blo[1], bhi[1], tb.L[1], tb.periodic[1]);
    const double ggz = axis_gap(G.gzl, G.gzh, blo[2], bhi[2], tb.L[2], tb.periodic[2]);
    r.pass = ggx * ggx + ggy * ggy + ggz * ggz <= ext * ext;
    r.wrap = (tb.periodic[0] && (dmax(G.gxh, bhi[0]) - dmin(G.gxl, blo[0]) > tb.halfL[0])) ||
             (tb.periodic[1] && (dmax(G.gyh, bhi[1]) - dmin(G.gyl, blo[1]) > tb.halfL[1])) ||
             (tb.periodic[2] && (dmax(G.gzh, bhi[2]) - dmin(G.gzl, blo[2]) > tb.halfL[2]));
    return r;
}

// Walk of the tree for a box U that encloses several consecutive groups: collects the bucket nodes (<= 32
// particles) within reach of U into s.ub. Every bucket a member group needs is among them: the group's box lies
// inside U and its hmax is not larger, every operation of the test is monotone, so a node that passes the group's
// test passes U's, and so do all its ancestors. Returns the number of buckets, or -1 if s.ub overflowed.
template <class S>
__device__ __forceinline__ int walk_collect(S& s, const GroupCtx& U, unsigned lane, unsigned lt, int64_t N,
                                            const double* __restrict__ x, const double* __restrict__ y,
                                            const double* __restrict__ z, const double* __restrict__ h,
                                            const NodeRec* __restrict__ nodes, const TravBox& tb, double rk_chi) {
    int sp = 1, nu = 0;
    __syncwarp();
    if (lane == 0) s.stack[0] = (N == 1) ? kLeafBit : 0u;
    __syncwarp();
    while (sp > 0) {
        int npop = min(sp, 32);
        if (sp > kStackCap - kStackSlack) npop = 1;
        const bool have = (int)lane < npop;
        const uint32_t e = have ? s.stack[sp - 1 - lane] : 0u;
        sp -= npop;
        __syncwarp();
        NodeHit r;
        r.pass = false; r.small = false;
        if (have) r = node_test(e, U, x, y, z, h, nodes, tb, rk_chi);
        const bool push = r.pass && !r.small, emit = r.pass && r.small;
        const unsigned pm = __ballot_sync(0xffffffffu, push), em = __ballot_sync(0xffffffffu, emit);
        if (push) {
            const int at = sp + 2 * __popc(pm & lt);
            s.stack[at] = (r.rhi == r.split + 1) ? (kLeafBit | (r.split + 1)) : (r.split + 1);
            s.stack[at + 1] = (r.rlo == r.split) ? (kLeafBit | r.split) : r.split;
        }
        sp += 2 * __popc(pm);
        if (nu + __popc(em) > kUbCap) return -1;
        if (emit) s.ub[nu + __popc(em & lt)] = e;
        nu += __popc(em);
        __syncwarp();
    }
    return nu;
}

// One group's buckets out of the collected ones (the same test with the group's own box), then stage 2.
template <bool DIRECT, class S>
__device__ __forceinline__ void refine(S& s, GroupCtx& G, int nu, unsigned lane, unsigned lt,
                                       const double* __restrict__ x, const double* __restrict__ y,
                                       const double* __restrict__ z, const double* __restrict__ h,
                                       const NodeRec* __restrict__ nodes, const TravBox& tb, double rk_chi) {
    G.nhit = 0u; G.nin = 0u; G.wpos = 0u; G.cpos = 0u; G.nspill = 0u; G.cspill = 0u; G.hard_overflow = false; G.ncs = 0u; G.anywrap = false;
    int nb = 0;
    __syncwarp();
    for (int base = 0; base < nu; base += 32) {
        const bool have = base + (int)lane < nu;
        NodeHit r;
        r.pass = false; r.wrap = false; r.rlo = 0u; r.rhi = 0u; r.prc = 0.f;
        if (have) r = node_test(s.ub[base + lane], G, x, y, z, h, nodes, tb, rk_chi);
        const unsigned em = __ballot_sync(0xffffffffu, r.pass);
        if (r.pass) {
            const int at = nb + __popc(em & lt);
            s.plo[at] = r.rlo | (r.wrap ? kWrapBit : 0u);
            s.pn[at] = r.rhi - r.rlo + 1;
            s.pkb[at] = bucket_bounds(r.prc, G);
        }
        nb += __popc(em);
        __syncwarp();
        if (nb > kPendCap - 32) { stage2<DIRECT>(s, G, nb, lane, lt, x, y, z, h, tb, rk_chi); nb = 0; }
    }
    __syncwarp();
    stage2<DIRECT>(s, G, nb, lane, lt, x, y, z, h, tb, rk_chi);
    __syncwarp();
}

// one complete walk of the tree for the group described by G (used when the shared walk overflowed s.ub)
template <bool DIRECT, class S>
__device__ __forceinline__ void walk(S& s, GroupCtx& G, unsigned lane, unsigned lt, int64_t N,
                                     const double* __restrict__ x, const double* __restrict__ y,
                                     const double* __restrict__ z, const double* __restrict__ h,
                                     const NodeRec* __restrict__ nodes, const TravBox& tb, double rk_chi) {
    G.nhit = 0u; G.nin = 0u; G.wpos = 0u; G.cpos = 0u; G.nspill = 0u; G.cspill = 0u; G.hard_overflow = false; G.ncs = 0u; G.anywrap = false;
    int sp = 1, nb = 0;
    __syncwarp();
    if (lane == 0) s.stack[0] = (N == 1) ? kLeafBit : 0u;
    __syncwarp();
    while (sp > 0) {
        int npop = min(sp, 32);
        if (sp > kStackCap - kStackSlack) npop = 1;
        const bool have = (int)lane < npop;
        const uint32_t e = have ? s.stack[sp - 1 - lane] : 0u;
        sp -= npop;
        __syncwarp();
        NodeHit r;
        r.pass = false; r.small = false; r.wrap = false; r.rlo = 0u; r.rhi = 0u; r.split = 0u; r.prc = 0.f;
        if (have) r = node_test(e, G, x, y, z, h, nodes, tb, rk_chi);
        const bool push = r.pass && !r.small, emit = r.pass && r.small;
        const unsigned pm = __ballot_sync(0xffffffffu, push), em = __ballot_sync(0xffffffffu, emit);
        if (push) {
            const int at = sp + 2 * __popc(pm & lt);
            s.stack[at] = (r.rhi == r.split + 1) ? (kLeafBit | (r.split + 1)) : (r.split + 1);
            s.stack[at + 1] = (r.rlo == r.split) ? (kLeafBit | r.split) : r.split;
        }
        sp += 2 * __popc(pm);
        if (emit) {
            const int at = nb + __popc(em & lt);
            s.plo[at] = r.rlo | (r.wrap ? kWrapBit : 0u);
            s.pn[at] = r.rhi - r.rlo + 1;
            s.pkb[at] = bucket_bounds(r.prc, G);
        }
        nb += __popc(em);
        __syncwarp();
        if (nb > kPendCap - 32) { stage2<DIRECT>(s, G, nb, lane, lt, x, y, z, h, tb, rk_chi); nb = 0; }
    }
    __syncwarp();
    stage2<DIRECT>(s, G, nb, lane, lt, x, y, z, h, tb, rk_chi);
    __syncwarp();
}

// Box and max h of a leaf group: the group is a tree node (or a single leaf), so its tight box and hmax are the record
// k_aabb_groups wrote for it (the exact min / max of its particles' positions and h): no reduction over the lanes.
struct GBox { double xl, yl, zl, xh, yh, zh, hm; };
__device__ __forceinline__ GBox group_box(uint32_t glo, uint32_t nq, const double* __restrict__ x,
                                          const double* __restrict__ y, const double* __restrict__ z,
                                          const double* __restrict__ h, const NodeRec* __restrict__ nodes) {
    GBox b;
    if (nq == 1u) {
        b.xl = b.xh = x[glo]; b.yl = b.yh = y[glo]; b.zl = b.zh = z[glo]; b.hm = h[glo];
    } else {
        // the node whose range is the whole group: its index is one end of the range
        const uint32_t root = ((uint32_t)__ldg(&nodes[glo].other) == glo + nq - 1u) ? glo : glo + nq - 1u;
        const double2* p = reinterpret_cast<const double2*>(nodes + root);
        const double2 v0 = __ldg(p), v1 = __ldg(p + 1), v2 = __ldg(p + 2), v3 = __ldg(p + 3);
        b.xl = v0.x; b.yl = v0.y; b.zl = v1.x; b.xh = v1.y; b.yh = v2.x; b.zh = v2.y; b.hm = v3.x;
    }
    return b;
}

__device__ __forceinline__ uint32_t warp_sum_u32(uint32_t v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ uint32_t warp_max_u32(uint32_t v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

template <int HC, int W>
__global__ void __launch_bounds__(W * 32, 2) k_traverse(
    int64_t N, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
    const double* __restrict__ h, const NodeRec* __restrict__ nodes, const uint32_t* __restrict__ grp_lo,
    TravBox tb, double rk_chi, TravOut out, uint32_t* work_counter, DevScalars* sc, uint32_t chunk) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // (values that every bucket of every group needs are passed through empty asm statements: the compiler otherwise
    // recomputes them inside the bucket loop -- a tenth of the kernel's instructions -- although registers are free)
    unsigned soff = (threadIdx.x >> 5) * (unsigned)sizeof(TravWarpSmemT<HC>);
    asm volatile("" : "+r"(soff));
    TravWarpSmemT<HC>& s = *reinterpret_cast<TravWarpSmemT<HC>*>(smem_raw + soff);
    const unsigned lane = lane_id();
    const unsigned lt = lanemask_lt();
    const uint32_t n_groups = sc->n_groups;
    const double reach_max = rk_chi * sc->h_max * 1.001;   // the largest cutoff radius of any particle (k_hmax ran before)
    unsigned mn = 0xffffffffu, mx = 0u, ncmax = 0u;
    uint16_t* const hit_row = out.hit_scratch + ((size_t)blockIdx.x * W + (threadIdx.x >> 5)) * (32 * kSpillCap);
    uint32_t* scr_row = out.scratch + ((size_t)blockIdx.x * W + (threadIdx.x >> 5)) * kScrCap;
    asm volatile("" : "+l"(scr_row));

    for (;;) {
        uint32_t g0 = 0;
        if (lane == 0) g0 = atomicAdd(work_counter, chunk);   // dynamic work distribution, chunk = 1 or kShare groups
        g0 = __shfl_sync(0xffffffffu, g0, 0);
        if (g0 >= n_groups) break;
        const uint32_t ng = min(chunk, n_groups - g0);
        // ---- one walk for the common box of the kShare consecutive groups (a contiguous slot range) ----
        // Sharing pays only if the groups are neighbours in space as well as in Morton order: compare the volume
        // within reach of the common box with the largest one of a member group.
        int nu = -1;
        if (ng > 1u) {
            GroupCtx U;
            U.sc = 1.0;
            U.gxl = U.gyl = U.gzl = 1e300; U.gxh = U.gyh = U.gzh = -1e300; U.ghm = 0.0;
            double vmax = 0.0, vmin = 1e300;
            for (uint32_t g = g0; g < g0 + ng; ++g) {
                const uint32_t glo = grp_lo[g], nq = grp_lo[g + 1] - glo;
                const GBox gb = group_box(glo, nq, x, y, z, h, nodes);
                const double rr = 2.0 * rk_chi * gb.hm;
                const double vg = (gb.xh - gb.xl + rr) * (gb.yh - gb.yl + rr) * (gb.zh - gb.zl + rr);
                vmax = dmax(vmax, vg); vmin = dmin(vmin, vg);
                U.gxl = dmin(U.gxl, gb.xl); U.gxh = dmax(U.gxh, gb.xh); U.gyl = dmin(U.gyl, gb.yl); U.gyh = dmax(U.gyh, gb.yh);
                U.gzl = dmin(U.gzl, gb.zl); U.gzh = dmax(U.gzh, gb.zh); U.ghm = dmax(U.ghm, gb.hm);
            }
            const double rr = 2.0 * rk_chi * U.ghm;
            const double vu = (U.gxh - U.gxl + rr) * (U.gyh - U.gyl + rr) * (U.gzh - U.gzl + rr);
            if (vu <= 3.0 * vmax && vmax <= 4.0 * vmin) {
                nu = walk_collect(s, U, lane, lt, N, x, y, z, h, nodes, tb, rk_chi);
                if (lane == 0) atomicAdd(nu >= 0 ? &sc->n_chunks_shared : &sc->n_chunks_overflow, 1u);
            }
        }
        for (uint32_t g = g0; g < g0 + ng; ++g) {
        const uint32_t glo = grp_lo[g], nq = grp_lo[g + 1] - glo;
        GroupCtx G;
        const bool qv = lane < nq;
        const uint32_t a = glo + (qv ? lane : 0);
        const double hq = h[a];
        G.xq = x[a]; G.yq = y[a]; G.zq = z[a];
        {
            const double rc = __dmul_rn(rk_chi, hq);
            G.rc2q = __dmul_rn(rc, rc);
        }
        {   // group box and max h
            const GBox gb = group_box(glo, nq, x, y, z, h, nodes);
            G.gxl = gb.xl; G.gxh = gb.xh; G.gyl = gb.yl; G.gyh = gb.yh; G.gzl = gb.zl; G.gzh = gb.zh; G.ghm = gb.hm;
        }
        {
            const double rcg = __dmul_rn(rk_chi, G.ghm);
            G.rc2g = __dmul_rn(rcg, rcg);
        }
        {
            // fp32 frame of this group: centre and half extents of its box, scale 2^-e with e the exponent of its reach
            // (every scaled quantity of the group is O(1) whatever the units). Usable if the scaled numbers are far
            // from fp32's limits and, on periodic axes, half extent + the largest reach of any particle stays below
            // L/2: then the periodic image of a candidate nearest to the centre is the one nearest to every query
            // that can reach it, and a wrong image can only turn a far miss into another far miss.
            const double rcg = rk_chi * G.ghm;
            const int eb = (__double2hiint(rcg) >> 20) & 0x7ff;
            const double hx = 0.5 * (G.gxh - G.gxl), hy = 0.5 * (G.gyh - G.gyl), hz = 0.5 * (G.gzh - G.gzl);
            G.sc = __hiloint2double((2046 - eb) << 20, 0);
            G.cx = 0.5 * (G.gxl + G.gxh); G.cy = 0.5 * (G.gyl + G.gyh); G.cz = 0.5 * (G.gzl + G.gzh);
            const double As = dmax(hx, dmax(hy, hz)) * G.sc;
            G.use32 = eb > 523 && eb < 1523 && As < 1e12 &&
                      (!tb.periodic[0] || hx + reach_max < tb.halfL[0]) && (!tb.periodic[1] || hy + reach_max < tb.halfL[1]) &&
                      (!tb.periodic[2] || hz + reach_max < tb.halfL[2]);
            if (!G.use32) G.sc = 1.0;
            G.ksc = rk_chi * G.sc;
            G.ex = (float)(hx * G.sc) * 1.000001f; G.ey = (float)(hy * G.sc) * 1.000001f; G.ez = (float)(hz * G.sc) * 1.000001f;
            G.twoA = 2.f * fmaxf(G.ex, fmaxf(G.ey, G.ez));
            G.rcg = (float)(rcg * G.sc) * 1.000001f;
            G.rc2g_f = (float)(G.rc2g * G.sc * G.sc);
            G.ax = (float)((G.xq - G.cx) * G.sc); G.ay = (float)((G.yq - G.cy) * G.sc); G.az = (float)((G.zq - G.cz) * G.sc);
            G.ra2 = (float)(G.rc2q * G.sc * G.sc);
            G.rca = (float)(rk_chi * hq * G.sc) * 1.000001f;
            G.kin_a = tb.kappa_f * G.ra2;
            asm volatile("" : "+f"(G.ex), "+f"(G.ey), "+f"(G.ez), "+f"(G.twoA), "+f"(G.rcg), "+f"(G.rc2g_f));
            asm volatile("" : "+d"(G.sc), "+d"(G.ksc), "+d"(G.cx), "+d"(G.cy), "+d"(G.cz));
        }
        if (!qv) { G.xq = -1e300; G.rc2q = 0.0; G.ax = G.ay = G.az = -1e18f; G.ra2 = 0.f; G.rca = 0.f; G.kin_a = 0.f; }   // lanes without a particle can never hit
        G.lptr = nullptr; G.cptr = scr_row; G.can_write = false;
        G.hspill = hit_row;

        if (nu >= 0) refine<false>(s, G, nu, lane, lt, x, y, z, h, nodes, tb, rk_chi);
        else walk<false>(s, G, lane, lt, N, x, y, z, h, nodes, tb, rk_chi);

        // ---- allocate from the exact counts: lists and candidate slots ----
        // A particle's list: its inner entries, then its shell entries (any order); every list starts at a multiple of
        // eight entries (16 B), so that rows are copied out as uint4
        const uint32_t nhit = qv ? G.nhit : 0u, nin = qv ? G.nin : 0u;
        const uint32_t nhit4 = (nhit + 7u) & ~7u;
        const uint32_t nc = G.ncs, nc4 = (nc + 3u) & ~3u;
        uint32_t incl = nhit4;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= (unsigned)o) incl += t;
        }
        const uint32_t total = __shfl_sync(0xffffffffu, incl, 31), total_exact = __reduce_add_sync(0xffffffffu, nhit);
        const uint32_t total_inner = __reduce_add_sync(0xffffffffu, nin);
        unsigned long long lbase = 0, bbase = 0;
        if (lane == 0) {
            lbase = atomicAdd(&sc->list_cursor, (unsigned long long)((total + 7u) & ~7u));
            bbase = atomicAdd(&sc->cslot_cursor, (unsigned long long)nc4);
            atomicAdd(&sc->n_neigh, (unsigned long long)total_exact);
            atomicAdd(&sc->n_inner, (unsigned long long)total_inner);
        }
        lbase = __shfl_sync(0xffffffffu, lbase, 0);
        bbase = __shfl_sync(0xffffffffu, bbase, 0);
        const bool fits = (lbase + ((total + 7u) & ~7u) <= out.list_cap) && (bbase + nc4 <= out.cslot_cap) &&
                          ((uint64_t)g < out.ginfo_cap) && (nc <= 65535u);
        const uint64_t my_start = lbase + (incl - nhit4);
        if (qv) {
            out.cnt[a] = nhit;
            out.cnt_in[a] = nin;
            out.lstart[a] = my_start;
        }
        if (fits) {
            if (lane == 0) {
                GroupRec r;
                r.cs_off_lo = (uint32_t)(bbase & 0xffffffffull); r.cs_off_hi = (uint32_t)(bbase >> 32);
                r.nc = nc | (G.anywrap ? 0x80000000u : 0u); r.pad = 0u;
                out.ginfo[g] = r;
            }
            const bool overflow = G.hard_overflow || (nc > (uint32_t)kScrCap);
            if (!overflow) {
                __syncwarp();
                {   // candidate slots, four per lane and copy (both sides 16-byte aligned; the padding is never read)
                    const uint4* src = reinterpret_cast<const uint4*>(scr_row);
                    uint4* dst = reinterpret_cast<uint4*>(out.cslot + bbase);
                    for (uint32_t j = lane; j < (nc4 >> 2); j += 32) dst[j] = src[j];
                }
                const bool spilled = __any_sync(0xffffffffu, (G.nspill | G.cspill) != 0u);
                if (!spilled) {
                    // every lane copies its own row, 16 bytes per store: a store instruction touches 32 lists, half a
                    // sector each, and consecutive instructions fill the sectors in L2; a row-by-row copy by the whole
                    // warp is coalesced but costs 30 times the instructions
                    // (the lane first moves its shell entries from the row top down to the end of its inner entries)
                    uint16_t* rowp = &s.hits[lane * (HC + kHitSlack + 8)];
                    for (uint32_t k = 0; k < nhit - nin; ++k) rowp[nin + k] = rowp[(HC + kHitSlack) - (nhit - nin) + k];
                    const uint4* src = reinterpret_cast<const uint4*>(rowp);
                    uint4* dst = reinterpret_cast<uint4*>(out.lists + my_start);
                    for (uint32_t k = 0; k < (nhit4 >> 3); ++k) dst[k] = src[k];
                } else {
                    // the warp copies one particle's list at a time: spilled inner part, inner part of the row, then
                    // the shell entries of the row and of the scratch (any order)
                    for (uint32_t p = 0; p < nq; ++p) {
                        const uint32_t np8 = __shfl_sync(0xffffffffu, nhit4, p);
                        uint64_t sp0 = lbase + (__shfl_sync(0xffffffffu, incl, p) - np8);
                        const uint32_t ns = __shfl_sync(0xffffffffu, G.nspill, p), wn = __shfl_sync(0xffffffffu, G.wpos, p);
                        const uint32_t cs = __shfl_sync(0xffffffffu, G.cspill, p), cn = __shfl_sync(0xffffffffu, G.cpos, p);
                        const uint16_t* src = hit_row + (size_t)p * kSpillCap;
                        for (uint32_t k = lane; k < ns; k += 32) out.lists[sp0 + k] = src[k];
                        for (uint32_t k = lane; k < wn; k += 32) out.lists[sp0 + ns + k] = s.hits[p * (HC + kHitSlack + 8) + k];
                        const uint64_t se = sp0 + ns + wn;
                        for (uint32_t k = lane; k < cn; k += 32) out.lists[se + k] = s.hits[p * (HC + kHitSlack + 8) + (HC + kHitSlack - cn) + k];
                        for (uint32_t k = lane; k < cs; k += 32) out.lists[se + cn + k] = src[kSpillCap - cs + k];
                    }
                }
            } else {
                // fallback: second walk writing directly at the now-known positions
                G.lptr = out.lists + my_start;
                G.lcend = G.lptr + nin;
                G.cptr = out.cslot + bbase;
                G.can_write = true;
                if (nu >= 0) refine<true>(s, G, nu, lane, lt, x, y, z, h, nodes, tb, rk_chi);
                else walk<true>(s, G, lane, lt, N, x, y, z, h, nodes, tb, rk_chi);
                if (lane == 0) atomicAdd(&sc->n_fallback, 1u);
            }
        }
        if (nc > 65535u && lane == 0) atomicAdd(&sc->n_cand_overflow, 1u);
        if (qv) { mn = min(mn, nhit); mx = max(mx, nhit); }
        ncmax = max(ncmax, nc);
        }   // groups of the chunk
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if (lane == 0) {
        if (mx >= mn) { atomicMin(&sc->nbr_min, mn); atomicMax(&sc->nbr_max, mx); }
        atomicMax(&sc->nc_max, ncmax);
    }
}

__global__ void k_trav_reset(uint32_t* work_counter, DevScalars* sc) {
    *work_counter = 0u;
    sc->nbr_min = 0xffffffffu; sc->nbr_max = 0u;
    sc->list_cursor = 0ull; sc->cslot_cursor = 0ull; sc->n_neigh = 0ull; sc->n_inner = 0ull;
    sc->nc_max = 0u; sc->n_cand_overflow = 0u; sc->n_chunks_shared = 0u; sc->n_chunks_overflow = 0u; sc->n_fallback = 0u;
}

constexpr int kTravBlocks = 148 * 2;     // persistent grid: two CTAs per SM (shared-memory bound)
size_t trav_scratch_entries() { return (size_t)kTravBlocks * kTravWarps * kScrCap; }
size_t trav_hit_scratch_entries() { return (size_t)kTravBlocks * kTravWarps * 32 * kSpillCap; }

int launch_traverse(sph_ctx* c) {
    // hit rows sized for the kernel's neighbour count: radius 2 -> 112 entries, 8 warps per CTA; M5 / M6 -> 224, 5 warps
    const bool wide = kern_radius(c->p.kernel) > 2.0;
    const int W = wide ? kTravWarpsR3 : kTravWarps;
    const int smem = wide ? (int)sizeof(TravWarpSmemT<kHitCapR3>) * kTravWarpsR3 : (int)sizeof(TravWarpSmemT<kHitCapR2>) * kTravWarps;
    if (wide) SPH_CUDA(c, cudaFuncSetAttribute(k_traverse<kHitCapR3, kTravWarpsR3>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    else SPH_CUDA(c, cudaFuncSetAttribute(k_traverse<kHitCapR2, kTravWarps>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));   // per device: every launch
    TravBox tb;
    double Lmax = 0.0;
    for (int k = 0; k < 3; ++k) {
        tb.L[k] = c->box.hi[k] - c->box.lo[k];
        tb.halfL[k] = 0.5 * tb.L[k];
        tb.periodic[k] = c->box.periodic[k];
        Lmax = fmax(Lmax, tb.L[k]);
    }
    tb.gg_pad = 1e-14 * Lmax;
    tb.gmax = (uint32_t)c->p.group_max;
    tb.lscan = c->p.leaf_reduction >= 1 ? c->lscan : nullptr;
    tb.kappa = fmin(1.0, ((1.0 + kShellEps) / c->p.chi) * ((1.0 + kShellEps) / c->p.chi));
    tb.kappa_f = (float)tb.kappa;
    const double rk_chi = kern_radius(c->p.kernel) * c->p.chi;
    TravOut out;
    out.cnt = c->cnt; out.cnt_in = c->cnt_in; out.lstart = c->lstart; out.lists = c->lists; out.list_cap = c->list_cap;
    out.cslot = c->cslot; out.cslot_cap = c->cslot_cap; out.scratch = c->trav_scratch; out.hit_scratch = c->trav_hit_scratch; out.ginfo = c->ginfo; out.ginfo_cap = c->ginfo_cap;
    uint32_t* wc = c->sort_counters + 8;   // spare counter word
    k_trav_reset<<<1, 1, 0, c->stream>>>(wc, c->d_sc);
    // persistent grid: two CTAs per SM (shared-memory bound), work handed out through an atomic counter
    const int64_t warps_needed = (c->N + 31) / 32;
    unsigned blocks = (unsigned)min((int64_t)kTravBlocks, (warps_needed + W - 1) / W);
    if (blocks == 0) blocks = 1;
    // Shared walks (kShare consecutive groups per warp) pay when there are many groups per warp and the groups of a
    // chunk are alike; api.cu switches them off for good if the last pass shared too few chunks.
    // SPH_FORCE_SHARE=1 (tests) forces shared walks whatever the problem size.
    const bool force = getenv("SPH_FORCE_SHARE") != nullptr;
    const uint32_t chunk = (force || (!c->share_disabled && c->n_groups >= (int64_t)32 * kTravBlocks * W)) ? kShare : 1u;
    c->last_chunk = chunk;
    if (wide)
        k_traverse<kHitCapR3, kTravWarpsR3><<<blocks, W * 32, smem, c->stream>>>(c->N, c->cur.x, c->cur.y, c->cur.z, c->cur.h, c->nodes,
                                                                              c->grp_lo, tb, rk_chi, out, wc, c->d_sc, chunk);
    else
        k_traverse<kHitCapR2, kTravWarps><<<blocks, W * 32, smem, c->stream>>>(c->N, c->cur.x, c->cur.y, c->cur.z, c->cur.h, c->nodes,
                                                                            c->grp_lo, tb, rk_chi, out, wc, c->d_sc, chunk);
    c->launches += 2;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

// ---- getter path: group-local lists -> global CSR over sorted slots (sph_get_neighbours) ----
__global__ void __launch_bounds__(256) k_cache_to_csr(int64_t N, const uint32_t* __restrict__ gscan,
                                                      const GroupRec* __restrict__ ginfo,
                                                      const uint32_t* __restrict__ cslot,
                                                      const uint32_t* __restrict__ cnt,
                                                      const uint32_t* __restrict__ cnt_in,
                                                      const uint64_t* __restrict__ lstart,
                                                      const uint16_t* __restrict__ lists,
                                                      const uint64_t* __restrict__ offs, uint32_t* __restrict__ idx,
                                                      int64_t first, int64_t count) {
    const int64_t a = first + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= first + count) return;
    const uint32_t g = gscan[a + 1] - 1u;          // gscan = exclusive scan of the group-start flags
    const GroupRec gr = ginfo[g];
    const uint32_t* cs = cslot + (((uint64_t)gr.cs_off_hi << 32) | gr.cs_off_lo);
    const uint16_t* li = lists + lstart[a];
    const uint32_t n = cnt[a];
    const uint64_t o = offs[a] - offs[first];
    for (uint32_t k = 0; k < n; ++k) idx[o + k] = cs[li[k]];
}

// lists of the sorted slots [first, first + count) into idx_out, which starts at the first slot's list
int launch_cache_to_csr(sph_ctx* c, uint32_t* idx_out, int64_t first, int64_t count) {
    k_cache_to_csr<<<div_up(count, 256), 256, 0, c->stream>>>(c->N, c->gscan, c->ginfo, c->cslot, c->cnt, c->cnt_in, c->lstart,
                                                              c->lists, c->offs, idx_out, first, count);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
