// common.cuh -- shared declarations of libsph_b200 (CUDA, sm_100a only). See include/sph_b200.h for the ABI and
// DESIGN.md for the kernel-by-kernel design. Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <utility>
#include <vector>

#include "../../include/sph_b200.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "libsph_b200 is written for sm_100a (B200) only"
#endif

namespace sph {

constexpr int kGroup = 32;          // leaf-group size bound: one warp lane per particle of a group
// Neighbour lists are split at R_kern (1 + kShellEps) max(h_a, h_b) (h at cache-build time): the entries beyond it
// (the shell kept for the chi tolerance) can only contribute once some smoothing length has grown by
// more than kShellEps since the build; density and forces skip them until then
constexpr double kShellEps = 0.02;
// growth beyond which the shell entries are read: (1 + kShellEps) less the margins of the traversal's classification
constexpr double kShellGrow = (1.0 + kShellEps) * (1.0 - 1e-5);
// B-spline kernels (reading O6): 0 = M4 (cubic), 1 = M5 (quartic), 2 = M6 (quintic);
// support radius in units of h and 3-D normalisation 1/pi, 1/(20 pi), 1/(120 pi)
// 3, 4, 5 = Wendland C2, C4, C6 on the support radius 2h: f = t^4 (1 + 2q), t^6 (1 + 3q + 35/12 q^2),
// t^8 (1 + 4q + 25/4 q^2 + 4 q^3) with t = 1 - q/2; normalisations 21/(16 pi), 495/(256 pi), 1365/(512 pi)
constexpr int kNumKernels = 6;
__host__ __device__ constexpr double kern_radius(int k) { return k == 1 ? 2.5 : (k == 2 ? 3.0 : 2.0); }
__host__ __device__ constexpr double kern_cnorm(int k) {
    return k == 0 ? 0.31830988618379067154 : (k == 1 ? 0.31830988618379067154 / 20.0 : (k == 2 ? 0.31830988618379067154 / 120.0 :
           (k == 3 ? 0.31830988618379067154 * 21.0 / 16.0 : (k == 4 ? 0.31830988618379067154 * 495.0 / 256.0 :
                                                                      0.31830988618379067154 * 1365.0 / 512.0))));
}

// Sorted-order particle fields (SoA). Two sets are kept; the permute writes the other one.
struct Fields {
    double *x, *y, *z, *vx, *vy, *vz, *ax, *ay, *az, *u, *du, *h, *m;
    uint32_t* id;
};
constexpr int kNumF64Fields = 13;

// One record per internal radix-tree node, 64 B: tight box, max h, and the integers the traversal needs.
// A node's index is one end of its key range (Karras convention); `other` is the other end; `split` is the
// left child's id (right child = split + 1); a child is a leaf iff it coincides with the range end on its side.
struct __align__(16) NodeRec {
    double lo[3], hi[3];
    double hmax;
    int32_t other, split;
};
static_assert(sizeof(NodeRec) == 64, "NodeRec must be 64 bytes");

// One leaf group's entry in the neighbour cache: where its candidate array (sorted-slot indices, u32) starts in the
// candidate pool and how many candidates it has (bit 31 of nc: some candidate may wrap around a periodic axis).
struct __align__(16) GroupRec { uint32_t cs_off_lo, cs_off_hi, nc, pad; };

enum Stage { ST_KEYS = 0, ST_SORT, ST_PERMUTE, ST_TREE, ST_AABB, ST_TRAVERSE, ST_SCAN, ST_DENSITY, ST_FORCES,
             ST_LEAPFROG, ST_COUNT };

enum State { S_FIELDS = 0, S_TREE = 1, S_DENSITY = 2, S_FORCES = 3 };

// Device-side scalars read back by the host (one small struct, copied with one cudaMemcpyAsync).
struct DevScalars {
    double dt;                       // global CFL minimum (G8), stored as a double; reduced with atomicMin on bits
    unsigned long long dt_bits;
    unsigned int n_exceeded;         // particles that exceeded chi h^n in the last density pass
    unsigned int n_noconv;           // particles that hit max_h_iter
    unsigned int h_iter_max;
    unsigned int nbr_min, nbr_max;
    unsigned int n_groups;
    unsigned int hmax_bits_hi;       // unused padding
    double h_max;                    // max h^n (periodic-box check)
    unsigned long long n_neigh;      // neighbour total (= offs[N])
    double t;                        // simulated time (sum of the dt actually used)
    // neighbour-cache allocation state of the last traversal (bump allocators + limits seen)
    unsigned long long list_cursor;  // 16-bit list entries handed out (each group's block padded to 8 entries)
    unsigned long long cslot_cursor; // candidate-pool entries handed out (each group's array padded to 4)
    unsigned int nc_max;             // largest candidate count of any group
    unsigned int n_cand_overflow;    // groups with more than 65535 candidates (16-bit local index overflow)
    unsigned int n_chunks_shared;    // traversal chunks that shared one walk / whose shared walk overflowed
    unsigned int n_chunks_overflow;
    double corr_dvmax2, corr_v2sum;  // corrector check G7: max |dv|^2, sum |v|^2 (reading A15)
    unsigned int tie_max;            // longest run of keys equal in their top 40 bits (sort prefix mode)
    unsigned int tie_max32;          // the same for the top 32 bits (runs longer than 65 are reported as 66)
    unsigned int mass_nonuniform;    // set at init if any two particle masses differ
    unsigned int n_fallback;         // groups that took the two-walk fallback (hit or bucket buffer overflow)
    unsigned int sort_redo;          // prefix-mode sort met a run of equal prefixes too long to repair: the tree kernels
                                     // of this build do nothing and the host sorts again with all eight passes
    unsigned long long n_inner;      // inner entries of all lists (the rest are shell entries, neigh.cu)
    unsigned long long n_grew;       // particles flagged by the last density pass (h' > kShellGrow h^n)
    unsigned long long sweeps;       // Newton sweeps + closing passes executed by the last density launch, summed over
                                     // particles (bench.py: measured flop count of k_density)
};

struct TimerRec { int stage; cudaEvent_t e0, e1; };

}  // namespace sph

struct sph_ctx {
    int64_t N = 0;
    sph_box box{};
    sph_params p{};
    cudaStream_t stream = nullptr;
    sph_allocator alloc{};
    int device = 0;                     // the CUDA device this context lives on (every ABI entry makes it current)
    int64_t bytes_allocated = 0;
    std::vector<std::pair<void*, size_t>> allocations;

    sph::Fields cur{}, alt{};
    double *rho = nullptr, *omega = nullptr, *P = nullptr, *cs = nullptr, *A = nullptr;   // A = 1/(rho^2 Omega)
    double *nax = nullptr, *nay = nullptr, *naz = nullptr, *ndu = nullptr;                // a^{n+1}, du/dt^{n+1}
    double* hnew = nullptr;                                                               // Newton output
    // shock switch (sph_params.av_switch): alpha_a in sorted order (two sets: the permute writes the other), alpha c_s
    double *alpha = nullptr, *alpha_alt = nullptr, *acs = nullptr;
    bool alpha_pending = false;         // the next force evaluation starts with the G13 update
    bool in_step = false;               // inside sph_step_leapfrog (the G13 update takes the step's dt, else 0)
    uint64_t *key = nullptr, *key_alt = nullptr;
    uint32_t *val = nullptr, *val_alt = nullptr;
    // radix sort scratch
    uint32_t* sort_hist = nullptr;      // [8][256] global digit histograms -> exclusive bases
    uint32_t* sort_status = nullptr;    // [8][tiles][256] decoupled look-back words
    uint32_t* sort_counters = nullptr;  // [8] dynamic tile ids
    int64_t sort_tiles = 0;
    // tree
    sph::NodeRec* nodes = nullptr;      // N-1
    int32_t* parent = nullptr;          // 2N-1
    uint32_t* visit = nullptr;          // N-1 atomic visit flags
    // groups
    uint32_t* gflag = nullptr;          // N   1 at the first slot of each leaf group
    uint32_t* gscan = nullptr;          // N+1 exclusive scan of gflag (u32)
    uint32_t* grp_lo = nullptr;         // Ng+1 first slot of group g (grp_lo[Ng] = N)
    // Alg. 1 variant (sph_params.leaf_reduction >= 1): removal mask (two buffers, the passes alternate) and its
    // exclusive scan = leaf id of every sorted slot (+1 from the slot's own flag)
    uint32_t *xi_a = nullptr, *xi_b = nullptr, *lscan = nullptr;
    uint32_t* xi_final = nullptr;       // the buffer holding the final mask of the last build
    int64_t n_groups = 0;
    // neighbour cache, group-local (a4): per group a candidate array (sorted slots of the particles
    // that passed the traversal's prefilter) and per particle an ascending list of 16-bit indices into it
    uint32_t* cnt = nullptr;            // N+1  list length of each sorted slot
    uint32_t* cnt_in = nullptr;         // N    of which inner entries (first segment of the list)
    uint8_t* grow = nullptr;            // N    1 if the last density solve left h' > kShellGrow h^n for this slot
    uint64_t* lstart = nullptr;         // N    first entry of each slot's list in `lists`
    uint16_t* lists = nullptr;
    uint64_t list_cap = 0;
    uint32_t* cslot = nullptr;          // candidate pool
    uint64_t cslot_cap = 0;
    uint32_t* trav_scratch = nullptr;   // per-warp candidate rows of the traversal grid
    uint16_t* trav_hit_scratch = nullptr;   // per-warp spill rows of the hit buffers
    sph::GroupRec* ginfo = nullptr;     // one per group
    uint64_t ginfo_cap = 0;
    uint32_t nc_max = 0;
    uint64_t* offs = nullptr;           // N+1  CSR offsets, built only by sph_get_neighbours
    uint64_t n_neigh = 0;
    // scan scratch
    uint64_t* scan_status = nullptr;
    uint32_t* scan_counter = nullptr;
    int64_t scan_tiles = 0;
    // scalars
    sph::DevScalars* d_sc = nullptr;
    sph::DevScalars* h_sc = nullptr;    // pinned
    double* d_dtstep = nullptr;         // dt used by predictor/corrector (device scalar)

    int state = sph::S_FIELDS;
    int restarts_last = 0;
    int64_t steps = 0;
    double t = 0.0;
    int64_t launches = 0;
    bool have_cfl_dt = false;
    double* corr_part = nullptr;        // per-block partials of the corrector check (2 x blocks)
    double cfl_mult = 1.0;              // CFL multiplier lambda_CFL (G9-G10)
    int recycles_last = 0;              // corrector re-cycles of the last step
    int last_sort_passes = 8;
    int sort_p0 = 0;                    // first radix pass: 0 = all eight passes; prefix modes: 3 = top 40 bits + repair,
                                        // 4 = top 32 bits + repair
    bool share_disabled = false;        // traversal: shared walks switched off (too few chunks could share)
    uint32_t last_chunk = 1;
    bool uniform_mass = false;          // all particle masses equal (density kernel variant)

    std::vector<sph::TimerRec> timers;  // open since the last stream synchronisation; folded into ms_acc there
    std::vector<cudaEvent_t> event_pool;
    double ms_acc[sph::ST_COUNT] = {0};
    char err[512] = {0};
};

namespace sph {

// ---- host-side helpers (api.cu) ----
int fail(sph_ctx* c, int code, const char* fmt, ...);
#define SPH_CUDA(c, call)                                                                       \
    do {                                                                                        \
        cudaError_t e_ = (call);                                                                \
        if (e_ != cudaSuccess)                                                                  \
            return sph::fail((c), e_ == cudaErrorMemoryAllocation ? SPH_ERR_OOM : SPH_ERR_DEVICE, \
                             "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)
#define SPH_TRY(expr)             \
    do {                          \
        int rc_ = (expr);         \
        if (rc_ != SPH_OK) return rc_; \
    } while (0)

inline unsigned int div_up(int64_t a, int64_t b) { return (unsigned int)((a + b - 1) / b); }

// ---- stage launchers (one per .cu file); each enqueues on c->stream and bumps c->launches ----
int launch_keys(sph_ctx* c);                                   // keys.cu
int launch_sort(sph_ctx* c);                                   // sort.cu   (key,val) -> sorted into key,val
int launch_permute(sph_ctx* c);                                // permute.cu
int launch_tree(sph_ctx* c);                                   // tree.cu   karras + groups
int launch_leaf_export(sph_ctx* c, uint64_t* codes, uint32_t* ids);   // tree.cu   Alg. 1 leaves -> codes + id map
int launch_aabb(sph_ctx* c);                                   // tree.cu
int launch_traverse(sph_ctx* c);                               // neigh.cu  single pass: walk, test, write cache
int launch_cache_to_csr(sph_ctx* c, uint32_t* idx_out, int64_t first, int64_t count);   // neigh.cu  group-local lists -> CSR (getter)
size_t trav_hit_scratch_entries();                              // neigh.cu  u16 entries of the traversal's hit spill rows
size_t trav_scratch_entries();                                  // neigh.cu  u32 entries of the traversal's scratch rows
int launch_scan_u32_u64(sph_ctx* c, const uint32_t* in, uint64_t* out, int64_t n, unsigned long long* total_out);  // scan.cu
int launch_scan_u32_u32(sph_ctx* c, const uint32_t* in, uint32_t* out, int64_t n, unsigned int* total_out);        // scan.cu
int launch_scan_groups(sph_ctx* c, const uint32_t* gflag, uint32_t* gscan, uint32_t* grp_lo, int64_t n);               // scan.cu
int launch_density(sph_ctx* c);                                // density.cu
int launch_forces(sph_ctx* c);                                 // forces.cu
int launch_alpha(sph_ctx* c, const double* dtp);               // alpha.cu  G12-G13 update of alpha_a, alpha c_s
int launch_predict(sph_ctx* c);                                // leapfrog.cu
int launch_correct(sph_ctx* c, bool with_check);                           // leapfrog.cu
int launch_hmax(sph_ctx* c);                                   // leapfrog.cu  max h^n -> d_sc->h_max
int launch_adopt_acc(sph_ctx* c);                              // leapfrog.cu  a^n <- a^{n+1} (white step)
int launch_set_dt(sph_ctx* c, double user_dt);                 // leapfrog.cu  device dt for predictor/corrector; t += dt
int launch_scatter_orig_f64(sph_ctx* c, const double* src_sorted, double* dst_orig, int ncomp);   // permute.cu
int launch_gather_orig_f64(sph_ctx* c, const double* src_orig, double* dst_sorted, int ncomp);    // permute.cu
int sort_scratch_bytes(int64_t N, int64_t* tiles, size_t* status_bytes);
int scan_scratch_tiles(int64_t N);

// ---- device helpers ----
#ifdef __CUDACC__
__device__ __forceinline__ unsigned lane_id() { return threadIdx.x & 31u; }
__device__ __forceinline__ unsigned lanemask_lt() { unsigned m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m; }

__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// M4 cubic B-spline f(q) and f'(q) (reading O6); branch-light form.
__device__ __forceinline__ void m4(double q, double& f, double& df);
// max(a, 0) by the sign bit (integer pipe): a = +-0 gives 0 either way
__device__ __forceinline__ double clamp_pos(double a) { return __double2hiint(a) >= 0 ? a : 0.0; }
// f(q) and f'(q) of kernel K. M5 and M6 in clamped-power form: f = sum_i c_i (a_i - q)_+^p
template <int K>
__device__ __forceinline__ void kern_f_df(double q, double& f, double& df) {
    if (K == 0) {
        m4(q, f, df);
    } else if (K == 1) {
        const double a = 2.5 - q, b = 1.5 - q, c = 0.5 - q;
        const double t1 = clamp_pos(a), t2 = clamp_pos(b), t3 = clamp_pos(c);
        const double c1 = t1 * t1 * t1, c2 = t2 * t2 * t2, c3 = t3 * t3 * t3;
        f = fma(10.0 * c3, t3, fma(-5.0 * c2, t2, c1 * t1));
        df = -4.0 * fma(10.0, c3, fma(-5.0, c2, c1));
    } else if (K >= 3) {
        // Wendland: q is clamped to the support radius (integer compare of the high word, q >= +0), so that t = 0
        // there and beyond and the polynomial factor cannot overflow for the density kernel's 1e100 padding entries;
        // f' in factored form
        const double qc = (__double2hiint(q) < 0x40000000) ? q : 2.0;
        const double t = fma(-0.5, qc, 1.0), t2 = t * t;
        if (K == 3) {
            const double t3 = t2 * t;
            f = t3 * t * fma(2.0, qc, 1.0);
            df = -5.0 * qc * t3;
        } else if (K == 4) {
            const double t5 = t2 * t2 * t;
            f = t5 * t * fma(qc, fma(35.0 / 12.0, qc, 3.0), 1.0);
            df = (-7.0 / 3.0) * qc * t5 * fma(5.0, qc, 2.0);
        } else {
            const double t4 = t2 * t2, t7 = t4 * t2 * t;
            f = t7 * t * fma(qc, fma(qc, fma(4.0, qc, 6.25), 4.0), 1.0);
            df = -2.75 * qc * t7 * fma(qc, fma(8.0, qc, 7.0), 2.0);
        }
    } else {
        const double a = 3.0 - q, b = 2.0 - q, c = 1.0 - q;
        const double t1 = clamp_pos(a), t2 = clamp_pos(b), t3 = clamp_pos(c);
        const double s1 = t1 * t1, s2 = t2 * t2, s3 = t3 * t3;
        const double q1 = s1 * s1, q2 = s2 * s2, q3 = s3 * s3;
        f = fma(15.0 * q3, t3, fma(-6.0 * q2, t2, q1 * t1));
        df = -5.0 * fma(15.0, q3, fma(-6.0, q2, q1));
    }
}
__device__ __forceinline__ void m4(double q, double& f, double& df) {
    double t2 = 2.0 - q;
    double fo = 0.25 * t2 * t2 * t2;          // outer branch 1 <= q < 2
    double dfo = -0.75 * t2 * t2;
    double fi = 1.0 + q * q * (0.75 * q - 1.5);   // inner branch q < 1
    double dfi = q * (2.25 * q - 3.0);
    // q >= +0: doubles order as their bit patterns, so the two range tests are integer compares of the high word
    // (exactly q < 1, q < 2) and stay off the FP64 pipe
    const int qh = __double2hiint(q);
    bool in = qh < 0x3FF00000, sup = qh < 0x40000000;
    f = in ? fi : (sup ? fo : 0.0);
    df = in ? dfi : (sup ? dfo : 0.0);
}
#endif

}  // namespace sph
