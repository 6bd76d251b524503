// api.cu -- the C ABI of include/sph_b200.h: context, memory, call-order state machine, step orchestration,
// getters/setters and per-stage CUDA-event timers. All arithmetic of the hot path lives in the kernels of the
// sibling .cu files; there is no CPU fallback anywhere in this library.
#include <math.h>
#include <stdarg.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "common.cuh"

using namespace sph;

namespace sph {

int fail(sph_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

static void* default_alloc(size_t bytes, void*) {
    void* p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
}
static void default_free(void* p, void*) { cudaFree(p); }

template <typename T>
static int dalloc(sph_ctx* c, T** out, size_t count) {
    size_t bytes = std::max<size_t>(count * sizeof(T), 256);
    void* p = c->alloc.alloc(bytes, c->alloc.user);
    if (!p) return fail(c, SPH_ERR_OOM, "device allocation of %zu bytes failed", bytes);
    c->allocations.emplace_back(p, bytes);
    c->bytes_allocated += (int64_t)bytes;
    *out = reinterpret_cast<T*>(p);
    return SPH_OK;
}
static void dfree(sph_ctx* c, void* p) {
    if (!p) return;
    auto it = std::find_if(c->allocations.begin(), c->allocations.end(), [p](const std::pair<void*, size_t>& a) { return a.first == p; });
    if (it != c->allocations.end()) { c->bytes_allocated -= (int64_t)it->second; c->allocations.erase(it); }
    c->alloc.release(p, c->alloc.user);
}

static int alloc_fields(sph_ctx* c, Fields& f) {
    const size_t N = (size_t)c->N;
    double *pos, *vel, *acc;
    SPH_TRY(dalloc(c, &pos, 3 * N));   // x|y|z contiguous so that 3-component copies are one kernel
    SPH_TRY(dalloc(c, &vel, 3 * N));
    SPH_TRY(dalloc(c, &acc, 3 * N));
    f.x = pos; f.y = pos + N; f.z = pos + 2 * N;
    f.vx = vel; f.vy = vel + N; f.vz = vel + 2 * N;
    f.ax = acc; f.ay = acc + N; f.az = acc + 2 * N;
    SPH_TRY(dalloc(c, &f.u, N));
    SPH_TRY(dalloc(c, &f.du, N));
    SPH_TRY(dalloc(c, &f.h, N));
    SPH_TRY(dalloc(c, &f.m, N));
    SPH_TRY(dalloc(c, &f.id, N));
    return SPH_OK;
}

// ---- timers ----
struct StageTimer {
    sph_ctx* c;
    StageTimer(sph_ctx* ctx, int stage) : c(ctx) {
        TimerRec r;
        r.stage = stage;
        r.e0 = get(); r.e1 = get();
        cudaEventRecord(r.e0, c->stream);
        c->timers.push_back(r);
    }
    ~StageTimer() { cudaEventRecord(c->timers.back().e1, c->stream); }
    cudaEvent_t get() {
        if (!c->event_pool.empty()) { cudaEvent_t e = c->event_pool.back(); c->event_pool.pop_back(); return e; }
        cudaEvent_t e; cudaEventCreate(&e); return e;
    }
};

// after a stream synchronisation every recorded stage timer is complete: add it to the per-stage totals and hand its
// events back to the pool (a long run keeps a bounded number of events)
static void fold_timers(sph_ctx* c) {
    for (auto& t : c->timers) {
        float v = 0.f;
        if (cudaEventElapsedTime(&v, t.e0, t.e1) == cudaSuccess) c->ms_acc[t.stage] += v; else cudaGetLastError();
        c->event_pool.push_back(t.e0);
        c->event_pool.push_back(t.e1);
    }
    c->timers.clear();
}

static int read_scalars(sph_ctx* c) {
    SPH_CUDA(c, cudaMemcpyAsync(c->h_sc, c->d_sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    fold_timers(c);
    return SPH_OK;
}

// Every ABI entry makes the context's device current for its duration (function attributes, launches and events are
// per device) and restores the caller's device on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const sph_ctx* c) {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

__global__ void k_iota(int64_t N, uint32_t* id) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) id[i] = (uint32_t)i;
}
__global__ void k_mass_uniform(int64_t N, const double* __restrict__ m, DevScalars* sc) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N && m[i] != m[0]) sc->mass_nonuniform = 1u;
}
__global__ void k_fill(int64_t N, double* p, double v) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) p[i] = v;
}
// fallback h0 = hfact (m V / M_tot)^(1/3) (reading A9); M_tot by a two-stage reduction in a fixed order (per-block
// partials over a fixed grid, then one block), so that the initial h is reproducible bit for bit
__global__ void __launch_bounds__(256) k_sum_partial(int64_t N, const double* __restrict__ m, double* __restrict__ part) {
    __shared__ double ws[8];
    double v = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) v += m[i];
    v = warp_sum(v);
    if (lane_id() == 0) ws[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = ws[0];
        for (int w = 1; w < 8; ++w) t += ws[w];
        part[blockIdx.x] = t;
    }
}
__global__ void k_sum_final(int nblocks, const double* __restrict__ part, double* out) {
    double t = 0.0;
    for (int b = 0; b < nblocks; ++b) t += part[b];
    *out = t;
}
__global__ void k_h0_fallback(int64_t N, const double* __restrict__ m, const double* mtot, double vol, double hfact, double* h) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) h[i] = hfact * cbrt(m[i] * vol / *mtot);
}

// (re)allocate one pool of the neighbour cache
template <typename T>
static int grow_pool(sph_ctx* c, T** pool, uint64_t* cap, uint64_t want) {
    if (*pool) dfree(c, *pool);
    *pool = nullptr;
    *cap = 0;
    // slack behind the capacity: k_forces prefetches list entries unconditionally while ANY octet of its warp has entries
    // left, so a lane with a short list reads up to (longest list of the warp + 15) entries past its own list's start;
    // a list holds at most 65535 entries (16-bit candidate indices), which bounds the overrun behind the last list
    SPH_TRY(dalloc(c, pool, (size_t)want + 65536 + 64));
    *cap = want;
    return SPH_OK;
}

// neighbour cache for the current tree and h^n: hmax -> AABB -> single traversal pass (count, allocate, fill per
// group from bump allocators). The pass is repeated with larger pools if one of them overflowed (first build,
// or a cache that grew by more than the slack since the previous step).
constexpr int kSortRedo = 1;   // cache_build: the prefix-mode sort gave up on a long run; sort again in full

static int cache_build(sph_ctx* c) {
    { StageTimer t(c, ST_AABB); SPH_TRY(launch_hmax(c)); SPH_TRY(launch_aabb(c)); }
    for (int attempt = 0;; ++attempt) {
        { StageTimer t(c, ST_TRAVERSE); SPH_TRY(launch_traverse(c)); }
        SPH_TRY(read_scalars(c));
        const DevScalars& s = *c->h_sc;
        if (s.sort_redo) { c->sort_p0 = 0; return kSortRedo; }
        for (int k = 0; k < 3; ++k)
            if (c->box.periodic[k] && !(2.0 * kern_radius(c->p.kernel) * c->p.chi * s.h_max < c->box.hi[k] - c->box.lo[k]))
                return fail(c, SPH_ERR_PERIODIC_TOO_SMALL, "periodic axis %d: 2 R_kern chi h_max = %g >= L = %g", k,
                            2.0 * kern_radius(c->p.kernel) * c->p.chi * s.h_max, c->box.hi[k] - c->box.lo[k]);
        if (s.n_cand_overflow)
            return fail(c, SPH_ERR_CAP, "%u leaf groups have more than 65535 candidates (16-bit local index)",
                        s.n_cand_overflow);
        if (getenv("SPH_DEBUG"))
            fprintf(stderr, "[sph] groups %u nc_max %u fallback %u nbr_min %u nbr_max %u lists %llu candidates %llu chunk %u shared %u overflow %u\n",
                    s.n_groups, s.nc_max, s.n_fallback, s.nbr_min, s.nbr_max, s.list_cursor, s.cslot_cursor, c->last_chunk,
                    s.n_chunks_shared, s.n_chunks_overflow);
        // next sort: prefix mode if ties stay short -- four passes (top 32 bits) if the runs of equal 32-bit prefixes are
        // short, else five (top 40 bits) if those are; a four-pass sort has no 40-bit census: it is followed by a
        // five-pass one when its own runs got long (the repair kernel's bound and the redo path guard that sort too)
        if (getenv("SPH_FULL_SORT")) c->sort_p0 = 0;
        else if (s.tie_max32 <= 64u) c->sort_p0 = 4;
        else if (c->last_sort_passes == 4 || s.tie_max <= 64u) c->sort_p0 = 3;
        else c->sort_p0 = 0;
        if (c->last_chunk > 1) {
            const uint64_t chunks = ((uint64_t)s.n_groups + c->last_chunk - 1) / c->last_chunk;
            if ((uint64_t)s.n_chunks_shared * 10 < chunks * 8 || (uint64_t)s.n_chunks_overflow * 50 > chunks)
                c->share_disabled = true;
        }
        c->n_groups = s.n_groups;
        c->nc_max = s.nc_max;
        c->n_neigh = s.n_neigh;
        bool redo = false;
        if (s.list_cursor > c->list_cap) {
            SPH_TRY(grow_pool(c, &c->lists, &c->list_cap, s.list_cursor + s.list_cursor / 8 + 4096));
            redo = true;
        }
        if (s.cslot_cursor > c->cslot_cap) {
            SPH_TRY(grow_pool(c, &c->cslot, &c->cslot_cap, s.cslot_cursor + s.cslot_cursor / 8 + 4096));
            redo = true;
        }
        if ((uint64_t)s.n_groups > c->ginfo_cap) {
            SPH_TRY(grow_pool(c, &c->ginfo, &c->ginfo_cap, (uint64_t)s.n_groups + s.n_groups / 8 + 64));
            redo = true;
        }
        if (!redo) break;
        if (attempt >= 2) return fail(c, SPH_ERR_DEVICE, "neighbour cache pools did not converge");
    }
    return SPH_OK;
}

static int check_ctx(sph_ctx* c) { return c ? SPH_OK : SPH_ERR_ARG; }

}  // namespace sph

extern "C" {

void sph_default_params(sph_params* p) {
    if (!p) return;
    memset(p, 0, sizeof(*p));
    p->hfact = 1.2; p->gamma = 5.0 / 3.0; p->chi = 1.1; p->lambda = 1.2; p->eps_h = 1e-6;
    p->alpha_av = 1.0; p->beta_av = 2.0; p->beta_u = 1.0; p->c_cour = 0.3; p->c_force = 0.25;
    p->max_h_iter = 50; p->max_restarts = 50; p->eos = 0; p->kernel = 0;
    p->cs0 = 1.0; p->r0 = 1.0; p->q = 0.0; p->GM = 0.0; p->soft = 0.0;
    p->eps_v = 0.0; p->lambda_stiff = 2.0; p->max_recycle = 10; p->group_max = kGroup; p->morton_bits = 21;
    p->av_switch = 0; p->alpha_min = 0.0; p->alpha_max = 1.0; p->sigma_decay = 0.1;
}

const char* sph_last_error(const sph_ctx* c) { return c ? c->err : "null context"; }

void sph_free(sph_ctx* c) {
    if (!c) return;
    DeviceGuard dg(c);
    cudaStreamSynchronize(c->stream);
    for (auto& t : c->timers) { cudaEventDestroy(t.e0); cudaEventDestroy(t.e1); }
    for (auto e : c->event_pool) cudaEventDestroy(e);
    for (auto& a : c->allocations) c->alloc.release(a.first, c->alloc.user);
    c->allocations.clear();
    if (c->h_sc) cudaFreeHost(c->h_sc);
    delete c;
}

int sph_init_ex(sph_ctx** out, int64_t N, sph_mem mem, const double* pos, const double* vel, const double* mass,
                const double* u, const double* h0, const sph_box* box, const sph_params* params, void* cuda_stream,
                const sph_allocator* allocator, int run_white_step) {
    if (!out) return SPH_ERR_ARG;
    *out = nullptr;
    if (N < 1 || N >= (1ll << 30) || !pos || !vel || !mass || !u || !box) return SPH_ERR_ARG;
    for (int k = 0; k < 3; ++k)
        if (!(box->hi[k] > box->lo[k])) return SPH_ERR_ARG;
    int dev = 0, count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count < 1) { cudaGetLastError(); return SPH_ERR_DEVICE; }
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return SPH_ERR_DEVICE;
    if (prop.major != 10) return SPH_ERR_DEVICE;   // sm_100a code only; no fallback path exists

    sph_ctx* c = new (std::nothrow) sph_ctx();
    if (!c) return SPH_ERR_OOM;
    *out = c;   // returned even on failure so that sph_last_error() can be read; caller frees it
    c->N = N;
    c->device = dev;
    c->box = *box;
    if (params) c->p = *params; else sph_default_params(&c->p);
    if (c->p.kernel < 0 || c->p.kernel >= kNumKernels) return fail(c, SPH_ERR_ARG, "kernel must be 0 (M4), 1 (M5), 2 (M6), 3 (Wendland C2), 4 (C4) or 5 (C6)");
    if (c->p.group_max == 0) c->p.group_max = kGroup;
    if (c->p.morton_bits == 0) c->p.morton_bits = 21;
    if (c->p.morton_bits != 21 && c->p.morton_bits != 10) return fail(c, SPH_ERR_ARG, "morton_bits must be 21 or 10 (0 = default 21)");
    if (c->p.group_max < 1 || c->p.group_max > kGroup) return fail(c, SPH_ERR_ARG, "group_max must be in 1..32 (0 = default 32)");
    if (c->p.leaf_reduction < 0 || c->p.leaf_reduction > 64) return fail(c, SPH_ERR_ARG, "leaf_reduction must be in 0..64");
    if (!(c->p.hfact > 0) || !(c->p.chi >= 1.0) || !(c->p.lambda > 1.0) || !(c->p.eps_h > 0) || c->p.max_h_iter < 1)
        return fail(c, SPH_ERR_ARG, "bad parameters");
    c->stream = (cudaStream_t)cuda_stream;
    if (allocator && allocator->alloc && allocator->release) c->alloc = *allocator;
    else { c->alloc.alloc = default_alloc; c->alloc.release = default_free; c->alloc.user = nullptr; }

    const size_t n = (size_t)N;
    SPH_TRY(alloc_fields(c, c->cur));
    SPH_TRY(alloc_fields(c, c->alt));
    SPH_TRY(dalloc(c, &c->rho, n)); SPH_TRY(dalloc(c, &c->omega, n)); SPH_TRY(dalloc(c, &c->P, n));
    SPH_TRY(dalloc(c, &c->cs, n)); SPH_TRY(dalloc(c, &c->A, n)); SPH_TRY(dalloc(c, &c->hnew, n));
    SPH_TRY(dalloc(c, &c->nax, 3 * n));
    c->nay = c->nax + n; c->naz = c->nax + 2 * n;
    SPH_TRY(dalloc(c, &c->ndu, n));
    SPH_TRY(dalloc(c, &c->key, n)); SPH_TRY(dalloc(c, &c->key_alt, n));
    SPH_TRY(dalloc(c, &c->val, n)); SPH_TRY(dalloc(c, &c->val_alt, n));
    size_t status_bytes;
    sort_scratch_bytes(N, &c->sort_tiles, &status_bytes);
    SPH_TRY(dalloc(c, &c->sort_hist, 8 * 256));
    SPH_TRY(dalloc(c, &c->sort_status, status_bytes / sizeof(uint32_t)));
    SPH_TRY(dalloc(c, &c->sort_counters, 16));
    SPH_TRY(dalloc(c, &c->nodes, n));
    SPH_TRY(dalloc(c, &c->parent, 2 * n));
    SPH_TRY(dalloc(c, &c->visit, n));
    SPH_TRY(dalloc(c, &c->gflag, n)); SPH_TRY(dalloc(c, &c->gscan, n + 1)); SPH_TRY(dalloc(c, &c->grp_lo, n + 1));
    if (c->p.av_switch) {
        if (!(c->p.alpha_max >= c->p.alpha_min) || !(c->p.alpha_min >= 0.0) || !(c->p.sigma_decay >= 0.0))
            return fail(c, SPH_ERR_ARG, "shock switch needs 0 <= alpha_min <= alpha_max and sigma_decay >= 0");
        SPH_TRY(dalloc(c, &c->alpha, n)); SPH_TRY(dalloc(c, &c->alpha_alt, n)); SPH_TRY(dalloc(c, &c->acs, n));
    }
    if (c->p.leaf_reduction >= 1) { SPH_TRY(dalloc(c, &c->xi_a, n)); SPH_TRY(dalloc(c, &c->xi_b, n)); SPH_TRY(dalloc(c, &c->lscan, n + 1)); }
    SPH_TRY(dalloc(c, &c->cnt, n + 1)); SPH_TRY(dalloc(c, &c->cnt_in, n + 1)); SPH_TRY(dalloc(c, &c->grow, n + 1)); SPH_TRY(dalloc(c, &c->lstart, n)); SPH_TRY(dalloc(c, &c->offs, n + 1));
    SPH_TRY(dalloc(c, &c->trav_scratch, trav_scratch_entries()));
    SPH_TRY(dalloc(c, &c->trav_hit_scratch, trav_hit_scratch_entries()));
    SPH_TRY(dalloc(c, &c->corr_part, 2 * (size_t)div_up(N, 256) + 2));
    // cache pools start empty: the first traversal only counts, then they are sized from its totals
    c->scan_tiles = scan_scratch_tiles(N);
    SPH_TRY(dalloc(c, &c->scan_status, (size_t)c->scan_tiles));
    SPH_TRY(dalloc(c, &c->scan_counter, 4));
    SPH_TRY(dalloc(c, &c->d_sc, 1));
    SPH_TRY(dalloc(c, &c->d_dtstep, 4));
    SPH_CUDA(c, cudaMallocHost((void**)&c->h_sc, sizeof(DevScalars)));
    SPH_CUDA(c, cudaMemsetAsync(c->d_sc, 0, sizeof(DevScalars), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(c->d_dtstep, 0, 4 * sizeof(double), c->stream));

    // inputs, original order: slot i holds particle i, id = iota
    const cudaMemcpyKind kind = (mem == SPH_MEM_HOST) ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    SPH_CUDA(c, cudaMemcpyAsync(c->cur.x, pos, 3 * n * sizeof(double), kind, c->stream));
    SPH_CUDA(c, cudaMemcpyAsync(c->cur.vx, vel, 3 * n * sizeof(double), kind, c->stream));
    SPH_CUDA(c, cudaMemcpyAsync(c->cur.m, mass, n * sizeof(double), kind, c->stream));
    SPH_CUDA(c, cudaMemcpyAsync(c->cur.u, u, n * sizeof(double), kind, c->stream));
    SPH_CUDA(c, cudaMemsetAsync(c->cur.ax, 0, 3 * n * sizeof(double), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(c->cur.du, 0, n * sizeof(double), c->stream));
    k_iota<<<div_up(N, 256), 256, 0, c->stream>>>(N, c->cur.id);
    c->launches++;
    if (h0) {
        SPH_CUDA(c, cudaMemcpyAsync(c->cur.h, h0, n * sizeof(double), kind, c->stream));
    } else {
        double vol = 1.0;
        for (int k = 0; k < 3; ++k) vol *= box->hi[k] - box->lo[k];
        double* mtot = c->d_dtstep + 1;
        const unsigned nb = (unsigned)std::min<int64_t>(592, (N + 255) / 256);   // corr_part holds >= 2 ceil(N / 256) doubles
        k_sum_partial<<<nb, 256, 0, c->stream>>>(N, c->cur.m, c->corr_part);
        k_sum_final<<<1, 1, 0, c->stream>>>((int)nb, c->corr_part, mtot);
        k_h0_fallback<<<div_up(N, 256), 256, 0, c->stream>>>(N, c->cur.m, mtot, vol, c->p.hfact, c->cur.h);
        c->launches += 3;
    }
    k_mass_uniform<<<div_up(N, 256), 256, 0, c->stream>>>(N, c->cur.m, c->d_sc);
    c->launches++;
    if (c->p.av_switch) {     // alpha starts at alpha_min; the white step's G13 (dt = 0) raises it to alpha_loc
        k_fill<<<div_up(N, 256), 256, 0, c->stream>>>(N, c->alpha, c->p.alpha_min);
        c->launches++;
    }
    SPH_CUDA(c, cudaGetLastError());
    SPH_TRY(read_scalars(c));
    c->uniform_mass = (c->h_sc->mass_nonuniform == 0u);
    c->state = S_FIELDS;
    if (run_white_step) {
        SPH_TRY(sph_build_tree(c));
        SPH_TRY(sph_compute_density(c));
        SPH_TRY(sph_compute_forces(c));
    }
    return SPH_OK;
}

int sph_init(sph_ctx** out, int64_t N, const double* pos_dev, const double* vel_dev, const double* mass_dev,
             const double* u_dev, const sph_box* box, double gamma, double hfact) {
    sph_params p;
    sph_default_params(&p);
    p.gamma = gamma;
    p.hfact = hfact;
    return sph_init_ex(out, N, SPH_MEM_DEVICE, pos_dev, vel_dev, mass_dev, u_dev, nullptr, box, &p, nullptr, nullptr, 1);
}

int sph_build_tree(sph_ctx* c) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    for (int attempt = 0;; ++attempt) {
        { StageTimer t(c, ST_KEYS); SPH_TRY(launch_keys(c)); }
        { StageTimer t(c, ST_SORT); SPH_TRY(launch_sort(c)); }
        { StageTimer t(c, ST_PERMUTE); SPH_TRY(launch_permute(c)); }
        { StageTimer t(c, ST_TREE); SPH_TRY(launch_tree(c)); }
        const int rc = cache_build(c);
        if (rc == SPH_OK) break;
        // the prefix-mode sort met a run too long to repair (the tree kernels then did nothing): the fields are a
        // valid permutation of the particles, so the build simply starts over with all eight radix passes
        if (rc != kSortRedo || attempt > 0) return rc == kSortRedo ? fail(c, SPH_ERR_DEVICE, "sort did not complete") : rc;
    }
    c->state = S_TREE;
    return SPH_OK;
}

int sph_compute_density(sph_ctx* c) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    if (c->state < S_TREE) return fail(c, SPH_ERR_ORDER, "sph_compute_density needs sph_build_tree first");
    int restarts = 0;
    for (;;) {
        { StageTimer t(c, ST_DENSITY); SPH_TRY(launch_density(c)); }
        SPH_TRY(read_scalars(c));
        if (c->h_sc->n_noconv)
            return fail(c, SPH_ERR_H_NOCONV, "%u particles did not converge in %d Newton iterations", c->h_sc->n_noconv,
                        c->p.max_h_iter);
        std::swap(c->cur.h, c->hnew);            // h^n <- h (all particles), Alg. 7 outer loop
        if (c->h_sc->n_exceeded == 0) break;
        if (++restarts > c->p.max_restarts)
            return fail(c, SPH_ERR_RESTARTS, "more than %d chi-restarts (%u particles still exceed chi h^n)",
                        c->p.max_restarts, c->h_sc->n_exceeded);
        SPH_TRY(cache_build(c));                 // positions unchanged: same keys, order and topology; new hmax, cache
    }
    c->restarts_last = restarts;
    c->state = S_DENSITY;
    return SPH_OK;
}

static int forces_eval(sph_ctx* c) {
    if (c->state < S_DENSITY) return fail(c, SPH_ERR_ORDER, "sph_compute_forces needs sph_compute_density first");
    { StageTimer t(c, ST_FORCES); SPH_TRY(launch_forces(c)); }
    c->have_cfl_dt = true;
    c->state = S_FORCES;
    return SPH_OK;
}

int sph_compute_forces(sph_ctx* c) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    c->alpha_pending = true;      // standalone evaluation: G13 with dt = 0 and the stored a^n
    c->in_step = false;
    SPH_TRY(forces_eval(c));
    // standalone evaluation (and the white step): the result becomes a^n, du/dt^n of the next predictor
    StageTimer t(c, ST_LEAPFROG);
    return launch_adopt_acc(c);
}

int sph_step_leapfrog(sph_ctx* c, double dt, double* dt_used) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    if (!c->have_cfl_dt) return fail(c, SPH_ERR_ORDER, "sph_step_leapfrog needs a force evaluation (a^n, dt) first");
    {
        StageTimer t(c, ST_LEAPFROG);
        SPH_TRY(launch_set_dt(c, dt));
        SPH_TRY(launch_predict(c));
    }
    c->state = S_FIELDS;
    SPH_TRY(sph_build_tree(c));
    SPH_TRY(sph_compute_density(c));
    c->alpha_pending = true;      // G12-G13 once per step, before the derivatives; re-cycles keep alpha
    c->in_step = true;
    const int rc_f = forces_eval(c);
    c->in_step = false;
    SPH_TRY(rc_f);
    const bool check = c->p.eps_v > 0.0;
    { StageTimer t(c, ST_LEAPFROG); SPH_TRY(launch_correct(c, check)); }
    c->recycles_last = 0;
    if (check) {
        // G6-G7 with reading A15: err = max|dv| / rms|v^{n+1}|; while it is not below eps_v, recalculate the
        // acceleration with v* <- v^{n+1} (same positions, h, rho, Omega, cache) and apply the correction again
        for (;;) {
            SPH_TRY(read_scalars(c));
            const double vrms = sqrt(c->h_sc->corr_v2sum / (double)c->N);
            const double err = vrms > 0.0 ? sqrt(c->h_sc->corr_dvmax2) / vrms : 0.0;
            if (err < c->p.eps_v || c->recycles_last >= c->p.max_recycle) break;
            c->recycles_last++;
            SPH_TRY(forces_eval(c));
            { StageTimer t(c, ST_LEAPFROG); SPH_TRY(launch_correct(c, true)); }
        }
        // G9-G10: halve the multiplier after a step that re-cycled, relax it towards 1 otherwise
        c->cfl_mult = c->recycles_last > 0 ? 0.5 * c->cfl_mult
                                            : (1.0 + c->p.lambda_stiff * c->cfl_mult) / (1.0 + c->p.lambda_stiff);
    }
    c->steps++;
    if (dt_used) {
        SPH_CUDA(c, cudaMemcpyAsync(dt_used, c->d_dtstep, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    }
    return SPH_OK;
}

static int copy_in(sph_ctx* c, sph_mem mem, const double* src, double* dst_sorted, int ncomp, double** stage) {
    if (!src) return SPH_OK;
    const size_t bytes = (size_t)ncomp * c->N * sizeof(double);
    const double* dev_src = src;
    if (mem == SPH_MEM_HOST) {
        if (!*stage) SPH_TRY(dalloc(c, stage, 3 * (size_t)c->N));
        SPH_CUDA(c, cudaMemcpyAsync(*stage, src, bytes, cudaMemcpyHostToDevice, c->stream));
        dev_src = *stage;
    }
    return launch_gather_orig_f64(c, dev_src, dst_sorted, ncomp);
}
static int copy_out(sph_ctx* c, sph_mem mem, const double* src_sorted, double* dst, int ncomp, double** stage) {
    if (!dst) return SPH_OK;
    const size_t bytes = (size_t)ncomp * c->N * sizeof(double);
    if (mem == SPH_MEM_HOST) {
        if (!*stage) SPH_TRY(dalloc(c, stage, 3 * (size_t)c->N));
        SPH_TRY(launch_scatter_orig_f64(c, src_sorted, *stage, ncomp));
        SPH_CUDA(c, cudaMemcpyAsync(dst, *stage, bytes, cudaMemcpyDeviceToHost, c->stream));
        return SPH_OK;
    }
    return launch_scatter_orig_f64(c, src_sorted, dst, ncomp);
}

int sph_set_fields(sph_ctx* c, sph_mem mem, const double* pos, const double* vel, const double* u, const double* h,
                   const double* acc, const double* dudt) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    double* stage = nullptr;   // one staging buffer reused in stream order
    int rc = SPH_OK;
    if ((rc = copy_in(c, mem, pos, c->cur.x, 3, &stage)) == SPH_OK && (rc = copy_in(c, mem, vel, c->cur.vx, 3, &stage)) == SPH_OK &&
        (rc = copy_in(c, mem, u, c->cur.u, 1, &stage)) == SPH_OK && (rc = copy_in(c, mem, h, c->cur.h, 1, &stage)) == SPH_OK &&
        (rc = copy_in(c, mem, acc, c->cur.ax, 3, &stage)) == SPH_OK)
        rc = copy_in(c, mem, dudt, c->cur.du, 1, &stage);
    if (stage) { cudaStreamSynchronize(c->stream); dfree(c, stage); }
    if (rc != SPH_OK) return rc;
    if (pos || vel || u || h) c->state = S_FIELDS;
    if (pos) c->sort_p0 = 0;   // unrelated positions: the previous order says nothing about the next sort's ties
    return SPH_OK;
}

int sph_get_fields(sph_ctx* c, sph_mem mem, double* pos, double* vel, double* u, double* h, double* rho, double* omega,
                   double* acc, double* dudt) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    if ((rho || omega) && c->state < S_DENSITY) return fail(c, SPH_ERR_ORDER, "rho/omega need sph_compute_density");
    double* stage = nullptr;
    int rc = SPH_OK;
    // with a host destination each field goes through the staging buffer; the D2H copy is stream-ordered
    // after its scatter and before the next scatter overwrites the buffer
    if ((rc = copy_out(c, mem, c->cur.x, pos, 3, &stage)) == SPH_OK && (rc = copy_out(c, mem, c->cur.vx, vel, 3, &stage)) == SPH_OK &&
        (rc = copy_out(c, mem, c->cur.u, u, 1, &stage)) == SPH_OK && (rc = copy_out(c, mem, c->cur.h, h, 1, &stage)) == SPH_OK &&
        (rc = copy_out(c, mem, c->rho, rho, 1, &stage)) == SPH_OK && (rc = copy_out(c, mem, c->omega, omega, 1, &stage)) == SPH_OK &&
        (rc = copy_out(c, mem, c->cur.ax, acc, 3, &stage)) == SPH_OK)
        rc = copy_out(c, mem, c->cur.du, dudt, 1, &stage);
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (stage) dfree(c, stage);
    if (rc != SPH_OK) return rc;
    if (e != cudaSuccess) return fail(c, SPH_ERR_DEVICE, "stream sync failed: %s", cudaGetErrorString(e));
    return SPH_OK;
}

static int copy_raw(sph_ctx* c, sph_mem mem, void* dst, const void* src_dev, size_t bytes) {
    if (!dst || bytes == 0) return SPH_OK;
    SPH_CUDA(c, cudaMemcpyAsync(dst, src_dev, bytes, mem == SPH_MEM_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice,
                                c->stream));
    return SPH_OK;
}

int sph_get_keys_perm(sph_ctx* c, sph_mem mem, uint64_t* sorted_keys, uint32_t* perm) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    if (c->state < S_TREE) return fail(c, SPH_ERR_ORDER, "no tree built");
    SPH_TRY(copy_raw(c, mem, sorted_keys, c->key, (size_t)c->N * sizeof(uint64_t)));
    SPH_TRY(copy_raw(c, mem, perm, c->cur.id, (size_t)c->N * sizeof(uint32_t)));
    SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    return SPH_OK;
}

__global__ void k_export_tree(int64_t N, const NodeRec* __restrict__ nodes, int32_t* left, int32_t* right, uint8_t* lflag,
                              uint8_t* rflag, int32_t* rlo, int32_t* rhi, double* aabb, double* hmax) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N - 1) return;
    const NodeRec r = nodes[i];
    const int32_t lo = min((int32_t)i, r.other), hi = max((int32_t)i, r.other);
    if (left) left[i] = r.split;
    if (right) right[i] = r.split + 1;
    if (lflag) lflag[i] = (lo == r.split);
    if (rflag) rflag[i] = (hi == r.split + 1);
    if (rlo) rlo[i] = lo;
    if (rhi) rhi[i] = hi;
    if (aabb) for (int k = 0; k < 3; ++k) { aabb[6 * i + k] = r.lo[k]; aabb[6 * i + 3 + k] = r.hi[k]; }
    if (hmax) hmax[i] = r.hmax;
}

int sph_get_tree(sph_ctx* c, sph_mem mem, int32_t* left, int32_t* right, uint8_t* lflag, uint8_t* rflag, int32_t* parent,
                 int32_t* range_lo, int32_t* range_hi, double* aabb, double* hmax) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    if (c->state < S_TREE) return fail(c, SPH_ERR_ORDER, "no tree built");
    const int64_t N = c->N, ni = N - 1;
    if (parent) {
        if (N == 1) { int32_t m1 = -1; SPH_CUDA(c, cudaMemcpyAsync(c->parent, &m1, 4, cudaMemcpyHostToDevice, c->stream)); }
        SPH_TRY(copy_raw(c, mem, parent, c->parent, (size_t)(2 * N - 1) * sizeof(int32_t)));
    }
    if (ni < 1) { SPH_CUDA(c, cudaStreamSynchronize(c->stream)); return SPH_OK; }
    // export through device temporaries (debug path), then copy to the caller's memory
    int32_t *t_i = nullptr; uint8_t* t_b = nullptr; double* t_d = nullptr;
    SPH_TRY(dalloc(c, &t_i, 4 * (size_t)ni));
    SPH_TRY(dalloc(c, &t_b, 2 * (size_t)ni));
    SPH_TRY(dalloc(c, &t_d, 7 * (size_t)ni));
    k_export_tree<<<div_up(ni, 256), 256, 0, c->stream>>>(N, c->nodes, t_i, t_i + ni, t_b, t_b + ni, t_i + 2 * ni, t_i + 3 * ni,
                                                          t_d, t_d + 6 * ni);
    c->launches++;
    int rc = SPH_OK;
    if ((rc = copy_raw(c, mem, left, t_i, ni * 4)) == SPH_OK && (rc = copy_raw(c, mem, right, t_i + ni, ni * 4)) == SPH_OK &&
        (rc = copy_raw(c, mem, lflag, t_b, ni)) == SPH_OK && (rc = copy_raw(c, mem, rflag, t_b + ni, ni)) == SPH_OK &&
        (rc = copy_raw(c, mem, range_lo, t_i + 2 * ni, ni * 4)) == SPH_OK &&
        (rc = copy_raw(c, mem, range_hi, t_i + 3 * ni, ni * 4)) == SPH_OK && (rc = copy_raw(c, mem, aabb, t_d, 6 * ni * 8)) == SPH_OK)
        rc = copy_raw(c, mem, hmax, t_d + 6 * ni, ni * 8);
    cudaStreamSynchronize(c->stream);
    dfree(c, t_i); dfree(c, t_b); dfree(c, t_d);
    return rc;
}

int sph_get_neighbours_range(sph_ctx* c, sph_mem mem, int64_t first, int64_t count, uint64_t* offs, uint32_t* idx, uint64_t cap) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    if (c->state < S_TREE) return fail(c, SPH_ERR_ORDER, "no neighbour cache built");
    if (first < 0 || count < 1 || first + count > c->N) return fail(c, SPH_ERR_ARG, "slot range [%lld, %lld) outside [0, N)", (long long)first, (long long)(first + count));
    // the cache is group-local (candidate arrays + 16-bit lists); convert to a CSR over sorted slots on request
    SPH_TRY(launch_scan_u32_u64(c, c->cnt, c->offs, c->N, nullptr));
    uint64_t ends[2] = {0, 0};
    SPH_CUDA(c, cudaMemcpyAsync(&ends[0], c->offs + first, sizeof(uint64_t), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA(c, cudaMemcpyAsync(&ends[1], c->offs + first + count, sizeof(uint64_t), cudaMemcpyDeviceToHost, c->stream));
    SPH_TRY(copy_raw(c, mem, offs, c->offs + first, (size_t)(count + 1) * sizeof(uint64_t)));
    SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    if (idx) {
        const uint64_t total = ends[1] - ends[0];
        if (cap < total) return fail(c, SPH_ERR_CAP, "idx capacity %llu < %llu neighbours", (unsigned long long)cap,
                                     (unsigned long long)total);
        uint32_t* tmp = nullptr;
        uint32_t* dst = idx;
        if (mem == SPH_MEM_HOST) { SPH_TRY(dalloc(c, &tmp, (size_t)total + 1)); dst = tmp; }
        int rc = launch_cache_to_csr(c, dst, first, count);
        if (rc == SPH_OK && tmp) rc = copy_raw(c, mem, idx, tmp, (size_t)total * sizeof(uint32_t));
        cudaStreamSynchronize(c->stream);
        if (tmp) dfree(c, tmp);
        if (rc != SPH_OK) return rc;
    }
    SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    return SPH_OK;
}

int sph_get_neighbours(sph_ctx* c, sph_mem mem, uint64_t* offs, uint32_t* idx, uint64_t cap) {
    SPH_TRY(check_ctx(c));
    return sph_get_neighbours_range(c, mem, 0, c->N, offs, idx, cap);
}

int sph_get_alpha(sph_ctx* c, sph_mem mem, double* alpha) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    if (!c->p.av_switch) return fail(c, SPH_ERR_ORDER, "sph_get_alpha needs sph_params.av_switch = 1");
    if (!alpha) return SPH_ERR_ARG;
    double* stage = nullptr;
    int rc = copy_out(c, mem, c->alpha, alpha, 1, &stage);
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (stage) dfree(c, stage);
    if (rc != SPH_OK) return rc;
    if (e != cudaSuccess) return fail(c, SPH_ERR_DEVICE, "stream sync failed: %s", cudaGetErrorString(e));
    return SPH_OK;
}

int sph_get_leaves(sph_ctx* c, sph_mem mem, int64_t* n_leaves, uint64_t* leaf_codes, uint32_t* id_map) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    if (c->p.leaf_reduction < 1) return fail(c, SPH_ERR_ORDER, "sph_get_leaves needs sph_params.leaf_reduction >= 1");
    if (c->state < S_TREE) return fail(c, SPH_ERR_ORDER, "no tree built");
    const int64_t N = c->N;
    uint32_t nl = 0;
    SPH_CUDA(c, cudaMemcpyAsync(&nl, c->lscan + N, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    uint64_t* t_codes = nullptr;
    uint32_t* t_ids = nullptr;
    uint64_t* codes = leaf_codes;
    uint32_t* ids = id_map;
    if (mem == SPH_MEM_HOST) {
        if (leaf_codes) { SPH_TRY(dalloc(c, &t_codes, (size_t)N)); codes = t_codes; }
        if (id_map) { SPH_TRY(dalloc(c, &t_ids, (size_t)N + 1)); ids = t_ids; }
    }
    int rc = launch_leaf_export(c, codes, ids);
    cudaStreamSynchronize(c->stream);
    if (rc == SPH_OK && t_codes) rc = copy_raw(c, mem, leaf_codes, t_codes, (size_t)nl * sizeof(uint64_t));
    if (rc == SPH_OK && t_ids) rc = copy_raw(c, mem, id_map, t_ids, ((size_t)nl + 1) * sizeof(uint32_t));
    cudaStreamSynchronize(c->stream);
    if (t_codes) dfree(c, t_codes);
    if (t_ids) dfree(c, t_ids);
    if (n_leaves) *n_leaves = (int64_t)nl;
    return rc;
}

int sph_reset_timers(sph_ctx* c) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    fold_timers(c);
    for (int k = 0; k < ST_COUNT; ++k) c->ms_acc[k] = 0.0;
    c->launches = 0;
    return SPH_OK;
}

int sph_get_stats(sph_ctx* c, sph_stats* out) {
    SPH_TRY(check_ctx(c));
    DeviceGuard dg(c);
    if (!out) return SPH_ERR_ARG;
    memset(out, 0, sizeof(*out));
    SPH_TRY(read_scalars(c));
    const double* ms = c->ms_acc;               // read_scalars synchronised and folded every open timer
    out->ms_keys = ms[ST_KEYS]; out->ms_sort = ms[ST_SORT]; out->ms_permute = ms[ST_PERMUTE]; out->ms_tree = ms[ST_TREE];
    out->ms_aabb = ms[ST_AABB]; out->ms_traverse = ms[ST_TRAVERSE]; out->ms_scan = ms[ST_SCAN];
    out->ms_density = ms[ST_DENSITY]; out->ms_forces = ms[ST_FORCES]; out->ms_leapfrog = ms[ST_LEAPFROG];
    for (int k = 0; k < ST_COUNT; ++k) out->ms_total += ms[k];
    const DevScalars& s = *c->h_sc;
    out->n_particles = c->N; out->n_groups = c->n_groups; out->n_neighbours = (int64_t)c->n_neigh;
    out->nbr_min = (int32_t)s.nbr_min; out->nbr_max = (int32_t)s.nbr_max;
    out->nbr_mean = c->N ? (double)c->n_neigh / (double)c->N : 0.0;
    out->h_iter_max = (int32_t)s.h_iter_max; out->restarts = c->restarts_last; out->steps = c->steps;
    out->kernel_launches = c->launches; out->dt = c->cfl_mult * s.dt; out->t = s.t; out->bytes_allocated = c->bytes_allocated;
    out->cand_max = (int32_t)s.nc_max; out->groups_fallback = (int32_t)s.n_fallback;
    out->chunks_shared = (int32_t)s.n_chunks_shared; out->share_chunk = (int32_t)c->last_chunk;
    out->sort_passes = c->last_sort_passes;
    out->sort_tie_max = (int32_t)(c->last_sort_passes == 4 ? s.tie_max32 : s.tie_max);
    out->recycles = c->recycles_last; out->cfl_mult = c->cfl_mult; out->density_sweeps = (int64_t)s.sweeps; out->n_inner = (int64_t)s.n_inner; out->n_grew = (int64_t)s.n_grew;
    return SPH_OK;
}

// ---- FP64 peak microbenchmark: 8 independent DFMA chains per thread ----
__global__ void __launch_bounds__(256) k_dfma(double* out, int iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    double s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == 123.456) out[0] = s;
}

int sph_measure_fp64_peak(double* tflops_out, void* cuda_stream) {
    if (!tflops_out) return SPH_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* d = nullptr;
    if (cudaMalloc(&d, 256) != cudaSuccess) return SPH_ERR_DEVICE;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = 148 * 8, iters = 1 << 15;
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, st);
        k_dfma<<<blocks, 256, 0, st>>>(d, iters, 0.999999, 1e-9);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return SPH_ERR_DEVICE; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double tf = 2.0 * 8.0 * (double)iters * blocks * 256 / (ms * 1e-3) * 1e-12;
        if (rep > 0) best = std::max(best, tf);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    *tflops_out = best;
    return SPH_OK;
}

}  // extern "C"
