/* sph_b200.h -- C ABI of libsph_b200: the single-GPU, per-timestep SPH hot path of arXiv:2503.09713
 * ("The SHAMROCK code: I - SPH on GPUs"; citations are lines of /root/reference/PAPER.md) as hand-written CUDA
 * for sm_100a (NVIDIA B200).
 *
 *   Morton keys -> onesweep radix sort + field permute -> Karras radix tree + bottom-up AABB/max-h ->
 *   warp-cooperative traversal writing a neighbour cache (count, scan, fill) -> Newton-Raphson h/density
 *   iteration with grad-h Omega -> symmetric grad-h force + artificial viscosity + CFL reduction ->
 *   leapfrog KDK with a global timestep.
 *
 * Conventions
 *   - Every function returns SPH_OK (0) or a negative sph_status; no exception crosses the ABI;
 *     sph_last_error() gives text for the last failure on that context.
 *   - There is no CPU fallback: without an sm_100 device sph_init* returns SPH_ERR_DEVICE.
 *   - Vector fields are SoA: pos = x[0..N) y[0..N) z[0..N) (3N contiguous doubles); same for vel, acc.
 *   - Pointers named *_dev are device pointers; getters/setters take a sph_mem flag saying whether the caller's
 *     buffers live on the host or on the device. The caller owns every buffer it passes; inputs are copied.
 *   - All work is enqueued on the CUDA stream given at init. Calls that must read a device scalar (neighbour
 *     total, chi-restart flag, optional dt_used) synchronise that stream; the others are asynchronous.
 *   - Particle order: callers always see ORIGINAL order (the order given to sph_init). Internally fields live
 *     in Morton-sorted order and an id array is carried through every sort; sph_get_keys_perm / sph_get_tree /
 *     sph_get_neighbours expose the sorted-order structures for parity checks.
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sph_ctx sph_ctx; /* opaque; owns all device state */

typedef enum {
  SPH_OK = 0,
  SPH_ERR_ARG = -1,                /* null pointer, N < 1, N >= 2^30, bad box, bad parameter            */
  SPH_ERR_DEVICE = -2,             /* no CUDA device of compute capability 10.x, or a CUDA call failed   */
  SPH_ERR_OOM = -3,                /* device allocation failed                                           */
  SPH_ERR_H_NOCONV = -4,           /* a particle did not converge within max_h_iter Newton iterations    */
  SPH_ERR_RESTARTS = -5,           /* more than max_restarts chi-restarts in one density solve           */
  SPH_ERR_PERIODIC_TOO_SMALL = -6, /* minimum image needs 2 R_kern chi h_max < L on every periodic axis  */
  SPH_ERR_ORDER = -7,              /* call sequence violated (e.g. forces before density)                */
  SPH_ERR_CAP = -8                 /* caller buffer too small (sph_get_neighbours)                       */
} sph_status;

typedef enum { SPH_MEM_HOST = 0, SPH_MEM_DEVICE = 1 } sph_mem;

/* Simulation box. Periodic axes wrap positions into [lo,hi) and use the minimum-image separation
 * (reading A4). The Morton grid is the cube of side max_k(hi_k - lo_k) anchored at lo (reading A1,
 * PAPER.md:582, 827); positions outside it clamp to the edge cells. */
typedef struct {
  double lo[3], hi[3];
  int32_t periodic[3];
} sph_box;

/* Parameters (defaults from sph_default_params; citation for each value). */
typedef struct {
  double hfact;    /* 1.2    h = hfact (m/rho)^(1/3), PAPER.md:1235-1237 (F1)                              */
  double gamma;    /* 5/3    adiabatic index, P = (gamma-1) rho u                            */
  double chi;      /* 1.1    tolerance on h growth / cache radius, PAPER.md:1245 (reading A2)               */
  double lambda;   /* 1.2    Newton step clamp, Alg. 7 l.11-13                               */
  double eps_h;    /* 1e-6   convergence |dh|/h^n, Alg. 7 l.5, 14 (value from north_star, reading A6)       */
  double alpha_av; /* 1.0    constant alpha^AV in Eq. 6, PAPER.md:56 (reading A10)                          */
  double beta_av;  /* 2.0    beta in Eq. 6                                                    */
  double beta_u;   /* 1.0    conductivity beta_u in Eq. 8; 0 disables                     */
  double c_cour;   /* 0.3                                                                  */
  double c_force;  /* 0.25                                                                  */
  int32_t max_h_iter;   /* 50  Newton iterations per particle per pass before SPH_ERR_H_NOCONV               */
  int32_t max_restarts; /* 50  chi-restarts per density solve before SPH_ERR_RESTARTS                        */
  int32_t eos;          /* 0 adiabatic; 1 locally isothermal c_s = cs0 (R/r0)^-q, du/dt = 0 (BASELINE cfg 3)  */
  int32_t kernel;       /* 0 M4 (default; all BASELINE configs), 1 M5, 2 M6, 3/4/5 Wendland C2/C4/C6 (O6) */
  double cs0, r0, q;    /* locally isothermal EOS; R = cylindrical radius about centre[]                     */
  double GM, soft;      /* fixed point mass a_ext = -GM d / (|d|^2 + soft^2)^(3/2); GM = 0 disables          */
  double centre[3];
  /* Leapfrog corrector check and re-cycle, G6-G7, and CFL multiplier, G9-G10
   * (PAPER.md:1337-1345); readings A15, A16. */
  double eps_v;         /* 0 (off; the paper uses 1e-2): after the corrector, while max|dv| / rms|v| >= eps_v the
                           acceleration is recalculated with v* <- v^{n+1} and the correction applied again   */
  double lambda_stiff;  /* 2.0  stiffness of the CFL multiplier relaxation (value not given in the paper)        */
  int32_t max_recycle;  /* 10   cap on re-cycles per step                                                        */
  int32_t group_max;    /* 32   particles per leaf group / traversal bucket, 1..32 (0 = 32): the paper's particles-per-
                           leaf knob of the leaf reduction (Fig. 16). Results do
                           not depend on it (the neighbour sets are exact for any grouping); the speed does           */
  int32_t morton_bits;  /* 21   grid bits per axis of the Morton code: 21 (63-bit codes) or 10, the paper's 32-bit variant
                           (SURVEY.md 8(f) item 4): the 30-bit code is kept in the top bits of the
                           64-bit key word (bits 62..33, the low 33 bits zero), sorted with four radix passes, ties
                           (particles of one 2^-10 cell) stay in their previous order; results do not depend on it   */
  int32_t leaf_reduction; /* 0  (off: leaf groups by the group_max rule). k >= 1: the paper's own leaf construction, Alg. 1
                           (PAPER.md:911-963): duplicate codes removed, then n_red = k - 1 reduction passes merge
                           sibling leaves; the leaf groups / traversal buckets are those reduced leaves (a leaf that
                           holds more than group_max particles is split by the group_max rule). The A/B variant of
                           SURVEY.md 8(f) item 1; results do not depend on it, the speed does (Fig. 16) */
  /* Shock switch (G11-G13; runscript values PAPER.md:1412-1415; reading A18 for
   * alpha_loc and tau, which the paper leaves to Price et al. 2018). */
  int32_t av_switch;    /* 0  (constant alpha_av, reading A10); 1: per-particle alpha_a, starting at alpha_min, updated by
                           the implicit step G13 between the smoothing-length update and the derivatives of every
                           evaluation (a standalone sph_compute_forces uses dt = 0 and the stored a^n)               */
  int32_t reserved4;
  double alpha_min;     /* 0.0 */
  double alpha_max;     /* 1.0 */
  double sigma_decay;   /* 0.1  PAPER.md:1412: tau = h / (sigma_decay c_s) */
} sph_params;

/* Device-memory hooks so that the host framework (PyTorch's caching allocator) owns device memory.
 * alloc returns a device pointer aligned to >= 256 B or NULL; release frees it. NULL hooks = cudaMalloc. */
typedef void* (*sph_alloc_fn)(size_t bytes, void* user);
typedef void (*sph_free_fn)(void* ptr, void* user);
typedef struct {
  sph_alloc_fn alloc;
  sph_free_fn release;
  void* user;
} sph_allocator;

/* Per-stage device time of the work since the last sph_reset_timers (CUDA events on the context's stream),
 * neighbour statistics of the current cache and iteration counts of the last density solve. */
typedef struct {
  double ms_keys, ms_sort, ms_permute, ms_tree, ms_aabb, ms_traverse, ms_scan, ms_density, ms_forces,
      ms_leapfrog, ms_total;
  int64_t n_particles, n_groups, n_neighbours;
  int32_t nbr_min, nbr_max;
  double nbr_mean;
  int32_t h_iter_max;    /* largest Newton iteration count of any particle in the last pass */
  int32_t restarts;      /* chi-restarts in the last density solve                           */
  int64_t steps;         /* leapfrog steps taken                                             */
  int64_t kernel_launches; /* CUDA kernels launched by this library since the last reset     */
  double dt;             /* current CFL timestep (G8)                                        */
  double t;              /* simulated time                                                   */
  int64_t bytes_allocated;
  /* neighbour-cache diagnostics of the last traversal pass */
  int32_t cand_max;        /* largest candidate array of any leaf group                                  */
  int32_t groups_fallback; /* groups that overflowed their buffers and were walked a second time          */
  int32_t chunks_shared;   /* chunks of consecutive groups that shared one tree walk (0: sharing off)     */
  int32_t share_chunk;     /* groups per chunk used by the last pass (1 or 4)                             */
  int32_t sort_passes;     /* radix passes of the last sort: 8, or 5 / 4 in prefix mode (top 40 / 32 bits + tie repair) */
  int32_t sort_tie_max;    /* longest run of keys equal in their top 40 bits (32 after a 4-pass sort) seen by the last sort */
  int32_t recycles;        /* corrector re-cycles of the last step (eps_v > 0)                              */
  int32_t reserved;
  double cfl_mult;         /* CFL multiplier lambda_CFL applied to the next internal dt                     */
  int64_t density_sweeps;  /* sweeps over the neighbour lists executed by the last density pass, summed over
                              particles: Newton sweeps + the closing pass at the converged h (Omega)         */
  int64_t n_inner;         /* entries of the cache's inner list segments (within R_kern 1.02 max(h_a, h_b) at build
                              time); the other n_neighbours - n_inner shell entries are skipped by density and forces
                              until some smoothing length has grown by 2 %                              */
  int64_t n_grew;          /* particles whose h grew past that bound in the last density pass                        */
} sph_stats;

void sph_default_params(sph_params* p);

/* sph_init: north_star's entry point. pos_dev/vel_dev (3N, SoA), mass_dev/u_dev (N) are DEVICE pointers.
 * Uses default parameters with the given gamma/hfact, the default (NULL) stream, cudaMalloc, and the
 * fallback initial smoothing length h0 = hfact (m V_box / M_tot)^(1/3) (reading A9). Then performs the
 * "white time step": build_tree -> compute_density -> compute_forces, so a^0 and dt^0 exist. */
int sph_init(sph_ctx** out, int64_t N, const double* pos_dev, const double* vel_dev, const double* mass_dev,
             const double* u_dev, const sph_box* box, double gamma, double hfact);

/* sph_init_ex: same with everything explicit. mem says where pos/vel/mass/u/h0 live. h0 (N) may be NULL.
 * params NULL = defaults. cuda_stream is a cudaStream_t (NULL = default stream). allocator may be NULL.
 * If run_white_step is 0 the caller drives sph_build_tree / sph_compute_density / sph_compute_forces.
 * The context lives on the CUDA device that is current at this call; every later call makes that device current
 * for its duration, so contexts on several devices may coexist in one process.
 * On failure: if the arguments themselves are invalid or no sm_100 device is present, *out is NULL; for any later
 * failure (allocation, a parameter out of range, an error of the white step) *out is a live context whose only
 * valid uses are sph_last_error() and sph_free(): the caller must free it. */
int sph_init_ex(sph_ctx** out, int64_t N, sph_mem mem, const double* pos, const double* vel, const double* mass,
                const double* u, const double* h0, const sph_box* box, const sph_params* params,
                void* cuda_stream, const sph_allocator* allocator, int run_white_step);

/* a1-a4: Morton keys -> stable LSD radix sort of (key, slot)
 * -> permute all fields into sorted order -> Karras radix tree (Table B2)
 * -> bottom-up AABB and max-h -> leaf groups (maximal nodes of <= 32 particles) -> traversal with
 * the group-group criterion and the object-object criterion with radius
 * R_kern chi max(h_a,h_b) -> neighbour cache (the count / prefix / fill of Alg. 5, done per leaf
 * group in one pass: hits are buffered on chip, counted, space is taken from a bump allocator, lists written).
 * The cache is group-local: per group the array of candidate slots, per particle a list of 16-bit indices into it,
 * inner entries first (d < R_kern 1.02 max(h_a, h_b) at build time), then the shell entries kept for the tolerance chi,
 * which density and forces skip until some h has grown by 2 % (exact); sph_get_neighbours converts to
 * a CSR over sorted slots. The pair test d^2 < (R_kern chi max(h_a, h_b))^2 is decided in packed fp32 wherever fp32 can
 * decide it and re-decided in IEEE fp64 otherwise, so the sets are those of the fp64 definition.
 * Synchronises the stream once (reads the totals; repeats the pass with larger pools if one overflowed). */
int sph_build_tree(sph_ctx* ctx);

/* a5: Alg. 7 per particle over the cache, with the safeguard of reading A5b; rho from F1
 * and Omega from Eq. 7 at the converged h. If any particle exceeds chi h^n, h^n <- h and the tree and cache are
 * rebuilt (outer loop of Alg. 7). Requires sph_build_tree. Synchronises once per pass. */
int sph_compute_density(sph_ctx* ctx);

/* a6: Eq. 3-6, 8-10 and the CFL timestep G8 reduced to a device scalar.
 * Requires sph_compute_density. Asynchronous. */
int sph_compute_forces(sph_ctx* ctx);

/* a7 + one full step: leapfrog KDK, G1-G5 in the order of Fig. G1:
 * predictor + periodic wrap -> sph_build_tree -> sph_compute_density -> sph_compute_forces -> corrector.
 * dt <= 0 uses the internal CFL dt from the previous force evaluation (reading A14), read on the device.
 * dt_used may be NULL (no extra synchronisation); otherwise receives the step actually taken. */
int sph_step_leapfrog(sph_ctx* ctx, double dt, double* dt_used);

/* Field access in ORIGINAL particle order; any pointer may be NULL (skipped). Setting pos/vel/u/h invalidates
 * the tree (state returns to "needs build_tree"); acc/dudt are a^n and du/dt^n used by the next predictor. */
int sph_set_fields(sph_ctx* ctx, sph_mem mem, const double* pos, const double* vel, const double* u,
                   const double* h, const double* acc, const double* dudt);
int sph_get_fields(sph_ctx* ctx, sph_mem mem, double* pos, double* vel, double* u, double* h, double* rho,
                   double* omega, double* acc, double* dudt);

/* Parity/debug getters, SORTED order, caller buffers per mem.
 * perm[i] = original id of the particle in sorted slot i. */
int sph_get_keys_perm(sph_ctx* ctx, sph_mem mem, uint64_t* sorted_keys, uint32_t* perm);
/* Tree tables of the N-1 internal nodes (Table B2 conventions: node index = one end of its range):
 * left/right child ids, leaf flags (1 = child is a leaf = sorted slot), parent (2N-1 entries: internal i at [i],
 * leaf j at [N-1+j], root -1), range lo/hi, aabb (6 per node: min xyz, max xyz), hmax. Any may be NULL. */
int sph_get_tree(sph_ctx* ctx, sph_mem mem, int32_t* left, int32_t* right, uint8_t* lflag, uint8_t* rflag,
                 int32_t* parent, int32_t* range_lo, int32_t* range_hi, double* aabb, double* hmax);
/* Neighbour cache as CSR over sorted slots: offs[N+1], idx[cap] (sorted-slot indices, unordered within a list).
 * idx may be NULL to query offs only; SPH_ERR_CAP if cap < offs[N]. */
int sph_get_neighbours(sph_ctx* ctx, sph_mem mem, uint64_t* offs, uint32_t* idx, uint64_t cap);
/* The same for the sorted slots [first, first + count) only (parity checks on samples of a large run, where the whole
 * CSR would be several GB): offs[count + 1] are the ABSOLUTE offsets offs_all[first .. first + count], idx[cap]
 * receives the lists of those slots back to back (list of slot first + k at idx[offs[k] - offs[0]]).
 * SPH_ERR_ARG if the range leaves [0, N); SPH_ERR_CAP if cap < offs[count] - offs[0]. */
int sph_get_neighbours_range(sph_ctx* ctx, sph_mem mem, int64_t first, int64_t count, uint64_t* offs, uint32_t* idx,
                             uint64_t cap);
/* Reduced leaves of Alg. 1 (only with sph_params.leaf_reduction >= 1; SPH_ERR_ORDER otherwise): *n_leaves, their
 * Morton codes leaf_codes[n_leaves] and the index map id_map[n_leaves + 1] (sorted slot of each kept code, closed by
 * N; leaf j holds the sorted slots [id_map[j], id_map[j+1]), Alg. 2). Buffers must hold N and N + 1
 * entries; either may be NULL. */
int sph_get_leaves(sph_ctx* ctx, sph_mem mem, int64_t* n_leaves, uint64_t* leaf_codes, uint32_t* id_map);
/* Shock-switch alpha_a in ORIGINAL particle order (sph_params.av_switch = 1; SPH_ERR_ORDER otherwise). */
int sph_get_alpha(sph_ctx* ctx, sph_mem mem, double* alpha);
int sph_get_stats(sph_ctx* ctx, sph_stats* out);
int sph_reset_timers(sph_ctx* ctx);
const char* sph_last_error(const sph_ctx* ctx);
void sph_free(sph_ctx* ctx);

/* Measured FP64 FMA throughput of the device in TFLOP/s (dependent-free DFMA microbenchmark; used as the
 * roofline denominator for the density and force kernels because MEASURED_PEAKS.json has no FP64 entry).
 * sm_mhz_out (may be NULL) is not measured here; bench.py samples clocks with nvidia-smi. */
int sph_measure_fp64_peak(double* tflops_out, void* cuda_stream);

/* An entry point that ALLOCATES NOTHING, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it): the exclusive prefix sum behind the neighbour-cache offsets (Alg. 5,
 * PAPER.md:1124-1130) and the stream compaction, as a variant of the library's decoupled look-back
 * scan whose scratch memory is a static device array of the library.
 *   in_dev[n]  (DEVICE) u32 counts;  out_dev[n + 1] (DEVICE) u64 exclusive prefix sums, out_dev[n] = total. The caller
 *   owns both; the work is enqueued on cuda_stream (a cudaStream_t, NULL = default stream) of the CURRENT device and the
 *   call returns without synchronising.
 *   Limit: n <= sph_scan_noalloc_max_items() = 2^24 = 16 777 216 (the static scratch is 65 792 bytes, held by every GPU
 *   that loads the library until the process exits); larger n: SPH_ERR_CAP. n < 1 or a null pointer: SPH_ERR_ARG; no
 *   usable device: SPH_ERR_DEVICE. sph_noalloc_last_error() gives the text of the calling thread's last failure.
 *   All calls on a device share the one scratch array. Each call clears what it uses, stream-ordered, before its
 *   kernel, so calls ordered on one stream (or by events) are safe back to back; calls that OVERLAP on the GPU (two
 *   streams without ordering between them) race on it and give wrong sums. Calls no cudaMalloc / cudaFree. */
int sph_scan_u32_noalloc(const uint32_t* in_dev, uint64_t* out_dev, int64_t n, void* cuda_stream);
int64_t sph_scan_noalloc_max_items(void);
const char* sph_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
