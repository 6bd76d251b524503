// density.cu -- a5: smoothing-length / density Newton-Raphson iteration (Alg. 7; F1-F2,
// PAPER.md:1235-1239; lambda clamp and chi tolerance PAPER.md:1245; sign safeguard DESIGN.md reading A5b), then
// rho = m (hfact/h)^3 and Omega (Eq. 7) at the converged h.
//
// One CTA of eight warps per leaf group. The group's candidate array is staged once into shared memory with
// cp.async copies: x, y, z, m of every candidate (groups with more candidates than fit gather from global memory). Every particle of the group
// is owned by one octet (8 lanes): warp w, octet o -> particle 4 w + o, so a warp iterates four independent Newton
// solves at once and the scalar update is executed 8-fold instead of 32-fold redundantly. The octet's lanes split
// the particle's neighbour list (16-bit indices into the staged candidates); r_ab and m_b are computed once and
// kept in registers for every Newton sweep (r does not depend on h): a sweep costs only the kernel evaluation and
// two three-step octet reductions. Lists longer than 96 entries re-gather the excess from shared memory per
// sweep. Groups whose buckets cannot wrap around a periodic axis use plain differences. No global gathers remain.
#include <type_traits>

#include "common.cuh"

namespace sph {

constexpr int kDensWarps = 8;
constexpr int kRegChunks = 10;    // 10 x 8 = 80 inner neighbours held in registers per octet (kernels of radius 2)
// M5 / M6 (radii 2.5 and 3: ~157 neighbours at h_fact 1.2 / 1.0) keep 20 x 8 = 160; their launches run 2 CTAs per SM
template <int K> constexpr int kRegChunksK = (K == 1 || K == 2) ? 20 : kRegChunks;

struct DensBox { double L[3], halfL[3]; int periodic[3]; };

template <bool WRAP>
__device__ __forceinline__ double sep_r(double xa, double ya, double za, const double* __restrict__ sx,
                                        const double* __restrict__ sy, const double* __restrict__ sz, uint32_t b,
                                        const DensBox& db) {
    double dx = xa - sx[b], dy = ya - sy[b], dz = za - sz[b];
    if (WRAP) {
        if (db.periodic[0]) { if (dx > db.halfL[0]) dx -= db.L[0]; else if (dx < -db.halfL[0]) dx += db.L[0]; }
        if (db.periodic[1]) { if (dy > db.halfL[1]) dy -= db.L[1]; else if (dy < -db.halfL[1]) dy += db.L[1]; }
        if (db.periodic[2]) { if (dz > db.halfL[2]) dz -= db.L[2]; else if (dz < -db.halfL[2]) dz += db.L[2]; }
    }
    // r = r2 / sqrt(r2) with the hardware reciprocal-square-root seed and one third-order refinement (relative error
    // ~1e-16, no range checks: r2 is a squared separation); the particle itself (r2 = 0) gives r = 0
    const double r2 = dx * dx + dy * dy + dz * dz;
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(r2));
    const double e = fma(r2, -(y0 * y0), 1.0);
    const double y = fma(fma(e, 0.375, 0.5), y0 * e, y0);
    return r2 > 0.0 ? r2 * y : 0.0;
}

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc)
                 : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
    asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

__device__ __forceinline__ double octet_sum(double v) {
    v += __shfl_xor_sync(0xffffffffu, v, 4);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    return v;
}

struct DensPar { double hfact, chi, lambda, eps_h; int max_iter; };

// f(q) and g(q) = (3 f + q f') / kGScale of kernel K: what a sweep sums (dW/dh = -C h^-4 (3 f + q f')). For M4 the two
// polynomials of each branch are evaluated directly (14 instead of 16 FP64 instructions per neighbour and sweep):
//   q < 1:      f = 1 + q^2 (3q/4 - 3/2),   g = 1 + q^2 (3q/2 - 5/2)
//   1 <= q < 2: f = (2-q)^3 / 4,            g = (2-q)^2 (2 - 2q) / 4          (g = (3 f + q f') / 3)
template <int K> constexpr double kGScale = (K == 0) ? 3.0 : 1.0;
template <int K>
__device__ __forceinline__ void kern_f_g(double q, double& f, double& g) {
    if (K == 0) {
        const double q2 = q * q, t = 2.0 - q;
        const double fi = fma(q2, fma(0.75, q, -1.5), 1.0), gi = fma(q2, fma(1.5, q, -2.5), 1.0);
        const double b = 0.25 * (t * t);
        const double fo = b * t, go = b * (t - q);
        const int qh = __double2hiint(q);                        // q >= +0: integer range tests, see m4()
        const bool in = qh < 0x3FF00000, sup = qh < 0x40000000;
        f = in ? fi : (sup ? fo : 0.0);
        g = in ? gi : (sup ? go : 0.0);
    } else {
        double df;
        kern_f_df<K>(q, f, df);
        g = fma(q, df, 3.0 * f);
    }
}
struct DensOut { double h, rho, om; bool exceeded, noconv, grew; int it; };

// UNIM: every candidate of the group has the same mass (checked while staging): the mass factors out of the sums
// and the per-neighbour mass registers disappear.
// GLOB: the candidate array is too large to stage; sx, sy, sz, sm are the global field arrays and a candidate index
// is translated through the group's candidate array cs first.
template <bool WRAP, bool UNIM, bool GLOB, int K>
__device__ __forceinline__ void octet_solve(double xa, double ya, double za, double ma, double h0, bool pv,
                                            const uint32_t* __restrict__ cs,
                                            const uint16_t* __restrict__ li, const uint32_t (&idx)[(kRegChunksK<K> + 1) / 2],
                                            int n, int ntot, unsigned sl, const double* __restrict__ sx, const double* __restrict__ sy,
                                            const double* __restrict__ sz, const double* __restrict__ sm,
                                            const DensBox& db, const DensPar& dp, DensOut& out) {
    double r[kRegChunksK<K>], mb[UNIM ? 1 : kRegChunksK<K>];
    const double m0 = ma;                              // UNIM: every particle has this mass
#pragma unroll
    for (int c = 0; c < kRegChunksK<K>; ++c) {
        const int k = c * 8 + (int)sl;
        r[c] = 1e100;                                  // q >> 2 (finite): outside the kernel support, contributes 0
        if (!UNIM) mb[c] = 0.0;
        if (k < n) {
            uint32_t b = (idx[c >> 1] >> (16 * (c & 1))) & 0xffffu;
            if (GLOB) b = cs[b];
            r[c] = sep_r<WRAP>(xa, ya, za, sx, sy, sz, b, db);
            if (!UNIM) mb[c] = sm[b];
        }
    }
    // sums over the list at smoothing length h: rs = sum m f(q), ss = sum m (3 f + q f')
    // `n` inner entries (registers, then re-gathered beyond them); the ntot - n shell entries lie beyond
    // R_kern (1 + kShellEps) h0 and are only read while h exceeds kShellGrow h0 (exact: they contribute nothing below)
    const double hlim = kShellGrow * h0;
    // (with_rho = false_type: the closing pass needs S only; the f polynomial then drops out at compile time)
    auto sums = [&](auto with_rho, double hcur, double hinv, double& rho_sum, double& S) {
        constexpr bool kRho = decltype(with_rho)::value;
        double rs = 0.0, ss = 0.0;
#pragma unroll
        for (int c = 0; c < kRegChunksK<K>; ++c) {
            double f, g;
            kern_f_g<K>(r[c] * hinv, f, g);
            if (UNIM) {
                if (kRho) rs += f;
                ss += g;
            } else {
                if (kRho) rs = fma(mb[c], f, rs);
                ss = fma(mb[c], g, ss);
            }
        }
        for (int k = kRegChunksK<K> * 8 + (int)sl; k < n; k += 8) {      // long lists: re-gather from smem
            uint32_t b = li[k];
            if (GLOB) b = cs[b];
            double f, g;
            const double mm = UNIM ? 1.0 : sm[b];
            kern_f_g<K>(sep_r<WRAP>(xa, ya, za, sx, sy, sz, b, db) * hinv, f, g);
            if (kRho) rs = fma(mm, f, rs);
            ss = fma(mm, g, ss);
        }
        if (hcur > hlim) {
            for (int k = n + (int)sl; k < ntot; k += 8) {
                uint32_t b = li[k];
                if (GLOB) b = cs[b];
                double f, g;
                const double mm = UNIM ? 1.0 : sm[b];
                kern_f_g<K>(sep_r<WRAP>(xa, ya, za, sx, sy, sz, b, db) * hinv, f, g);
                rs = fma(mm, f, rs);
                ss = fma(mm, g, ss);
            }
        }
        if (kRho) rs = octet_sum(rs);
        ss = octet_sum(ss);
        const double c3 = (UNIM ? m0 : 1.0) * kern_cnorm(K) * hinv * hinv * hinv;
        rho_sum = c3 * rs;            // Eq. 1-2
        S = -c3 * hinv * (kGScale<K> * ss);   // sum_b m_b dW/dh
    };

    const double inv_lambda = 1.0 / dp.lambda, h0inv = 1.0 / h0;
    double h = h0;
    bool exceeded = false, converged = false, active = pv;
    int it = 0;
    while (__any_sync(0xffffffffu, active)) {      // the four octets of a warp iterate together
        double rho_sum, S;
        const double hinv = 1.0 / h;                                // the one reciprocal of a sweep besides f / f'
        sums(std::true_type{}, h, hinv, rho_sum, S);
        if (active) {
            ++it;
            const double hf = dp.hfact * hinv;
            const double rho_h = ma * hf * hf * hf;                 // F1
            const double f = rho_sum - rho_h;                       // F2
            const double fp = S + 3.0 * rho_h * hinv;               // exact derivative (reading A5)
            double hnew = h - f / fp;                               // Alg. 7 l.10
            if (!(fp > 0.0) || (hnew - h) * f > 0.0 || !(hnew == hnew))
                hnew = (f > 0.0) ? h * inv_lambda : h * dp.lambda;  // safeguard 2b
            if (hnew > h * dp.lambda) hnew = h * dp.lambda;         // Alg. 7 l.11-13
            else if (hnew < h * inv_lambda) hnew = h * inv_lambda;
            const double eps = fabs(hnew - h) * h0inv;              // Alg. 7 l.14
            if (hnew > h0 * dp.chi) { hnew = h0 * dp.chi; exceeded = true; }   // Alg. 7 l.15-17
            h = hnew;
            if (!exceeded && eps <= dp.eps_h) converged = true;
            if (exceeded || converged || it >= dp.max_iter) active = false;
        }
    }
    double rho_sum, S;
    const double hinv = 1.0 / h;
    sums(std::false_type{}, h, hinv, rho_sum, S);      // closing pass at the converged h: Omega needs S only
    const double hf = dp.hfact * hinv;
    const double rho_a = ma * hf * hf * hf;
    out.h = h;
    out.rho = rho_a;
    out.om = 1.0 + h / (3.0 * rho_a) * S;                           // Eq. 7 with dh/drho = -h/(3 rho)
    out.exceeded = exceeded;
    out.grew = h > hlim;
    out.noconv = pv && !exceeded && !converged;
    out.it = it;
}

template <bool UNIM, bool GLOB, int K>
__global__ void __launch_bounds__(kDensWarps * 32, (UNIM && (K == 0 || K >= 3)) ? 3 : 2) k_density(
    const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
    const double* __restrict__ m, const double* __restrict__ hn, const uint32_t* __restrict__ grp_lo,
    const GroupRec* __restrict__ ginfo, const uint32_t* __restrict__ cslot, const uint32_t* __restrict__ cnt,
    const uint32_t* __restrict__ cnt_in, uint8_t* __restrict__ grow, const uint64_t* __restrict__ lstart, const uint16_t* __restrict__ lists, DensBox db, DensPar dp, uint32_t ncap,
    uint32_t nc_lo, uint32_t nc_hi,
    double* __restrict__ hout, double* __restrict__ rho, double* __restrict__ omega, DevScalars* sc) {
    extern __shared__ __align__(16) double dsm[];
    double* sx = dsm;
    double* sy = sx + ncap;
    double* sz = sy + ncap;
    double* sm = sz + ncap;
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
    const unsigned sub = lane >> 3, sl = lane & 7u;
    const uint32_t g = blockIdx.x;
    const uint32_t glo = grp_lo[g], nq = grp_lo[g + 1] - glo;
    const GroupRec gr = ginfo[g];
    const uint32_t* cs = cslot + (((uint64_t)gr.cs_off_hi << 32) | gr.cs_off_lo);
    const uint32_t nc = gr.nc & 0x7fffffffu;
    if (nc <= nc_lo || nc > nc_hi) return;       // this launch serves the groups with nc in (nc_lo, nc_hi]
    const bool gwrap = (gr.nc >> 31) != 0u;

    // this octet's particle (loads issued before the staging loop so that their latency overlaps it)
    const uint32_t q = 4u * warp + sub;
    const bool pv = q < nq;
    const uint32_t a = glo + (pv ? q : 0u);
    const double xa = x[a], ya = y[a], za = z[a], ma = m[a], h0 = hn[a];
    const uint16_t* li = lists + lstart[a];
    const int ntot = pv ? (int)cnt[a] : 0, n = pv ? (int)cnt_in[a] : 0;

    // ---- stage the candidate array (slots are mostly runs of consecutive indices: coalesced sectors) ----
    if (!GLOB) {
        for (uint32_t c = threadIdx.x; c < nc; c += kDensWarps * 32) {
            const uint32_t s = cs[c];
            cp_async8(sx + c, x + s); cp_async8(sy + c, y + s); cp_async8(sz + c, z + s); cp_async8(sm + c, m + s);
        }
    } else {
        sx = const_cast<double*>(x); sy = const_cast<double*>(y); sz = const_cast<double*>(z); sm = const_cast<double*>(m);
    }
    // the first 96 (M5, M6: 160) list entries of the octet's particle (two 16-bit indices per register), in flight together with
    // the staging copies
    uint32_t idx[(kRegChunksK<K> + 1) / 2];
#pragma unroll
    for (int c = 0; c < kRegChunksK<K>; c += 2) {
        const int k0 = c * 8 + (int)sl, k1 = k0 + 8;
        const uint32_t i0 = (k0 < n) ? (uint32_t)li[k0] : 0u, i1 = (c + 1 < kRegChunksK<K> && k1 < n) ? (uint32_t)li[k1] : 0u;
        idx[c >> 1] = i0 | (i1 << 16);
    }
    cp_async_wait_all();
    __syncthreads();

    DensOut o;
    if (gwrap) octet_solve<true, UNIM, GLOB, K>(xa, ya, za, ma, h0, pv, cs, li, idx, n, ntot, sl, sx, sy, sz, sm, db, dp, o);
    else octet_solve<false, UNIM, GLOB, K>(xa, ya, za, ma, h0, pv, cs, li, idx, n, ntot, sl, sx, sy, sz, sm, db, dp, o);

    if (pv && sl == 0u) {
        hout[a] = o.h;
        rho[a] = o.rho;
        omega[a] = o.om;
        grow[a] = o.grew ? 1 : 0;
    }
    const unsigned exc = __ballot_sync(0xffffffffu, pv && sl == 0u && o.exceeded);
    const unsigned ncv = __ballot_sync(0xffffffffu, sl == 0u && o.noconv);
    unsigned itm = (unsigned)o.it;
#pragma unroll
    for (int ofs = 16; ofs > 0; ofs >>= 1) itm = max(itm, __shfl_xor_sync(0xffffffffu, itm, ofs));
    // executed sweeps of this warp's particles: Newton sweeps + the closing pass at the final h (bench.py's flop count)
    unsigned swp = (pv && sl == 0u) ? (unsigned)o.it + 1u : 0u;
#pragma unroll
    for (int ofs = 16; ofs > 0; ofs >>= 1) swp += __shfl_xor_sync(0xffffffffu, swp, ofs);
    const unsigned gm = __ballot_sync(0xffffffffu, pv && sl == 0u && o.grew);
    if (lane == 0) {
        if (exc) atomicAdd(&sc->n_exceeded, (unsigned)__popc(exc));
        if (ncv) atomicAdd(&sc->n_noconv, (unsigned)__popc(ncv));
        atomicMax(&sc->h_iter_max, itm);
        atomicAdd(&sc->sweeps, (unsigned long long)swp);
        if (gm) atomicAdd(&sc->n_grew, (unsigned long long)__popc(gm));
    }
}

__global__ void k_density_reset(DevScalars* sc) { sc->n_exceeded = 0; sc->n_noconv = 0; sc->h_iter_max = 0; sc->sweeps = 0ull; sc->n_grew = 0ull; }

template <bool UNIM, bool GLOB, int K>
static int density_launch_k(sph_ctx* c, size_t smem, const DensBox& db, const DensPar& dp, uint32_t ncap, uint32_t lo,
                            uint32_t hi) {
    if (!GLOB)   // per device: set on every launch
        SPH_CUDA(c, cudaFuncSetAttribute(k_density<UNIM, GLOB, K>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    k_density<UNIM, GLOB, K><<<(unsigned)c->n_groups, kDensWarps * 32, smem, c->stream>>>(
        c->cur.x, c->cur.y, c->cur.z, c->cur.m, c->cur.h, c->grp_lo, c->ginfo, c->cslot, c->cnt, c->cnt_in, c->grow, c->lstart, c->lists, db, dp,
        ncap, lo, hi, c->hnew, c->rho, c->omega, c->d_sc);
    c->launches++;
    return SPH_OK;
}

template <bool UNIM, bool GLOB>
static int density_launch(sph_ctx* c, size_t smem, const DensBox& db, const DensPar& dp, uint32_t ncap, uint32_t lo,
                          uint32_t hi) {
    if (c->p.kernel == 0) return density_launch_k<UNIM, GLOB, 0>(c, smem, db, dp, ncap, lo, hi);
    if (c->p.kernel == 1) return density_launch_k<UNIM, GLOB, 1>(c, smem, db, dp, ncap, lo, hi);
    if (c->p.kernel == 2) return density_launch_k<UNIM, GLOB, 2>(c, smem, db, dp, ncap, lo, hi);
    if (c->p.kernel == 3) return density_launch_k<UNIM, GLOB, 3>(c, smem, db, dp, ncap, lo, hi);
    if (c->p.kernel == 4) return density_launch_k<UNIM, GLOB, 4>(c, smem, db, dp, ncap, lo, hi);
    return density_launch_k<UNIM, GLOB, 5>(c, smem, db, dp, ncap, lo, hi);
}

int launch_density(sph_ctx* c) {
    DensBox db;
    for (int k = 0; k < 3; ++k) {
        db.L[k] = c->box.hi[k] - c->box.lo[k];
        db.halfL[k] = 0.5 * db.L[k];
        db.periodic[k] = c->box.periodic[k];
    }
    DensPar dp;
    dp.hfact = c->p.hfact; dp.chi = c->p.chi; dp.lambda = c->p.lambda; dp.eps_h = c->p.eps_h; dp.max_iter = c->p.max_h_iter;
    k_density_reset<<<1, 1, 0, c->stream>>>(c->d_sc);
    c->launches++;
    // The staged candidate array sizes the CTA's shared memory, hence the occupancy: groups are served in size
    // classes (a CTA whose group belongs to another class exits at once), so that a few crowded groups (density
    // jumps, disc mid-plane) do not cost everyone else their occupancy: up to kSmall candidates; up to kStage (what
    // fits in shared memory at all); beyond that, a variant that gathers from global memory (poor initial h only).
    const uint32_t kSmall = 768, kStage = 227 * 1024 / 32;
    const uint32_t bounds[4] = {0u, kSmall, kStage, 0x7fffffffu};
    for (int cls = 0; cls < 3; ++cls) {
        const uint32_t lo = bounds[cls], hi = bounds[cls + 1];
        if (c->nc_max <= lo) break;                      // nc = 0 cannot occur (a particle is its own neighbour)
        const uint32_t ncap = cls == 2 ? 0u : ((c->nc_max < hi ? c->nc_max : hi) + 31u) & ~31u;
        const size_t smem = (size_t)ncap * 4 * sizeof(double);
        if (c->uniform_mass) {      // all masses equal (checked once at init): no per-neighbour mass registers
            if (cls == 2) SPH_TRY((density_launch<true, true>(c, smem, db, dp, ncap, lo, hi)));
            else SPH_TRY((density_launch<true, false>(c, smem, db, dp, ncap, lo, hi)));
        } else {
            if (cls == 2) SPH_TRY((density_launch<false, true>(c, smem, db, dp, ncap, lo, hi)));
            else SPH_TRY((density_launch<false, false>(c, smem, db, dp, ncap, lo, hi)));
        }
    }
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
