// density.cu -- a5: smoothing-length / density Newton-Raphson iteration (Alg. 7; F1-F2,
// PAPER.md:1235-1239; lambda clamp and chi tolerance PAPER.md:1245; sign safeguard DESIGN.md reading A5b), then
// rho = m (hfact/h)^3 and Omega (Eq. 7) at the converged h.
//
// One CTA of four warps per leaf group. The group's candidate array (the slot ranges of its bucket table) is
// staged once into shared memory with coalesced loads: x, y, z, m of every candidate. Each warp then takes every
// fourth particle of the group; the 32 lanes split that particle's neighbour list (16-bit indices into the staged
// candidates, read coalesced). r_ab and m_b are computed once per particle and kept in registers for every Newton
// sweep (r does not depend on h): a sweep costs only the kernel evaluation and two warp reductions. Lists longer
// than 96 entries take a path that re-gathers from shared memory per sweep. No global gathers remain.
#include "common.cuh"

namespace sph {

constexpr int kDensWarps = 4;
constexpr int kRegChunks = 3;     // 3 x 32 = 96 neighbours held in registers

struct DensBox { double L[3], halfL[3]; int periodic[3]; };

__device__ __forceinline__ double wrap_sep(double d, double L, double halfL, int periodic) {
    if (periodic) {
        if (d > halfL) d -= L;
        else if (d < -halfL) d += L;
    }
    return d;
}

__global__ void __launch_bounds__(kDensWarps * 32) k_density(
    const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
    const double* __restrict__ m, const double* __restrict__ hn, const uint32_t* __restrict__ grp_lo,
    const GroupRec* __restrict__ ginfo, const BucketRec* __restrict__ bkt, const uint32_t* __restrict__ cnt,
    const uint64_t* __restrict__ lstart, const uint16_t* __restrict__ lists, DensBox db, double hfact, double chi,
    double lambda, double eps_h, int max_iter, uint32_t ncap, double* __restrict__ hout, double* __restrict__ rho,
    double* __restrict__ omega, DevScalars* sc) {
    extern __shared__ __align__(16) double dsm[];
    double* sx = dsm;
    double* sy = sx + ncap;
    double* sz = sy + ncap;
    double* sm = sz + ncap;
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
    const uint32_t g = blockIdx.x;
    const uint32_t glo = grp_lo[g], nq = grp_lo[g + 1] - glo;
    const GroupRec gr = ginfo[g];
    const BucketRec* tab = bkt + (((uint64_t)gr.bkt_off_hi << 32) | gr.bkt_off_lo);

    // ---- stage the candidate array: one bucket (<= 32 consecutive slots) per warp iteration ----
    for (uint32_t j = warp; j < gr.nb; j += kDensWarps) {
        const BucketRec b0 = tab[j];
        const uint32_t n = tab[j + 1].cstart - b0.cstart;
        if (lane < n) {
            const uint32_t s = b0.lo + lane, c = b0.cstart + lane;
            sx[c] = x[s]; sy[c] = y[s]; sz[c] = z[s]; sm[c] = m[s];
        }
    }
    __syncthreads();

    double out_h = 0.0, out_rho = 0.0, out_om = 0.0;
    unsigned n_exc = 0, n_noconv = 0, it_max = 0;
    const double inv_lambda = 1.0 / lambda;

    for (uint32_t q = warp; q < nq; q += kDensWarps) {
        const uint32_t a = glo + q;
        const uint16_t* li = lists + lstart[a];
        const int n = (int)cnt[a];
        const double xa = x[a], ya = y[a], za = z[a], ma = m[a], h0 = hn[a];
        double r[kRegChunks], mb[kRegChunks];
#pragma unroll
        for (int c = 0; c < kRegChunks; ++c) {
            const int k = c * 32 + (int)lane;
            r[c] = 0.0; mb[c] = 0.0;
            if (k < n) {
                const uint32_t b = li[k];
                const double dx = wrap_sep(xa - sx[b], db.L[0], db.halfL[0], db.periodic[0]);
                const double dy = wrap_sep(ya - sy[b], db.L[1], db.halfL[1], db.periodic[1]);
                const double dz = wrap_sep(za - sz[b], db.L[2], db.halfL[2], db.periodic[2]);
                r[c] = sqrt(dx * dx + dy * dy + dz * dz);
                mb[c] = sm[b];
            }
        }
        // sums over the list at smoothing length h: rs = sum m f(q), ss = sum m (3 f + q f')
        auto sums = [&](double h, double& rho_sum, double& S) {
            const double hinv = 1.0 / h;
            double rs = 0.0, ss = 0.0;
#pragma unroll
            for (int c = 0; c < kRegChunks; ++c) {
                double qq = r[c] * hinv, f, df;
                m4(qq, f, df);
                rs = fma(mb[c], f, rs);
                ss = fma(mb[c], fma(qq, df, 3.0 * f), ss);
            }
            for (int k = kRegChunks * 32 + (int)lane; k < n; k += 32) {      // long lists: re-gather from smem
                const uint32_t b = li[k];
                const double dx = wrap_sep(xa - sx[b], db.L[0], db.halfL[0], db.periodic[0]);
                const double dy = wrap_sep(ya - sy[b], db.L[1], db.halfL[1], db.periodic[1]);
                const double dz = wrap_sep(za - sz[b], db.L[2], db.halfL[2], db.periodic[2]);
                double qq = sqrt(dx * dx + dy * dy + dz * dz) * hinv, f, df;
                const double mm = sm[b];
                m4(qq, f, df);
                rs = fma(mm, f, rs);
                ss = fma(mm, fma(qq, df, 3.0 * f), ss);
            }
            rs = warp_sum(rs);
            ss = warp_sum(ss);
            const double c3 = kCnorm * hinv * hinv * hinv;
            rho_sum = c3 * rs;            // Eq. 1-2
            S = -c3 * hinv * ss;          // sum_b m_b dW/dh
        };

        double h = h0;
        bool exceeded = false, converged = false;
        int it = 0;
        while (it < max_iter) {
            ++it;
            double rho_sum, S;
            sums(h, rho_sum, S);
            const double hf = hfact / h;
            const double rho_h = ma * hf * hf * hf;                 // F1
            const double f = rho_sum - rho_h;                       // F2
            const double fp = S + 3.0 * rho_h / h;                  // exact derivative (reading A5)
            double hnew = h - f / fp;                               // Alg. 7 l.10
            if (!(fp > 0.0) || (hnew - h) * f > 0.0 || !(hnew == hnew))
                hnew = (f > 0.0) ? h * inv_lambda : h * lambda;     // safeguard 2b
            if (hnew > h * lambda) hnew = h * lambda;               // Alg. 7 l.11-13
            else if (hnew < h * inv_lambda) hnew = h * inv_lambda;
            const double eps = fabs(hnew - h) / h0;                 // Alg. 7 l.14
            if (hnew > h0 * chi) { hnew = h0 * chi; exceeded = true; }   // Alg. 7 l.15-17
            h = hnew;
            if (exceeded) break;
            if (eps <= eps_h) { converged = true; break; }
        }
        double rho_sum, S;
        sums(h, rho_sum, S);
        const double hf = hfact / h;
        const double rho_a = ma * hf * hf * hf;
        if (lane == (q >> 2)) {                                     // lane j keeps this warp's j-th particle
            out_h = h;
            out_rho = rho_a;
            out_om = 1.0 + h / (3.0 * rho_a) * S;                   // Eq. 7 with dh/drho = -h/(3 rho)
            n_exc += exceeded;
            n_noconv += (!exceeded && !converged);
        }
        it_max = max(it_max, (unsigned)it);
    }
    {
        const uint32_t q = warp + kDensWarps * lane;
        if (q < nq) {
            hout[glo + q] = out_h;
            rho[glo + q] = out_rho;
            omega[glo + q] = out_om;
        }
    }
    const unsigned any_exc = __ballot_sync(0xffffffffu, n_exc != 0), any_nc = __ballot_sync(0xffffffffu, n_noconv != 0);
    if (lane == 0) {
        if (any_exc) atomicAdd(&sc->n_exceeded, (unsigned)__popc(any_exc));
        if (any_nc) atomicAdd(&sc->n_noconv, (unsigned)__popc(any_nc));
        atomicMax(&sc->h_iter_max, it_max);
    }
}

__global__ void k_density_reset(DevScalars* sc) { sc->n_exceeded = 0; sc->n_noconv = 0; sc->h_iter_max = 0; }

int launch_density(sph_ctx* c) {
    static bool attr_set = false;
    if (!attr_set) {
        SPH_CUDA(c, cudaFuncSetAttribute(k_density, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        attr_set = true;
    }
    DensBox db;
    for (int k = 0; k < 3; ++k) {
        db.L[k] = c->box.hi[k] - c->box.lo[k];
        db.halfL[k] = 0.5 * db.L[k];
        db.periodic[k] = c->box.periodic[k];
    }
    const uint32_t ncap = (c->nc_max + 31u) & ~31u;
    const size_t smem = (size_t)ncap * 4 * sizeof(double);
    if (smem > 227 * 1024)
        return fail(c, SPH_ERR_CAP, "a leaf group has %u candidates: more than the density kernel can stage (%d)",
                    c->nc_max, 227 * 1024 / 32);
    k_density_reset<<<1, 1, 0, c->stream>>>(c->d_sc);
    k_density<<<(unsigned)c->n_groups, kDensWarps * 32, smem, c->stream>>>(
        c->cur.x, c->cur.y, c->cur.z, c->cur.m, c->cur.h, c->grp_lo, c->ginfo, c->bkt, c->cnt, c->lstart, c->lists, db,
        c->p.hfact, c->p.chi, c->p.lambda, c->p.eps_h, c->p.max_h_iter, ncap, c->hnew, c->rho, c->omega,
        c->d_sc);
    c->launches += 2;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
