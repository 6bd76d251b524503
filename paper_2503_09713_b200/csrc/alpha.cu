// alpha.cu -- shock switch: per-particle artificial-viscosity alpha_a evolved by the implicit step G13
// (G11-G13; constants alpha_min = 0, alpha_max = 1, sigma_decay = 0.1 of the runscript,
// PAPER.md:1412-1415). alpha_loc and tau are not in PAPER.md (it defers to Price et al. 2018, Sect. 2.2.9): DESIGN.md
// reading A18 -- SPH first-derivative estimates d_j f |_a = -(1 / (Omega_a rho_a)) sum_b m_b (f_a - f_b) r_hat_j F_ab(h_a)
// of v* (divergence, curl, full tensor) and of a^n (divergence), d(div v)/dt = div a - sum_ij (d_j v_i)(d_i v_j),
// xi = (div v)^2 / ((div v)^2 + |curl v|^2), A = xi max(-d(div v)/dt, 0), alpha_loc = clamp(10 h^2 A / c_s^2),
// tau = h / (sigma_decay c_s). Runs between the smoothing-length update and the derivatives (Fig. G1).
//
// Same structure as forces.cu: one CTA of eight warps per leaf group, the group's candidate fields (x y z, v, a^n, m)
// staged in shared memory in chunks, one octet of lanes per particle splitting its neighbour list, ten accumulators
// reduced over the octet. Off by default (sph_params.av_switch); not on the path bench.py times.
#include "common.cuh"

namespace sph {

constexpr int kAlphaWarps = 8;
constexpr int kAChunk = 640;
constexpr int kARows = 10;      // x y z vx vy vz ax ay az m

struct AlphaArgs {
    double L[3], halfL[3];
    int periodic[3];
    double alpha_min, alpha_max, sigma_decay;
};

struct AlphaIn {
    const double *x, *y, *z, *vx, *vy, *vz, *ax, *ay, *az, *m, *h, *rho, *omega, *cs;
    const uint32_t* grp_lo;
    const GroupRec* ginfo;
    const uint32_t* cslot;
    const uint32_t* cnt;
    const uint32_t* cnt_in;
    const uint64_t* lstart;
    const uint16_t* lists;
};

__device__ __forceinline__ void cp_async8a(double* smem_dst, const double* gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc)
                 : "memory");
}

template <int K>
__global__ void __launch_bounds__(kAlphaWarps * 32, 2) k_alpha(AlphaIn in, AlphaArgs aa, const double* __restrict__ dtp,
                                                               double* __restrict__ alpha, double* __restrict__ acs) {
    extern __shared__ __align__(16) double asm_[];
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
    const unsigned sub = lane >> 3, sl = lane & 7u;
    const uint32_t g = blockIdx.x;
    const uint32_t glo = in.grp_lo[g], nq = in.grp_lo[g + 1] - glo;
    const GroupRec gr = in.ginfo[g];
    const uint32_t* cs = in.cslot + (((uint64_t)gr.cs_off_hi << 32) | gr.cs_off_lo);
    const uint32_t nc = gr.nc & 0x7fffffffu;
    const bool gwrap = (gr.nc >> 31) != 0u;
    const uint32_t q = 4u * warp + sub;
    const bool pv = q < nq;
    const uint32_t a = glo + (pv ? q : 0u);
    const double xa = in.x[a], ya = in.y[a], za = in.z[a];
    const double va[3] = {in.vx[a], in.vy[a], in.vz[a]}, an[3] = {in.ax[a], in.ay[a], in.az[a]};
    const double ha = in.h[a], hinv = 1.0 / ha;
    const double ca4 = kern_cnorm(K) * (hinv * hinv) * (hinv * hinv);
    const uint16_t* li = in.lists + in.lstart[a];
    const uint32_t n = pv ? in.cnt[a] : 0u;      // all entries are read: inner, then shell
    double gv[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, diva = 0.0;
    for (uint32_t c0 = 0; c0 < nc; c0 += kAChunk) {
        const uint32_t c1 = min(nc, c0 + (uint32_t)kAChunk);
        if (c0 > 0) __syncthreads();
        for (uint32_t c = c0 + threadIdx.x; c < c1; c += kAlphaWarps * 32) {
            const uint32_t s = cs[c], d = c - c0;
            cp_async8a(asm_ + d, in.x + s); cp_async8a(asm_ + kAChunk + d, in.y + s); cp_async8a(asm_ + 2 * kAChunk + d, in.z + s);
            cp_async8a(asm_ + 3 * kAChunk + d, in.vx + s); cp_async8a(asm_ + 4 * kAChunk + d, in.vy + s);
            cp_async8a(asm_ + 5 * kAChunk + d, in.vz + s); cp_async8a(asm_ + 6 * kAChunk + d, in.ax + s);
            cp_async8a(asm_ + 7 * kAChunk + d, in.ay + s); cp_async8a(asm_ + 8 * kAChunk + d, in.az + s);
            cp_async8a(asm_ + 9 * kAChunk + d, in.m + s);
        }
        asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        // the octet's lanes split the list; entries outside the staged chunk are skipped (one chunk in the usual case)
        for (uint32_t k = sl;; k += 8u) {
            const uint32_t cl = (k < n) ? (uint32_t)li[k] : 0xffffffffu;
            const bool act = cl - c0 < c1 - c0;
            if (act) {
                const uint32_t b = cl - c0;
                double dx = xa - asm_[b], dy = ya - asm_[kAChunk + b], dz = za - asm_[2 * kAChunk + b];
                if (gwrap) {
                    if (aa.periodic[0]) { if (dx > aa.halfL[0]) dx -= aa.L[0]; else if (dx < -aa.halfL[0]) dx += aa.L[0]; }
                    if (aa.periodic[1]) { if (dy > aa.halfL[1]) dy -= aa.L[1]; else if (dy < -aa.halfL[1]) dy += aa.L[1]; }
                    if (aa.periodic[2]) { if (dz > aa.halfL[2]) dz -= aa.L[2]; else if (dz < -aa.halfL[2]) dz += aa.L[2]; }
                }
                const double r2 = dx * dx + dy * dy + dz * dz;
                if (r2 > 0.0) {
                    const double r = sqrt(r2), rinv = 1.0 / r;
                    double f, df;
                    kern_f_df<K>(r * hinv, f, df);
                    const double wF = asm_[9 * kAChunk + b] * ca4 * df * rinv;       // m_b F_ab(h_a) / r
                    const double t[3] = {wF * dx, wF * dy, wF * dz};
#pragma unroll
                    for (int i = 0; i < 3; ++i) {
                        const double dv = va[i] - asm_[(3 + i) * kAChunk + b];
#pragma unroll
                        for (int j = 0; j < 3; ++j) gv[i][j] = fma(dv, t[j], gv[i][j]);
                        diva = fma(an[i] - asm_[(6 + i) * kAChunk + b], t[i], diva);
                    }
                }
            }
            if (__ballot_sync(0xffffffffu, k + 8u < n) == 0u) break;
        }
    }
#pragma unroll
    for (int ofs = 4; ofs > 0; ofs >>= 1) {
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) gv[i][j] += __shfl_xor_sync(0xffffffffu, gv[i][j], ofs);
        diva += __shfl_xor_sync(0xffffffffu, diva, ofs);
    }
    if (pv && sl == 0u) {
        const double norm = -1.0 / (in.omega[a] * in.rho[a]);
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) gv[i][j] *= norm;
        diva *= norm;
        const double divv = gv[0][0] + gv[1][1] + gv[2][2];
        const double cx = gv[2][1] - gv[1][2], cy = gv[0][2] - gv[2][0], cz = gv[1][0] - gv[0][1];
        const double curl2 = cx * cx + cy * cy + cz * cz;
        double trs = 0.0;
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) trs += gv[i][j] * gv[j][i];
        const double ddivdt = diva - trs;
        const double den = divv * divv + curl2;
        const double xi = den > 0.0 ? divv * divv / den : 1.0;
        const double A = xi * fmax(-ddivdt, 0.0);
        const double c = in.cs[a];
        double aloc;
        if (c > 0.0) aloc = fmin(fmax(10.0 * ha * ha * A / (c * c), aa.alpha_min), aa.alpha_max);
        else aloc = A > 0.0 ? aa.alpha_max : aa.alpha_min;
        const double xdt = c > 0.0 ? *dtp * aa.sigma_decay * c / ha : 0.0;          // dt / tau
        const double anew = fmax((alpha[a] + aloc * xdt) / (1.0 + xdt), aloc);      // G13
        alpha[a] = anew;
        acs[a] = anew * c;
    }
}

template <int K>
static int alpha_launch_k(sph_ctx* c, const AlphaIn& in, const AlphaArgs& aa, const double* dtp) {
    const int smem = kARows * kAChunk * (int)sizeof(double);
    SPH_CUDA(c, cudaFuncSetAttribute(k_alpha<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    k_alpha<K><<<(unsigned)c->n_groups, kAlphaWarps * 32, smem, c->stream>>>(in, aa, dtp, c->alpha, c->acs);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

// v = cur.v (v* inside a step), a^n = cur.a, c_s from k_eos (c->cs); dtp = device scalar with the step's dt (0 for a
// standalone evaluation)
int launch_alpha(sph_ctx* c, const double* dtp) {
    AlphaArgs aa;
    for (int k = 0; k < 3; ++k) {
        aa.L[k] = c->box.hi[k] - c->box.lo[k];
        aa.halfL[k] = 0.5 * aa.L[k];
        aa.periodic[k] = c->box.periodic[k];
    }
    aa.alpha_min = c->p.alpha_min; aa.alpha_max = c->p.alpha_max; aa.sigma_decay = c->p.sigma_decay;
    AlphaIn in;
    in.x = c->cur.x; in.y = c->cur.y; in.z = c->cur.z; in.vx = c->cur.vx; in.vy = c->cur.vy; in.vz = c->cur.vz;
    in.ax = c->cur.ax; in.ay = c->cur.ay; in.az = c->cur.az; in.m = c->cur.m; in.h = c->cur.h; in.rho = c->rho;
    in.omega = c->omega; in.cs = c->cs;
    in.grp_lo = c->grp_lo; in.ginfo = c->ginfo; in.cslot = c->cslot; in.cnt = c->cnt; in.cnt_in = c->cnt_in; in.lstart = c->lstart; in.lists = c->lists;
    switch (c->p.kernel) {
        case 0: return alpha_launch_k<0>(c, in, aa, dtp);
        case 1: return alpha_launch_k<1>(c, in, aa, dtp);
        case 2: return alpha_launch_k<2>(c, in, aa, dtp);
        case 3: return alpha_launch_k<3>(c, in, aa, dtp);
        case 4: return alpha_launch_k<4>(c, in, aa, dtp);
        default: return alpha_launch_k<5>(c, in, aa, dtp);
    }
}

}  // namespace sph
