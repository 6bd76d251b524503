// leapfrog.cu -- a7: leapfrog kick-drift-kick with a global timestep (G1-G5, order of
// Fig. G1; u integrated like v, reading A13). Elementwise and HBM-bound. The timestep is
// read from device memory so that a step needs no host round trip for dt (reading A14).
#include <utility>

#include "common.cuh"

namespace sph {

void adopt_new_acc(sph_ctx* c);

struct WrapBox { double lo[3], hi[3], L[3]; int periodic[3]; };

__device__ __forceinline__ double wrap_pos(double r, double lo, double hi, double L, int periodic) {
    if (periodic) {
        if (r >= hi) r -= L;
        else if (r < lo) r += L;
        if (r >= hi) r = lo;       // r + L rounded up to hi
    }
    return r;
}

// G1-G3: v_half = v + dt/2 a; r += dt v_half (wrapped); v* = v_half + dt/2 a; same for u with du/dt
__global__ void __launch_bounds__(256) k_predict(int64_t N, Fields f, WrapBox wb, const double* __restrict__ dtp) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double dt = *dtp, hdt = 0.5 * dt;
    {
        double a = f.ax[i], vh = f.vx[i] + hdt * a;
        f.x[i] = wrap_pos(f.x[i] + dt * vh, wb.lo[0], wb.hi[0], wb.L[0], wb.periodic[0]);
        f.vx[i] = vh + hdt * a;
    }
    {
        double a = f.ay[i], vh = f.vy[i] + hdt * a;
        f.y[i] = wrap_pos(f.y[i] + dt * vh, wb.lo[1], wb.hi[1], wb.L[1], wb.periodic[1]);
        f.vy[i] = vh + hdt * a;
    }
    {
        double a = f.az[i], vh = f.vz[i] + hdt * a;
        f.z[i] = wrap_pos(f.z[i] + dt * vh, wb.lo[2], wb.hi[2], wb.L[2], wb.periodic[2]);
        f.vz[i] = vh + hdt * a;
    }
    {
        double d = f.du[i], uh = f.u[i] + hdt * d;
        f.u[i] = uh + hdt * d;
    }
}

// G5: v = v* + dt/2 (a_new - a_old) (same for u); a_old <- a_new is a swap of the two buffers on the host
// (adopt_new_acc). With ERR the kernel also reduces, per block
// and in a fixed order, the two quantities of the corrector check G6-G7 (reading A15):
// max |dv|^2 and sum |v^{n+1}|^2.
template <bool ERR>
__global__ void __launch_bounds__(256) k_correct(int64_t N, Fields f, const double* __restrict__ nax,
                                                 const double* __restrict__ nay, const double* __restrict__ naz,
                                                 const double* __restrict__ ndu, const double* __restrict__ dtp,
                                                 double* __restrict__ part_max, double* __restrict__ part_sum) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double d2 = 0.0, v2 = 0.0;
    if (i < N) {
        const double hdt = 0.5 * *dtp;
        double a, dv, v;
        a = nax[i]; dv = hdt * (a - f.ax[i]); v = f.vx[i] + dv; f.vx[i] = v; d2 = dv * dv; v2 = v * v;
        a = nay[i]; dv = hdt * (a - f.ay[i]); v = f.vy[i] + dv; f.vy[i] = v; d2 += dv * dv; v2 += v * v;
        a = naz[i]; dv = hdt * (a - f.az[i]); v = f.vz[i] + dv; f.vz[i] = v; d2 += dv * dv; v2 += v * v;
        a = ndu[i]; f.u[i] = f.u[i] + hdt * (a - f.du[i]);
    }
    if (ERR) {
        __shared__ double smax[8], ssum[8];
        d2 = warp_max(d2);
        v2 = warp_sum(v2);
        if (lane_id() == 0) { smax[threadIdx.x >> 5] = d2; ssum[threadIdx.x >> 5] = v2; }
        __syncthreads();
        if (threadIdx.x == 0) {
            double m = smax[0], t = ssum[0];
            for (int w = 1; w < 8; ++w) { m = fmax(m, smax[w]); t += ssum[w]; }
            part_max[blockIdx.x] = m;
            part_sum[blockIdx.x] = t;
        }
    }
}

// second stage of the corrector-check reduction: one block, fixed order (bitwise reproducible)
__global__ void __launch_bounds__(256) k_corr_final(int nblocks, const double* __restrict__ part_max,
                                                    const double* __restrict__ part_sum, DevScalars* sc) {
    __shared__ double smax[256], ssum[256];
    double m = 0.0, t = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += 256) { m = fmax(m, part_max[b]); t += part_sum[b]; }
    smax[threadIdx.x] = m; ssum[threadIdx.x] = t;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) {
            smax[threadIdx.x] = fmax(smax[threadIdx.x], smax[threadIdx.x + w]);
            ssum[threadIdx.x] += ssum[threadIdx.x + w];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { sc->corr_dvmax2 = smax[0]; sc->corr_v2sum = ssum[0]; }
}

__global__ void __launch_bounds__(256) k_hmax(int64_t N, const double* __restrict__ h, DevScalars* sc) {
    double v = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
        v = fmax(v, h[i]);
    v = warp_max(v);
    if (lane_id() == 0) atomicMax((unsigned long long*)&sc->h_max, (unsigned long long)__double_as_longlong(v));
}
__global__ void k_hmax_reset(DevScalars* sc) { sc->h_max = 0.0; }

__global__ void k_set_dt(double* dtp, DevScalars* sc, double user_dt, double cfl_mult) {
    const double dt = (user_dt > 0.0) ? user_dt : cfl_mult * sc->dt;       // G9: both terms of G8 are linear in the C's
    *dtp = dt;
    sc->t += dt;
}

int launch_predict(sph_ctx* c) {
    WrapBox wb;
    for (int k = 0; k < 3; ++k) {
        wb.lo[k] = c->box.lo[k]; wb.hi[k] = c->box.hi[k]; wb.L[k] = c->box.hi[k] - c->box.lo[k];
        wb.periodic[k] = c->box.periodic[k];
    }
    k_predict<<<div_up(c->N, 256), 256, 0, c->stream>>>(c->N, c->cur, wb, c->d_dtstep);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int launch_correct(sph_ctx* c, bool with_check) {
    const unsigned nb = div_up(c->N, 256);
    if (with_check) {
        k_correct<true><<<nb, 256, 0, c->stream>>>(c->N, c->cur, c->nax, c->nay, c->naz, c->ndu, c->d_dtstep, c->corr_part,
                                                   c->corr_part + nb);
        k_corr_final<<<1, 256, 0, c->stream>>>((int)nb, c->corr_part, c->corr_part + nb, c->d_sc);
        c->launches++;
    } else {
        k_correct<false><<<nb, 256, 0, c->stream>>>(c->N, c->cur, c->nax, c->nay, c->naz, c->ndu, c->d_dtstep, nullptr, nullptr);
    }
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    adopt_new_acc(c);
    return SPH_OK;
}

int launch_hmax(sph_ctx* c) {
    k_hmax_reset<<<1, 1, 0, c->stream>>>(c->d_sc);
    unsigned blocks = (unsigned)min((int64_t)148 * 4, (c->N + 255) / 256);
    k_hmax<<<blocks, 256, 0, c->stream>>>(c->N, c->cur.h, c->d_sc);
    c->launches += 2;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

// a^n <- a^{n+1}, du/dt^n <- du/dt^{n+1}: the buffers change places (nothing is copied; stream order keeps every
// kernel already enqueued on its own pointers)
void adopt_new_acc(sph_ctx* c) {
    std::swap(c->cur.ax, c->nax); std::swap(c->cur.ay, c->nay); std::swap(c->cur.az, c->naz);
    std::swap(c->cur.du, c->ndu);
}
int launch_adopt_acc(sph_ctx* c) {      // white step / standalone force evaluation: no velocity correction
    adopt_new_acc(c);
    return SPH_OK;
}

int launch_set_dt(sph_ctx* c, double user_dt) {
    k_set_dt<<<1, 1, 0, c->stream>>>(c->d_dtstep, c->d_sc, user_dt, c->cfl_mult);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
