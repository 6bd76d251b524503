// keys.cu -- a1: 63-bit Morton keys (3 x 21 bits) from fp64 positions (grid 2^21 per axis,
// PAPER.md:582; cube embedding, reading A1). HBM-bound: 24 B read + 12 B written per particle.
#include "common.cuh"

namespace sph {

// spread the low 21 bits of v so that bit i moves to bit 3 i
__device__ __forceinline__ uint64_t spread21(uint64_t v) {
    v &= 0x1fffffull;
    v = (v | (v << 32)) & 0x001f00000000ffffull;
    v = (v | (v << 16)) & 0x001f0000ff0000ffull;
    v = (v | (v << 8)) & 0x100f00f00f00f00full;
    v = (v | (v << 4)) & 0x10c30c30c30c30c3ull;
    v = (v | (v << 2)) & 0x1249249249249249ull;
    return v;
}

__device__ __forceinline__ uint64_t quantise(double x, double lo, double Lc) {
    // IEEE division (not a multiply by the reciprocal): the quantised cell decides integer results downstream
    double t = __ddiv_rn(__dsub_rn(x, lo), Lc);
    uint64_t v = 0;
    if (t > 0.0) {
        double g = floor(t * 2097152.0);   // exact scaling by 2^21
        v = (g >= 2097151.0) ? 2097151ull : (uint64_t)g;
    }
    return v;
}

__global__ void __launch_bounds__(256) k_morton(int64_t N, const double* __restrict__ x, const double* __restrict__ y,
                                                const double* __restrict__ z, double lox, double loy, double loz,
                                                double Lc, uint64_t keep, uint64_t* __restrict__ key, uint32_t* __restrict__ val) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    uint64_t X = quantise(x[i], lox, Lc), Y = quantise(y[i], loy, Lc), Z = quantise(z[i], loz, Lc);
    // X0 Y0 Z0 X1 Y1 Z1 ... with X0 the most significant: X bit j -> key bit 3 j + 2
    // keep = all ones, or the top 30 code bits only (morton_bits = 10: floor(t 2^10) = floor(t 2^21) >> 11 per axis)
    key[i] = ((spread21(X) << 2) | (spread21(Y) << 1) | spread21(Z)) & keep;
    val[i] = (uint32_t)i;
}

int launch_keys(sph_ctx* c) {
    double Lc = 0.0;
    for (int k = 0; k < 3; ++k) Lc = fmax(Lc, c->box.hi[k] - c->box.lo[k]);
    k_morton<<<div_up(c->N, 256), 256, 0, c->stream>>>(c->N, c->cur.x, c->cur.y, c->cur.z, c->box.lo[0], c->box.lo[1],
                                                       c->box.lo[2], Lc,
                                                       c->p.morton_bits == 10 ? ~((1ull << 33) - 1ull) : ~0ull, c->key, c->val);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
