// oracle/sph_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, single-threaded, fp64 restatement of what the SPH hot path of arXiv:2503.09713 ("The SHAMROCK
// code: I - SPH on GPUs", /root/reference/PAPER.md) computes. It exists only so that tests/, smoke() and
// bench.py's cpu_baseline / --impl reference legs can check and time the CUDA path against it. It shares no
// code with paper_2503_09713_b200/csrc and nothing in the product may call it.
//
// Build: g++ -std=c++17 -O2 -ffp-contract=off -fPIC -shared (see oracle/__init__.py). No FMA contraction, no
// fast-math, no threads. Every function cites the passage of PAPER.md it follows; where the paper is silent
// or garbled the reading of SURVEY.md 8(c) / DESIGN.md "Readings" (A1..A14, G1, G2) is taken and named.
//
// Parity pins (tests/test_oracle_*.py, -m "not gpu"): every function below is pinned by something other than
// itself -- worked examples printed in the paper (delta/prefix example PAPER.md:833-869, Table B2
// PAPER.md:899-907), brute force, closed forms (int W dV = 1, W(0) = 1/(pi h^3)), the unique-root bisection
// for h, conservation identities (sum m a = 0, sum m (v.a + du/dt) = 0), Galilean invariance, the exact
// Riemann solution for the Sod tube; the magnitudes the identities cannot see -- the 1/2 and v_sig of Eq. 5-6, the
// 1/2, beta_u and mean density of Eq. 8-9, F_ab(h_a) against F_ab(h_b), the force term and the pair maximum of G8 --
// by five two-particle cases worked by hand (tests/golden/pair_forces.txt). "parity unpinned": none.
//
// Layout convention: vectors are SoA, pos = x[0..N) y[0..N) z[0..N) contiguous (3N doubles).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <numeric>
#include <vector>

extern "C" {

struct orc_box {
    double lo[3], hi[3];
    int32_t periodic[3];
};

struct orc_params {
    double hfact;      // PAPER.md:1237 (h_fact = 1.2 for M4)
    double gamma;      // adiabatic index, P = (gamma-1) rho u
    double chi;        // tolerance 1.1
    double lambda;     // Newton clamp 1.2
    double eps_h;      // 1e-6 (north_star; eps_C not given)
    double alpha_av;   // constant alpha (reading A10)
    double beta_av;    // beta = 2
    double beta_u;     // conductivity
    double c_cour;     // 0.3
    double c_force;    // 0.25
    int32_t max_h_iter;
    int32_t max_restarts;
    int32_t eos;       // 0 adiabatic, 1 locally isothermal cs = cs0 (R/r0)^-q (BASELINE config 3)
    int32_t newton_literal;  // reading A5: 0 = exact derivative (3 rho(h)/h), 1 = Alg. 7 line 9 as printed
    double cs0, r0, q;
    double GM, soft;   // fixed softened point mass (BASELINE config 3); GM = 0 disables
    double centre[3];
    double eps_v;        // leapfrog corrector check G7: 1e-2 in the paper; 0 disables (reading A15)
    double lambda_stiff; // stiffness of the CFL multiplier G10; value not given, reading A16
    int32_t max_recycle; // cap on corrector re-cycles per step
    int32_t kernel;      // 0 = M4, 1 = M5, 2 = M6, 3-5 = Wendland C2, C4, C6 (informational here: the selector is orc_set_kernel)
    // shock switch (G11-G13; runscript constants PAPER.md:1412-1415; reading A18)
    double alpha_min, alpha_max, sigma_decay;
    int32_t av_switch;   // 0 = constant alpha_av (reading A10); 1 = per-particle alpha_a evolved by G13
    int32_t pad_;
};

}  // extern "C"

namespace {

// ---- O6: Schoenberg (1946) B-spline kernels M4 (cubic), M5 (quartic), M6 (quintic); the paper names them
// (M6 with h_fact = 1.0 in its physics tests) but prints neither f nor C_norm: textbook
// forms, q = r/h, 3-D normalisations 1/pi, 1/(20 pi), 1/(120 pi), support radii 2, 2.5, 3.
// The kernel in use is a file-level selector set through orc_set_kernel (test infrastructure, single-threaded);
// 0 = M4 (default), 1 = M5, 2 = M6.
// Wendland (1995) functions C2, C4, C6 (also named at PAPER.md:43, not printed either), 3 = C2, 4 = C4, 5 = C6: the 3-D
// forms on the support radius 2h, with t = 1 - q/2,
//   C2: f = t^4 (1 + 2q),                      C_norm = 21 / (16 pi)
//   C4: f = t^6 (1 + 3q + 35/12 q^2),          C_norm = 495 / (256 pi)
//   C6: f = t^8 (1 + 4q + 25/4 q^2 + 4 q^3),   C_norm = 1365 / (512 pi)
// (pins in tests/test_oracle_sph.py: unit volume integral, f(0) = 1, f' against finite differences of W.)
int g_kernel = 0;
#define kRkern (g_kernel == 1 ? 2.5 : g_kernel == 2 ? 3.0 : 2.0)
#define kInvPi 0.31830988618379067154
#define kCnorm (g_kernel == 0 ? kInvPi : g_kernel == 1 ? kInvPi / 20.0 : g_kernel == 2 ? kInvPi / 120.0 : \
                g_kernel == 3 ? kInvPi * 21.0 / 16.0 : g_kernel == 4 ? kInvPi * 495.0 / 256.0 : kInvPi * 1365.0 / 512.0)

inline double pw(double x, int n) { double r = 1.0; for (int i = 0; i < n; ++i) r *= x; return x > 0.0 ? r : 0.0; }

inline double f_m4(double q) {          // f(q) of the selected kernel (name kept from the M4-only version)
    if (g_kernel == 1) return pw(2.5 - q, 4) - 5.0 * pw(1.5 - q, 4) + 10.0 * pw(0.5 - q, 4);
    if (g_kernel == 2) return pw(3.0 - q, 5) - 6.0 * pw(2.0 - q, 5) + 15.0 * pw(1.0 - q, 5);
    if (g_kernel == 3) return pw(1.0 - 0.5 * q, 4) * (1.0 + 2.0 * q);
    if (g_kernel == 4) return pw(1.0 - 0.5 * q, 6) * (1.0 + 3.0 * q + 35.0 / 12.0 * q * q);
    if (g_kernel == 5) return pw(1.0 - 0.5 * q, 8) * (1.0 + 4.0 * q + 6.25 * q * q + 4.0 * q * q * q);
    if (q < 1.0) return 1.0 - 1.5 * q * q + 0.75 * q * q * q;
    if (q < 2.0) { double t = 2.0 - q; return 0.25 * t * t * t; }
    return 0.0;
}
inline double df_m4(double q) {         // f'(q)
    if (g_kernel == 1) return -4.0 * (pw(2.5 - q, 3) - 5.0 * pw(1.5 - q, 3) + 10.0 * pw(0.5 - q, 3));
    if (g_kernel == 2) return -5.0 * (pw(3.0 - q, 4) - 6.0 * pw(2.0 - q, 4) + 15.0 * pw(1.0 - q, 4));
    // product rule on t^n p(q), dt/dq = -1/2
    if (g_kernel == 3) return -2.0 * pw(1.0 - 0.5 * q, 3) * (1.0 + 2.0 * q) + 2.0 * pw(1.0 - 0.5 * q, 4);
    if (g_kernel == 4) return -3.0 * pw(1.0 - 0.5 * q, 5) * (1.0 + 3.0 * q + 35.0 / 12.0 * q * q) + pw(1.0 - 0.5 * q, 6) * (3.0 + 35.0 / 6.0 * q);
    if (g_kernel == 5) return -4.0 * pw(1.0 - 0.5 * q, 7) * (1.0 + 4.0 * q + 6.25 * q * q + 4.0 * q * q * q) +
                              pw(1.0 - 0.5 * q, 8) * (4.0 + 12.5 * q + 12.0 * q * q);
    if (q < 1.0) return -3.0 * q + 2.25 * q * q;
    if (q < 2.0) { double t = 2.0 - q; return -0.75 * t * t; }
    return 0.0;
}
// W = C h^-3 f(q)   (Eq. 2)
inline double W(double r, double h) { return kCnorm / (h * h * h) * f_m4(r / h); }
// F_ab(h) = r_hat . grad_a W = C h^-4 f'(q)   (Eq. 10)
inline double Fab(double r, double h) { return kCnorm / (h * h * h * h) * df_m4(r / h); }
// dW/dh = -C h^-4 [3 f(q) + q f'(q)]
inline double dWdh(double r, double h) {
    double q = r / h;
    return -kCnorm / (h * h * h * h) * (3.0 * f_m4(q) + q * df_m4(q));
}

// ---- minimum-image separation (reading A4): positions are kept wrapped into [lo,hi).
inline double min_image(double d, double L, int periodic) {
    if (periodic) {
        if (d > 0.5 * L) d -= L;
        else if (d < -0.5 * L) d += L;
    }
    return d;
}

struct Sep { double dx, dy, dz, d2; };
inline Sep separation(const double* x, const double* y, const double* z, int64_t a, int64_t b,
                      const orc_box& box) {
    Sep s;
    s.dx = min_image(x[a] - x[b], box.hi[0] - box.lo[0], box.periodic[0]);
    s.dy = min_image(y[a] - y[b], box.hi[1] - box.lo[1], box.periodic[1]);
    s.dz = min_image(z[a] - z[b], box.hi[2] - box.lo[2], box.periodic[2]);
    s.d2 = s.dx * s.dx + s.dy * s.dy + s.dz * s.dz;
    return s;
}

// gamma_o/o with the cache tolerance chi (App. E summary PAPER.md:1221; reading A2): strict <, self included.
inline bool interacts(double d2, double ha, double hb, double chi) {
    double rc = (kRkern * chi) * std::max(ha, hb);
    return d2 < rc * rc;
}

inline int clz64(uint64_t v) { return v ? __builtin_clzll(v) : 64; }
inline int clz32(uint32_t v) { return v ? __builtin_clz(v) : 32; }

// delta operator (Eq. B2) on the sorted list, with Karras' index tie-break for equal keys
// (reading O3): common-prefix length of the 96-bit strings (key, index).
inline int delta_idx(const uint64_t* k, int64_t i, int64_t j) {
    if (k[i] != k[j]) return clz64(k[i] ^ k[j]);
    return 64 + clz32((uint32_t)i ^ (uint32_t)j);
}

struct TreeOut {
    int32_t *left, *right;
    uint8_t *lflag, *rflag;
    int32_t *parent;   // [0,N-1): parent of internal node; [N-1, 2N-1): parent of leaf j at N-1+j; root: -1
    int32_t *rlo, *rhi;
};

// O3: radix tree from its recursive definition: the node covering the sorted range [i,j]
// splits where the first differing bit between its end keys changes; index convention of Table B2.
void build_node(const uint64_t* k, int64_t N, int64_t i, int64_t j, int32_t self, int32_t parent, TreeOut& t) {
    int d = delta_idx(k, i, j);
    // split: last index g in [i,j) whose key shares more than d leading bits with key_i
    int64_t g = i;
    for (int64_t s = i + 1; s < j; ++s)
        if (delta_idx(k, i, s) > d) g = s;
    t.rlo[self] = (int32_t)i;
    t.rhi[self] = (int32_t)j;
    t.parent[self] = parent;
    t.left[self] = (int32_t)g;
    t.right[self] = (int32_t)(g + 1);
    t.lflag[self] = (g == i);
    t.rflag[self] = (g + 1 == j);
    if (g == i) t.parent[N - 1 + g] = self; else build_node(k, N, i, g, (int32_t)g, self, t);
    if (g + 1 == j) t.parent[N - 1 + g + 1] = self; else build_node(k, N, g + 1, j, (int32_t)(g + 1), self, t);
}

struct Box6 { double lo[3], hi[3]; double hmax; };

Box6 node_box(int32_t node, bool leaf, const TreeOut& t, const double* x, const double* y, const double* z,
              const double* h, double* aabb, double* hmax) {
    Box6 b;
    if (leaf) {
        b.lo[0] = b.hi[0] = x[node]; b.lo[1] = b.hi[1] = y[node]; b.lo[2] = b.hi[2] = z[node];
        b.hmax = h[node];
        return b;
    }
    Box6 l = node_box(t.left[node], t.lflag[node], t, x, y, z, h, aabb, hmax);
    Box6 r = node_box(t.right[node], t.rflag[node], t, x, y, z, h, aabb, hmax);
    for (int c = 0; c < 3; ++c) { b.lo[c] = std::min(l.lo[c], r.lo[c]); b.hi[c] = std::max(l.hi[c], r.hi[c]); }
    b.hmax = std::max(l.hmax, r.hmax);
    for (int c = 0; c < 3; ++c) { aabb[6 * (int64_t)node + c] = b.lo[c]; aabb[6 * (int64_t)node + 3 + c] = b.hi[c]; }
    hmax[node] = b.hmax;
    return b;
}

// EOS (O8): adiabatic P = (gamma-1) rho u, cs = sqrt(gamma P / rho); locally isothermal P = cs(R)^2 rho.
inline void eos(const orc_params& p, double rho, double u, double x, double y, double& P, double& cs) {
    if (p.eos == 0) {
        P = (p.gamma - 1.0) * rho * u;
        cs = std::sqrt(p.gamma * P / rho);
    } else {
        double dx = x - p.centre[0], dy = y - p.centre[1];
        double R = std::sqrt(dx * dx + dy * dy);
        cs = p.cs0 * std::pow(R / p.r0, -p.q);
        P = cs * cs * rho;
    }
}

}  // namespace

extern "C" {

// ---- exported scalar kernel functions (pins: quadrature, continuity, W(0)) ----
void orc_set_kernel(int32_t k) { g_kernel = (k >= 1 && k <= 5) ? k : 0; }
double orc_f(double q) { return f_m4(q); }
double orc_df(double q) { return df_m4(q); }
double orc_W(double r, double h) { return W(r, h); }
double orc_F(double r, double h) { return Fab(r, h); }
double orc_dWdh(double r, double h) { return dWdh(r, h); }

// ---- O1: Morton keys (grid 2^21 per axis PAPER.md:582; cube embedding, reading A1).
// key bit (62-3j) = X bit (20-j), (61-3j) = Y, (60-3j) = Z, bit 63 = 0.
void orc_morton_keys(int64_t N, const double* pos, const orc_box* box, uint64_t* key) {
    double Lc = 0.0;
    for (int c = 0; c < 3; ++c) Lc = std::max(Lc, box->hi[c] - box->lo[c]);
    for (int64_t i = 0; i < N; ++i) {
        uint64_t X[3];
        for (int c = 0; c < 3; ++c) {
            double t = (pos[c * N + i] - box->lo[c]) / Lc;
            uint64_t v = 0;
            if (t > 0.0) {
                double g = std::floor(t * 2097152.0);
                v = (g >= 2097151.0) ? 2097151u : (uint64_t)g;
            }
            X[c] = v;
        }
        uint64_t m = 0;
        for (int j = 0; j < 21; ++j)      // j = 0 is the most significant coordinate bit (X0 of PAPER.md:827)
            for (int c = 0; c < 3; ++c) {
                uint64_t bit = (X[c] >> (20 - j)) & 1u;
                m |= bit << (62 - 3 * j - c);
            }
        key[i] = m;
    }
}

// The paper's 32-bit variant ("beta-bit" codes, 582 and 378: a 2^10 grid per axis, 30-bit codes): the same
// definition on the 2^beta grid, 1 <= beta <= 21; the code occupies the low 3 beta bits (X0 at bit 3 beta - 1).
void orc_morton_keys_beta(int64_t N, const double* pos, const orc_box* box, int32_t beta, uint64_t* key) {
    double Lc = 0.0;
    for (int c = 0; c < 3; ++c) Lc = std::max(Lc, box->hi[c] - box->lo[c]);
    const double ng = (double)(1ull << beta);
    for (int64_t i = 0; i < N; ++i) {
        uint64_t X[3];
        for (int c = 0; c < 3; ++c) {
            double t = (pos[c * N + i] - box->lo[c]) / Lc;
            uint64_t v = 0;
            if (t > 0.0) {
                double g = std::floor(t * ng);
                v = (g >= ng - 1.0) ? (uint64_t)(ng - 1.0) : (uint64_t)g;
            }
            X[c] = v;
        }
        uint64_t m = 0;
        for (int j = 0; j < beta; ++j)
            for (int c = 0; c < 3; ++c) {
                uint64_t bit = (X[c] >> (beta - 1 - j)) & 1u;
                m |= bit << (3 * beta - 1 - 3 * j - c);
            }
        key[i] = m;
    }
}

// worked example of PAPER.md:857-869 on beta-bit codes: delta, mask u << (beta - delta), prefix = a & mask.
int32_t orc_delta_beta(uint64_t a, uint64_t b, int32_t beta) {
    uint64_t xr = a ^ b;
    if (xr == 0) return beta;
    return clz64(xr) - (64 - beta);
}
uint64_t orc_prefix_mask(uint64_t a, uint64_t b, int32_t beta) {
    uint64_t u = (beta == 64) ? ~0ull : ((1ull << beta) - 1ull);
    int s = beta - orc_delta_beta(a, b, beta);
    return (s >= 64) ? 0 : ((u << s) & u);
}

// ---- O2: sort by key: stable => ties by ascending input index.
void orc_sort(int64_t N, const uint64_t* key, uint32_t* perm, uint64_t* sorted_key) {
    std::vector<uint32_t> p(N);
    std::iota(p.begin(), p.end(), 0u);
    std::stable_sort(p.begin(), p.end(), [&](uint32_t a, uint32_t b) { return key[a] < key[b]; });
    for (int64_t i = 0; i < N; ++i) { perm[i] = p[i]; sorted_key[i] = key[p[i]]; }
}

// ---- Alg. 1 (App. C1-C2): removal mask xi over the SORTED Morton codes.
// Lines 1-5: xi_i = (i == 0) or (m_i != m_{i-1}) (duplicates removed). Lines 6-22, n_red times: for every i,
// i_-1 and i_-2 are the two kept indices before i, i_+1 the kept index after it; with delta_0 = delta(mu_i, mu_i+1),
// delta_-1 = delta(mu_i-1, mu_i), delta_-2 = delta(mu_i-2, mu_i-1), the code stays kept unless
// delta_0 < delta_-1 and delta_-2 < delta_-1 (it is then the second leaf of a two-leaf parent).
// Readings (A17): "for i in parallel" is taken as a synchronous pass -- every i reads the mask as it was when
// the pass began; a neighbour that does not exist (i_-1, i_-2 < 0 or i_+1 >= n) gives delta = -1, Karras' convention
// for out-of-range indices; delta is the common-prefix length of the full 64-bit words (Eq. B2).
void orc_leaf_reduction(int64_t N, const uint64_t* skey, int32_t n_red, uint8_t* xi) {
    if (N < 1) return;
    for (int64_t i = 0; i < N; ++i) xi[i] = (i == 0) || (skey[i] != skey[i - 1]);        // l.1-5
    std::vector<uint8_t> old((size_t)N);
    for (int32_t pass = 0; pass < n_red; ++pass) {                                         // l.6
        std::memcpy(old.data(), xi, (size_t)N);
        for (int64_t i = 0; i < N; ++i) {                                                  // l.7
            int64_t im1 = i - 1;                                                           // l.8-10
            while (im1 >= 0 && !old[im1]) --im1;
            int64_t im2 = im1 - 1;                                                         // l.11-13
            while (im2 >= 0 && !old[im2]) --im2;
            int64_t ip1 = i + 1;                                                           // l.14-16
            while (ip1 < N && !old[ip1]) ++ip1;
            const int d0 = (ip1 < N) ? clz64(skey[i] ^ skey[ip1]) : -1;                    // l.17
            const int dm1 = (im1 >= 0) ? clz64(skey[im1] ^ skey[i]) : -1;                  // l.18
            const int dm2 = (im2 >= 0) ? clz64(skey[im2] ^ skey[im1]) : -1;                // l.19
            xi[i] = (!(d0 < dm1 && dm2 < dm1)) && old[i];                                  // l.20-22
        }
    }
}

// Stream compaction of the kept codes (Fig. D2): leaf codes mu_leaf and the index map id (the index
// of every kept code before compaction, closed by id[n_leaf] = N): leaf j holds the sorted objects [id_j, id_j+1)
// (Alg. 2). Returns n_leaf.
int64_t orc_leaf_compact(int64_t N, const uint64_t* skey, const uint8_t* xi, uint64_t* leaf_code, uint32_t* id_map) {
    int64_t n = 0;
    for (int64_t i = 0; i < N; ++i)
        if (xi[i]) { leaf_code[n] = skey[i]; id_map[n] = (uint32_t)i; ++n; }
    id_map[n] = (uint32_t)N;
    return n;
}

// ---- O3: radix tree tables (Table B2). Arrays of N-1 internal nodes; parent has 2N-1.
void orc_tree(int64_t N, const uint64_t* skey, int32_t* left, int32_t* right, uint8_t* lflag, uint8_t* rflag,
              int32_t* parent, int32_t* rlo, int32_t* rhi) {
    if (N < 2) { if (N == 1) parent[0] = -1; return; }
    TreeOut t{left, right, lflag, rflag, parent, rlo, rhi};
    build_node(skey, N, 0, N - 1, 0, -1, t);
}

// ---- O4: node boxes and hmax (tight boxes, PAPER.md:93 for hmax; north_star (3)). aabb: 6 per internal node
// (xmin,ymin,zmin,xmax,ymax,zmax); x,y,z,h in sorted order.
void orc_aabb(int64_t N, const int32_t* left, const int32_t* right, const uint8_t* lflag, const uint8_t* rflag,
              const double* x, const double* y, const double* z, const double* h, double* aabb, double* hmax) {
    if (N < 2) return;
    TreeOut t{(int32_t*)left, (int32_t*)right, (uint8_t*)lflag, (uint8_t*)rflag, nullptr, nullptr, nullptr};
    node_box(0, false, t, x, y, z, h, aabb, hmax);
}

// ---- O5: neighbour sets, plain definition, O(N^2). CSR, each list ascending. Returns the total; fills idx
// only if cap >= total.
int64_t orc_neighbours_brute(int64_t N, const double* pos, const double* h, const orc_box* box, double chi,
                             uint64_t* offs, uint32_t* idx, int64_t cap) {
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    int64_t total = 0;
    for (int64_t a = 0; a < N; ++a) {
        offs[a] = (uint64_t)total;
        for (int64_t b = 0; b < N; ++b) {
            Sep s = separation(x, y, z, a, b, *box);
            if (interacts(s.d2, h[a], h[b], chi)) {
                if (total < cap) idx[total] = (uint32_t)b;
                ++total;
            }
        }
    }
    offs[N] = (uint64_t)total;
    return total;
}

// Same sets through a uniform cell grid (validated against brute force in tests). For each a the grid gives
// G(a) = {b : d^2 < (R chi h_a)^2}; N(a) = G(a) U {b : a in G(b)} because (R chi max(ha,hb))^2 =
// max((R chi ha)^2, (R chi hb)^2) in floating point (squaring is monotone).
int64_t orc_neighbours_grid(int64_t N, const double* pos, const double* h, const orc_box* box, double chi,
                            uint64_t* offs, uint32_t* idx, int64_t cap) {
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    const double* P[3] = {x, y, z};
    double lo[3], L[3];
    for (int c = 0; c < 3; ++c) {
        if (box->periodic[c]) { lo[c] = box->lo[c]; L[c] = box->hi[c] - box->lo[c]; }
        else {
            double mn = std::numeric_limits<double>::infinity(), mx = -mn;
            for (int64_t i = 0; i < N; ++i) { mn = std::min(mn, P[c][i]); mx = std::max(mx, P[c][i]); }
            lo[c] = mn; L[c] = std::max(mx - mn, 1e-300) * (1.0 + 1e-9);
        }
    }
    // cell size ~ twice the median search radius, at most 128 cells per axis and at least 1
    std::vector<double> hs(h, h + N);
    std::nth_element(hs.begin(), hs.begin() + N / 2, hs.end());
    double cell = std::max(2.0 * kRkern * chi * hs[N / 2], 1e-300);
    int nc[3];
    for (int c = 0; c < 3; ++c) nc[c] = (int)std::min(128.0, std::max(1.0, std::floor(L[c] / cell)));
    auto cell_of = [&](int c, double v) {
        int k = (int)std::floor((v - lo[c]) / L[c] * nc[c]);
        return std::min(std::max(k, 0), nc[c] - 1);
    };
    int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
    std::vector<int64_t> start(ncell + 1, 0);
    std::vector<int64_t> cid(N);
    for (int64_t i = 0; i < N; ++i) {
        cid[i] = ((int64_t)cell_of(0, x[i]) * nc[1] + cell_of(1, y[i])) * nc[2] + cell_of(2, z[i]);
        ++start[cid[i] + 1];
    }
    for (int64_t c = 0; c < ncell; ++c) start[c + 1] += start[c];
    std::vector<uint32_t> order(N);
    { std::vector<int64_t> fill(start.begin(), start.end() - 1);
      for (int64_t i = 0; i < N; ++i) order[fill[cid[i]]++] = (uint32_t)i; }

    std::vector<std::vector<uint32_t>> lists(N);
    std::vector<int> cells[3];
    for (int64_t a = 0; a < N; ++a) {
        double ra = kRkern * chi * h[a];
        const double pa[3] = {x[a], y[a], z[a]};
        for (int c = 0; c < 3; ++c) {
            cells[c].clear();
            double w = L[c] / nc[c];
            int k0 = (int)std::floor((pa[c] - ra - lo[c]) / w) - 1;   // one spare cell each side
            int k1 = (int)std::floor((pa[c] + ra - lo[c]) / w) + 1;
            if (k1 - k0 + 1 >= nc[c]) { for (int k = 0; k < nc[c]; ++k) cells[c].push_back(k); }
            else for (int k = k0; k <= k1; ++k) {
                if (box->periodic[c]) cells[c].push_back(((k % nc[c]) + nc[c]) % nc[c]);
                else if (k >= 0 && k < nc[c]) cells[c].push_back(k);
            }
        }
        for (int i : cells[0]) for (int j : cells[1]) for (int k : cells[2]) {
            int64_t c = ((int64_t)i * nc[1] + j) * nc[2] + k;
            for (int64_t s = start[c]; s < start[c + 1]; ++s) {
                uint32_t b = order[s];
                Sep sp = separation(x, y, z, a, b, *box);
                if (sp.d2 < ra * ra) {                     // b in G(a)
                    lists[a].push_back(b);
                    if ((int64_t)b != a && !(sp.d2 < (kRkern * chi * h[b]) * (kRkern * chi * h[b])))
                        lists[b].push_back((uint32_t)a);   // a enters N(b) only through h_a
                }
            }
        }
    }
    int64_t total = 0;
    for (int64_t a = 0; a < N; ++a) {
        auto& l = lists[a];
        std::sort(l.begin(), l.end());
        l.erase(std::unique(l.begin(), l.end()), l.end());
        offs[a] = (uint64_t)total;
        for (uint32_t b : l) { if (total < cap) idx[total] = b; ++total; }
    }
    offs[N] = (uint64_t)total;
    return total;
}

// ---- O7: one pass of Alg. 7's inner loop for every particle over a given cache built
// with h^n = hn; per-particle stopping (reading A7); safeguard 2b (reading A5b). Then rho = m (hfact/h)^3
// (F1) and Omega (Eq. 7) at the final h. Returns the number of particles
// that exceeded chi h^n (eps = -1 in Alg. 7 l.15-17); -1 if max_h_iter was hit.
int64_t orc_density(int64_t N, const double* pos, const double* m, const double* hn, const uint64_t* offs,
                    const uint32_t* idx, const orc_box* box, const orc_params* p, double* h_out,
                    double* rho_out, double* omega_out, int32_t* iters_out, uint8_t* exceeded_out) {
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    int64_t n_exc = 0;
    bool noconv = false;
    for (int64_t a = 0; a < N; ++a) {
        double h = hn[a];
        bool exceeded = false, converged = false;
        int it = 0;
        auto sums = [&](double hh, double& rho_sum, double& S) {
            rho_sum = 0.0; S = 0.0;
            for (uint64_t s = offs[a]; s < offs[a + 1]; ++s) {
                uint32_t b = idx[s];
                double r = std::sqrt(separation(x, y, z, a, b, *box).d2);
                rho_sum += m[b] * W(r, hh);          // Eq. 1
                S += m[b] * dWdh(r, hh);
            }
        };
        while (it < p->max_h_iter) {
            ++it;
            double rho_sum, S;
            sums(h, rho_sum, S);
            double rho_h = m[a] * (p->hfact / h) * (p->hfact / h) * (p->hfact / h);   // F1
            double f = rho_sum - rho_h;                                               // F2
            double fp = S + 3.0 * (p->newton_literal ? rho_sum : rho_h) / h;          // Alg. 7 l.9 / A5
            double hnew = h - f / fp;                                                 // Alg. 7 l.10
            if (!(fp > 0.0) || (hnew - h) * f > 0.0 || !(hnew == hnew))               // 2b safeguard
                hnew = (f > 0.0) ? h / p->lambda : h * p->lambda;
            if (hnew > h * p->lambda) hnew = h * p->lambda;                           // Alg. 7 l.11-13
            else if (hnew < h / p->lambda) hnew = h / p->lambda;
            double eps = std::fabs(hnew - h) / hn[a];                                 // Alg. 7 l.14
            if (hnew > hn[a] * p->chi) { hnew = hn[a] * p->chi; exceeded = true; }    // Alg. 7 l.15-17
            h = hnew;
            if (exceeded) break;
            if (eps <= p->eps_h) { converged = true; break; }
        }
        if (!exceeded && !converged) noconv = true;
        double rho_sum, S;
        sums(h, rho_sum, S);
        double rho = m[a] * (p->hfact / h) * (p->hfact / h) * (p->hfact / h);
        h_out[a] = h;
        rho_out[a] = rho;
        omega_out[a] = 1.0 + h / (3.0 * rho) * S;    // Eq. 7 with dh/drho = -h/(3 rho) from F1
        if (iters_out) iters_out[a] = it;
        if (exceeded_out) exceeded_out[a] = exceeded;
        n_exc += exceeded;
    }
    return noconv ? -1 : n_exc;
}

// Pin for O7: h_a as the unique root of g_a(h) = sum_b m_b C f(r_ab/h) - m_a hfact^3 (reading A5b), found by
// plain bisection over ALL particles (no cache, no Newton).
void orc_h_bisect(int64_t N, const double* pos, const double* m, const orc_box* box, double hfact,
                  const double* h_lo, const double* h_hi, double* h_out) {
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    std::vector<double> r(N);
    for (int64_t a = 0; a < N; ++a) {
        for (int64_t b = 0; b < N; ++b) r[b] = std::sqrt(separation(x, y, z, a, b, *box).d2);
        auto g = [&](double h) {
            double s = 0.0;
            for (int64_t b = 0; b < N; ++b) s += m[b] * kCnorm * f_m4(r[b] / h);
            return s - m[a] * hfact * hfact * hfact;
        };
        double lo = h_lo[a], hi = h_hi[a];
        for (int it = 0; it < 200; ++it) {
            double mid = 0.5 * (lo + hi);
            if (mid == lo || mid == hi) break;
            if (g(mid) > 0.0) hi = mid; else lo = mid;
        }
        h_out[a] = 0.5 * (lo + hi);
    }
}

// ---- Shock switch (G11-G13). The paper gives the implicit update G13 and the runscript constants
// (alpha_min = 0, alpha_max = 1, sigma_decay = 0.1) but neither alpha_loc nor tau: it defers to
// Price et al. (2018) Sect. 2.2.9, which is not in /root/reference. Reading A18 restates that section as far
// as this build could: with the SPH first-derivative estimate of any field f at particle a,
//     d_j f |_a = -(1 / (Omega_a rho_a)) sum_b m_b (f_a - f_b) r_hat_j F_ab(h_a),
//   div v, curl v and the tensor d_j v_i from v* (G12), div a from a^n,
//   d(div v)/dt = div a - sum_ij (d_j v_i)(d_i v_j),
//   xi = (div v)^2 / ((div v)^2 + |curl v|^2)   (1 if both vanish),
//   A = xi max(-d(div v)/dt, 0),  alpha_loc = min(max(10 h^2 A / c_s^2, alpha_min), alpha_max)
//       (c_s = 0: alpha_max if A > 0, else alpha_min),
//   tau = h / (sigma_decay c_s)   (c_s = 0: no decay),
//   G13: alpha^{n+1} = max((alpha^n + alpha_loc dt/tau) / (1 + dt/tau), alpha_loc).
// Outputs: alpha_out; divv_out, curlv_out (|curl v|), aloc_out may be null.
void orc_alpha_update(int64_t N, const double* pos, const double* vel, const double* acc, const double* m,
                      const double* h, const double* rho, const double* omega, const double* u, const uint64_t* offs,
                      const uint32_t* idx, const orc_box* box, const orc_params* p, double dt, const double* alpha_in,
                      double* alpha_out, double* divv_out, double* curlv_out, double* aloc_out) {
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    for (int64_t a = 0; a < N; ++a) {
        double gv[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};   // gv[i][j] = d_j v_i
        double diva = 0.0;
        for (uint64_t s = offs[a]; s < offs[a + 1]; ++s) {
            uint32_t b = idx[s];
            if ((int64_t)b == a) continue;
            Sep sp = separation(x, y, z, a, b, *box);
            double r = std::sqrt(sp.d2);
            if (!(r > 0.0)) continue;
            const double rh[3] = {sp.dx / r, sp.dy / r, sp.dz / r};
            const double Fa = Fab(r, h[a]);
            for (int i = 0; i < 3; ++i) {
                const double dv = vel[i * N + a] - vel[i * N + b];
                for (int j = 0; j < 3; ++j) gv[i][j] += m[b] * dv * rh[j] * Fa;
                diva += m[b] * (acc[i * N + a] - acc[i * N + b]) * rh[i] * Fa;
            }
        }
        const double norm = -1.0 / (omega[a] * rho[a]);
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) gv[i][j] *= norm;
        diva *= norm;
        const double divv = gv[0][0] + gv[1][1] + gv[2][2];
        const double cx = gv[2][1] - gv[1][2], cy = gv[0][2] - gv[2][0], cz = gv[1][0] - gv[0][1];
        const double curl2 = cx * cx + cy * cy + cz * cz;
        double trs = 0.0;
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) trs += gv[i][j] * gv[j][i];
        const double ddivdt = diva - trs;
        const double den = divv * divv + curl2;
        const double xi = den > 0.0 ? divv * divv / den : 1.0;
        const double A = xi * std::max(-ddivdt, 0.0);
        double P, cs;
        eos(*p, rho[a], u[a], x[a], y[a], P, cs);
        double aloc;
        if (cs > 0.0) aloc = std::min(std::max(10.0 * h[a] * h[a] * A / (cs * cs), p->alpha_min), p->alpha_max);
        else aloc = A > 0.0 ? p->alpha_max : p->alpha_min;
        const double xdt = cs > 0.0 ? dt * p->sigma_decay * cs / h[a] : 0.0;                  // dt / tau
        alpha_out[a] = std::max((alpha_in[a] + aloc * xdt) / (1.0 + xdt), aloc);                // G13
        if (divv_out) divv_out[a] = divv;
        if (curlv_out) curlv_out[a] = std::sqrt(curl2);
        if (aloc_out) aloc_out[a] = aloc;
    }
}

// per-particle alpha for the next orc_forces call (null = the constant p->alpha_av of reading A10); test infrastructure,
// single-threaded: a file-level selector like the kernel choice
const double* g_alpha = nullptr;
void orc_set_alpha(const double* alpha) { g_alpha = alpha; }

// ---- O8 + O9: forces (Eq. 3-6, 8-10; minus sign G1, q inside the sum G2), per-particle CFL
// candidates (G8; v_sig^dt reading A12) and their global minimum.
double orc_forces(int64_t N, const double* pos, const double* vel, const double* m, const double* h,
                  const double* rho, const double* omega, const double* u, const uint64_t* offs,
                  const uint32_t* idx, const orc_box* box, const orc_params* p, double* acc, double* dudt) {
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    const double *vx = vel, *vy = vel + N, *vz = vel + 2 * N;
    std::vector<double> P(N), cs(N);
    for (int64_t a = 0; a < N; ++a) eos(*p, rho[a], u[a], x[a], y[a], P[a], cs[a]);
    double dt_min = std::numeric_limits<double>::infinity();
    for (int64_t a = 0; a < N; ++a) {
        double ax = 0.0, ay = 0.0, az = 0.0, du = 0.0;
        double vsig_dt = cs[a];
        for (uint64_t s = offs[a]; s < offs[a + 1]; ++s) {
            uint32_t b = idx[s];
            if ((int64_t)b == a) continue;
            Sep sp = separation(x, y, z, a, b, *box);
            double r = std::sqrt(sp.d2);
            if (!(r > 0.0)) continue;                       // coincident particles: r_hat undefined
            double rx = sp.dx / r, ry = sp.dy / r, rz = sp.dz / r;
            double dvx = vx[a] - vx[b], dvy = vy[a] - vy[b], dvz = vz[a] - vz[b];
            double w = dvx * rx + dvy * ry + dvz * rz;      // v_ab . r_hat_ab
            double vsa = (g_alpha ? g_alpha[a] : p->alpha_av) * cs[a] + p->beta_av * std::fabs(w);   // Eq. 6
            double vsb = (g_alpha ? g_alpha[b] : p->alpha_av) * cs[b] + p->beta_av * std::fabs(w);
            double qa = (w < 0.0) ? -0.5 * rho[a] * vsa * w : 0.0;          // Eq. 5
            double qb = (w < 0.0) ? -0.5 * rho[b] * vsb * w : 0.0;
            double Fa = Fab(r, h[a]), Fb = Fab(r, h[b]);                    // Eq. 10
            double ta = (P[a] + qa) / (rho[a] * rho[a] * omega[a]);
            double tb = (P[b] + qb) / (rho[b] * rho[b] * omega[b]);
            double coef = m[b] * (ta * Fa + tb * Fb);
            ax -= coef * rx; ay -= coef * ry; az -= coef * rz;              // Eq. 3 (with G1's minus sign)
            du += m[b] * ta * w * Fa;                                       // Eq. 4 (G2: inside the sum)
            if (p->eos == 0 && p->beta_u != 0.0) {
                double vsu = std::sqrt(std::fabs(P[a] - P[b]) / (0.5 * (rho[a] + rho[b])));   // Eq. 9
                du += m[b] * p->beta_u * vsu * (u[a] - u[b]) * 0.5 *
                      (Fa / (omega[a] * rho[a]) + Fb / (omega[b] * rho[b]));                  // Eq. 8
            }
            if (r < kRkern * std::max(h[a], h[b])) vsig_dt = std::max(vsig_dt, vsa);           // A12
        }
        if (p->GM != 0.0) {                                 // fixed softened point mass (config 3)
            double dx = x[a] - p->centre[0], dy = y[a] - p->centre[1], dz = z[a] - p->centre[2];
            double d2 = dx * dx + dy * dy + dz * dz + p->soft * p->soft;
            double inv = p->GM / (d2 * std::sqrt(d2));
            ax -= inv * dx; ay -= inv * dy; az -= inv * dz;
        }
        if (p->eos != 0) du = 0.0;
        acc[a] = ax; acc[N + a] = ay; acc[2 * N + a] = az;
        dudt[a] = du;
        double an = std::sqrt(ax * ax + ay * ay + az * az);
        double dta = p->c_cour * h[a] / vsig_dt;                            // G8
        if (an > 0.0) dta = std::min(dta, p->c_force * std::sqrt(h[a] / an));
        dt_min = std::min(dt_min, dta);
    }
    return dt_min;
}

// ---- single evaluation: neighbours at h^n -> Alg. 7 with chi-restarts (outer while) ->
// forces. h is in/out (h^n in, converged h out). mode 0 = brute-force neighbour search, 1 = cell grid.
// Returns restarts >= 0, or -1 (h iteration cap), -2 (restart cap). If offs_out/idx_out are non-null and
// cap suffices they receive the final cache.
// alpha (may be null): per-particle shock-switch alpha, in/out; a_prev = a^n (null: zeros) and dt_alpha = the step's dt
// enter G12-G13, evaluated between the smoothing-length update and the derivatives (Fig. G1).
static int32_t evaluate_impl(int64_t N, const double* pos, const double* vel, const double* m, const double* u,
                             double* h, const orc_box* box, const orc_params* p, int32_t mode, double* rho,
                             double* omega, double* acc, double* dudt, double* dt_out, int64_t* n_neigh_out,
                             std::vector<uint64_t>& offs, std::vector<uint32_t>& idx, double* alpha = nullptr,
                             const double* a_prev = nullptr, double dt_alpha = 0.0) {
    offs.assign(N + 1, 0);
    idx.clear();
    std::vector<double> hn(h, h + N), hnew(N);
    int32_t restarts = 0;
    for (;;) {
        auto search = mode ? orc_neighbours_grid : orc_neighbours_brute;
        int64_t total = search(N, pos, hn.data(), box, p->chi, offs.data(), nullptr, 0);
        idx.resize(total);
        search(N, pos, hn.data(), box, p->chi, offs.data(), idx.data(), total);
        int64_t ne = orc_density(N, pos, m, hn.data(), offs.data(), idx.data(), box, p, hnew.data(), rho, omega,
                                 nullptr, nullptr);
        if (ne < 0) return -1;
        if (ne == 0) break;
        hn = hnew;                      // h^n <- current h for all particles, rebuild, rerun
        if (++restarts > p->max_restarts) return -2;
    }
    std::memcpy(h, hnew.data(), N * sizeof(double));
    if (p->av_switch && alpha) {
        std::vector<double> zeros, anew(N);
        if (!a_prev) { zeros.assign(3 * N, 0.0); a_prev = zeros.data(); }
        orc_alpha_update(N, pos, vel, a_prev, m, h, rho, omega, u, offs.data(), idx.data(), box, p, dt_alpha, alpha,
                         anew.data(), nullptr, nullptr, nullptr);
        std::memcpy(alpha, anew.data(), N * sizeof(double));
        g_alpha = alpha;
    }
    double dt = orc_forces(N, pos, vel, m, h, rho, omega, u, offs.data(), idx.data(), box, p, acc, dudt);
    g_alpha = nullptr;
    if (dt_out) *dt_out = dt;
    if (n_neigh_out) *n_neigh_out = (int64_t)idx.size();
    return restarts;
}

int32_t orc_evaluate(int64_t N, const double* pos, const double* vel, const double* m, const double* u,
                     double* h, const orc_box* box, const orc_params* p, int32_t mode, double* rho,
                     double* omega, double* acc, double* dudt, double* dt_out, int64_t* n_neigh_out) {
    std::vector<uint64_t> offs;
    std::vector<uint32_t> idx;
    return evaluate_impl(N, pos, vel, m, u, h, box, p, mode, rho, omega, acc, dudt, dt_out, n_neigh_out, offs, idx);
}
// the same with the shock switch: alpha in/out (white step: a^n = 0, dt = 0, so alpha rises to alpha_loc at once)
int32_t orc_evaluate_alpha(int64_t N, const double* pos, const double* vel, const double* m, const double* u,
                           double* h, const orc_box* box, const orc_params* p, int32_t mode, double* rho,
                           double* omega, double* acc, double* dudt, double* dt_out, int64_t* n_neigh_out, double* alpha) {
    std::vector<uint64_t> offs;
    std::vector<uint32_t> idx;
    return evaluate_impl(N, pos, vel, m, u, h, box, p, mode, rho, omega, acc, dudt, dt_out, n_neigh_out, offs, idx, alpha);
}

// ---- O10: one leapfrog KDK step (G1-G5; order of Fig. G1; u integrated
// like v, reading A13). State in/out: pos, vel, u, h, acc, dudt (a^n, du/dt^n on entry; ^{n+1} on exit).
// Returns restarts or a negative error like orc_evaluate; dt_next receives the CFL dt for the next step (A14).
//
// Corrector check and re-cycle (G6-G7), only if p->eps_v > 0. Reading A15: G7 as printed divides
// max|dv| by the rms of dv itself, which is >= 1 for any data and can never be below eps_v = 1e-2; the check is
// taken as in Phantom (which the paper says it follows): err = max_i |dv_i| / sqrt((1/N) sum_j |v_j^{n+1}|^2), 0 if
// all velocities vanish. While err >= eps_v (at most max_recycle times): the acceleration is recalculated with
// v* <- v^{n+1} (and u* <- u^{n+1}) on the same positions, h, rho, Omega and neighbour cache, and the correction
// dv = dt/2 (a_new - a_previous) is applied again. CFL multiplier (G9-G10): *cfl_mult is
// halved after a step that re-cycled, else relaxed by (1 + stiff * mult) / (1 + stiff) (reading A16: lambda_stiff is
// not given in the paper; it is a parameter); dt_next = mult * G8, as both terms of G8 are linear in the C's.
static int32_t step_impl(int64_t N, double* pos, double* vel, const double* m, double* u, double* h, double* acc,
                         double* dudt, const orc_box* box, const orc_params* p, int32_t mode, double dt, double* rho,
                         double* omega, double* dt_next, double* cfl_mult, int32_t* n_recycle, double* alpha) {
    std::vector<double> a_old(acc, acc + 3 * N), du_old(dudt, dudt + N);
    for (int c = 0; c < 3; ++c) {
        double L = box->hi[c] - box->lo[c];
        for (int64_t i = 0; i < N; ++i) {
            double vh = vel[c * N + i] + 0.5 * dt * a_old[c * N + i];        // G1
            double r = pos[c * N + i] + dt * vh;                            // G2
            if (box->periodic[c]) {                                         // wrap into [lo,hi)
                if (r >= box->hi[c]) r -= L;
                else if (r < box->lo[c]) r += L;
                if (r >= box->hi[c]) r = box->lo[c];                        // r + L rounding up to hi
            }
            pos[c * N + i] = r;
            vel[c * N + i] = vh + 0.5 * dt * a_old[c * N + i];              // G3
        }
    }
    for (int64_t i = 0; i < N; ++i) {
        double uh = u[i] + 0.5 * dt * du_old[i];
        u[i] = uh + 0.5 * dt * du_old[i];
    }
    std::vector<uint64_t> offs;
    std::vector<uint32_t> idx;
    double dt_raw = 0.0;
    int32_t rc = evaluate_impl(N, pos, vel, m, u, h, box, p, mode, rho, omega, acc, dudt, &dt_raw, nullptr, offs, idx,
                               alpha, a_old.data(), dt);   // G4 (with G12-G13 before it if the switch is on)
    if (rc < 0) return rc;
    int32_t recycles = 0;
    for (;;) {
        double dvmax2 = 0.0, v2sum = 0.0;
        for (int64_t i = 0; i < N; ++i) {
            double d2 = 0.0, v2 = 0.0;
            for (int c = 0; c < 3; ++c) {
                const double dv = 0.5 * dt * (acc[c * N + i] - a_old[c * N + i]);                                 // G5, G6
                vel[c * N + i] = vel[c * N + i] + dv;
                d2 += dv * dv;
                v2 += vel[c * N + i] * vel[c * N + i];
            }
            dvmax2 = std::max(dvmax2, d2);
            v2sum += v2;
            u[i] = u[i] + 0.5 * dt * (dudt[i] - du_old[i]);
        }
        if (!(p->eps_v > 0.0) || recycles >= p->max_recycle) break;
        const double vrms = std::sqrt(v2sum / (double)N);
        const double err = vrms > 0.0 ? std::sqrt(dvmax2) / vrms : 0.0;                                           // G7 (A15)
        if (err < p->eps_v) break;
        ++recycles;
        a_old.assign(acc, acc + 3 * N);
        du_old.assign(dudt, dudt + N);
        if (p->av_switch && alpha) g_alpha = alpha;      // alpha is not evolved again within a step
        dt_raw = orc_forces(N, pos, vel, m, h, rho, omega, u, offs.data(), idx.data(), box, p, acc, dudt);
        g_alpha = nullptr;
    }
    double mult = cfl_mult ? *cfl_mult : 1.0;
    if (p->eps_v > 0.0) {
        mult = recycles > 0 ? 0.5 * mult : (1.0 + p->lambda_stiff * mult) / (1.0 + p->lambda_stiff);              // G9-G10
        if (cfl_mult) *cfl_mult = mult;
    }
    if (dt_next) *dt_next = mult * dt_raw;
    if (n_recycle) *n_recycle = recycles;
    return rc;
}

int32_t orc_step2(int64_t N, double* pos, double* vel, const double* m, double* u, double* h, double* acc,
                  double* dudt, const orc_box* box, const orc_params* p, int32_t mode, double dt, double* rho,
                  double* omega, double* dt_next, double* cfl_mult, int32_t* n_recycle) {
    return step_impl(N, pos, vel, m, u, h, acc, dudt, box, p, mode, dt, rho, omega, dt_next, cfl_mult, n_recycle, nullptr);
}
int32_t orc_step3(int64_t N, double* pos, double* vel, const double* m, double* u, double* h, double* acc,
                  double* dudt, const orc_box* box, const orc_params* p, int32_t mode, double dt, double* rho,
                  double* omega, double* dt_next, double* cfl_mult, int32_t* n_recycle, double* alpha) {
    return step_impl(N, pos, vel, m, u, h, acc, dudt, box, p, mode, dt, rho, omega, dt_next, cfl_mult, n_recycle, alpha);
}

int32_t orc_step(int64_t N, double* pos, double* vel, const double* m, double* u, double* h, double* acc,
                 double* dudt, const orc_box* box, const orc_params* p, int32_t mode, double dt, double* rho,
                 double* omega, double* dt_next) {
    orc_params q = *p;
    q.eps_v = 0.0;                                   // the plain step of G1-G5: no corrector check
    return orc_step2(N, pos, vel, m, u, h, acc, dudt, box, &q, mode, dt, rho, omega, dt_next, nullptr, nullptr);
}

}  // extern "C"
