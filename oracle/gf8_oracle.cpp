// gf8_oracle.cpp -- the CPU oracle for the GeoFP8 codec hot path (arXiv 2607.07494).
//
// TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load this.  The product (paper_2607_07494_b200/) never links, imports
// or calls it, and shares no code, table, header or constant generator with it.
//
// Plain, slow, double-precision C++17.  Every function follows the paper's statement of the
// operation (PAPER.md line cited) or, where the paper is silent, the reading listed in
// DESIGN.md "Readings" (S1..S15).  No blocking, fusion or reordering beyond the formula; OpenMP is
// used only as `parallel for` over independent output rows.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"):
//   FP8 tables        exhaustive closed form, encode(decode(c))==c, midpoints-to-even, saturation
//   quantizer         amax*scale lands on fmax; |err| <= half a code step; zero tensor
//   whitening         round trip, T A_bar T = rho I, explicit Kronecker product (Eq. 7-10, 15),
//                     k=d vs Cholesky form of Eq. 14, dense == low-rank
//   identity factors  codec == Euclidean FP8 bit for bit
//   Jacobi / subspace residuals, trace, 2x2 closed form, exact-rank-k one-step, brute force
//   factor            symmetry, trace, convergence to the generating covariance
//   reduce            == mean of per-rank dequantisation; R=1 == dequantise
//   sync scale / hits own amax == plain quantizer; doubled amax halves every value; hand-worked hit counts
//                     (tests/golden/boundary_hits_example.txt); counts against the decoded table
//   error feedback    zero residual == plain quantizer; worked example (tests/golden/ef_worked_example.txt); the
//                     telescoping identity sum deq_t = sum u_t + R_0 - R_T; |R| <= half the widest code gap
// Parity unpinned: the paper's printed Table I / II values (they need the authors' gradients).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#include <limits>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

// ------------------------------------------------------------------------------------------------
// O4 / S7.  FP8 formats of ref [24], cited by PAPER.md:23 "FP8 format".
//   fmt 0 = E4M3: 1-4-3, bias 7, no infinities, NaN = S.1111.111, subnormal step 2^-9, max 448.
//   fmt 1 = E5M2: 1-5-2, bias 15, IEEE-like inf / NaN, subnormal step 2^-16, max 57344.
// ------------------------------------------------------------------------------------------------
static inline int fmt_mbits(int fmt) { return fmt == 0 ? 3 : 2; }
static inline int fmt_bias(int fmt)  { return fmt == 0 ? 7 : 15; }

double gf8o_fp8_max(int fmt) { return fmt == 0 ? 448.0 : 57344.0; }

// Value of one code, from the format definition (sign, exponent field, mantissa field).
double gf8o_fp8_to_double(int fmt, uint8_t c) {
    const int p = fmt_mbits(fmt), bias = fmt_bias(fmt);
    const int s = c >> 7;
    const int e = (c & 0x7F) >> p;
    const int m = c & ((1 << p) - 1);
    const int emax = fmt == 0 ? 15 : 31;
    double v;
    if (fmt == 0 && e == emax && m == 7) v = std::numeric_limits<double>::quiet_NaN();
    else if (fmt == 1 && e == emax) v = (m == 0) ? std::numeric_limits<double>::infinity()
                                                 : std::numeric_limits<double>::quiet_NaN();
    else if (e == 0) v = std::ldexp((double)m, 1 - bias - p);               // subnormal
    else v = std::ldexp(1.0 + (double)m / (double)(1 << p), e - bias);      // normal
    return s ? -v : v;
}

// Round-to-nearest, ties to even integer, written out (independent of the FP environment).
static inline double rne_int(double x) {
    double f = std::floor(x), r = x - f;
    if (r > 0.5) return f + 1.0;
    if (r < 0.5) return f;
    return (std::fmod(f, 2.0) == 0.0) ? f : f + 1.0;
}

// FP32 -> FP8, round to nearest even, saturate to +-max finite (infinity is never produced);
// NaN in -> NaN code (0x7F); -0 keeps its sign.  (S7, S13)
uint8_t gf8o_fp8_from_float(int fmt, float y) {
    const int p = fmt_mbits(fmt), bias = fmt_bias(fmt);
    if (std::isnan(y)) return 0x7F;
    const uint8_t sign = std::signbit(y) ? 0x80 : 0x00;
    double a = std::fabs((double)y);
    const double fmax = gf8o_fp8_max(fmt);
    if (a > fmax) a = fmax;                         // includes +-inf
    if (a == 0.0) return sign;
    int e;                                           // a = f * 2^e, f in [0.5,1)  =>  floor(log2 a) = e-1
    (void)std::frexp(a, &e);
    int E = e - 1;
    if (E < 1 - bias) E = 1 - bias;                  // subnormal range shares the min-normal quantum
    const double quantum = std::ldexp(1.0, E - p);
    double q = rne_int(a / quantum);                 // exact division by a power of two
    double v = q * quantum;
    if (v > fmax) v = fmax;                          // rounded up past the largest finite value
    if (v == 0.0) return sign;
    (void)std::frexp(v, &e);
    E = e - 1;
    int ef, mf;
    if (E < 1 - bias) { ef = 0; mf = (int)std::ldexp(v, bias - 1 + p); }
    else { ef = E + bias; mf = (int)((std::ldexp(v, -E) - 1.0) * (double)(1 << p)); }
    return (uint8_t)(sign | (ef << p) | mf);
}

// ------------------------------------------------------------------------------------------------
// O4.  Quantize (Eq. 16 "scaling, FP8 quantization"; Alg. 1 l.12-13; S6, S13).
//   x        m x n FP32 row-major (already rounded from double by the caller: x = (float)W~)
//   scaling  0 = one scale per tensor, 1 = one per 128x128 block (edge blocks partial)
//   amax     = largest |x| taken on the bit pattern (NaN / inf dominate, order independent)
//   scale    = fmax / amax, scale_inv = amax / fmax, each ONE IEEE FP32 division;
//              amax == 0, amax not finite, or scale not finite  =>  scale = scale_inv = 1
//   code     = rne_sat_fp8(x * scale), one FP32 multiply
// ------------------------------------------------------------------------------------------------
static inline uint32_t f2u(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }
static inline float u2f(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }

static void quantize_region(int fmt, const float* x, int64_t ld, int64_t r0, int64_t r1, int64_t c0,
                            int64_t c1, uint8_t* codes, float* scale_inv_out) {
    uint32_t ab = 0;
    for (int64_t i = r0; i < r1; ++i)
        for (int64_t j = c0; j < c1; ++j) ab = std::max(ab, f2u(x[i * ld + j]) & 0x7FFFFFFFu);
    const float amax = u2f(ab);
    const float fmax = (float)gf8o_fp8_max(fmt);
    float scale = fmax / amax, scale_inv = amax / fmax;
    if (amax == 0.0f || !std::isfinite(amax) || !std::isfinite(scale)) { scale = 1.0f; scale_inv = 1.0f; }
    for (int64_t i = r0; i < r1; ++i)
        for (int64_t j = c0; j < c1; ++j) {
            volatile float y = x[i * ld + j] * scale;      // one FP32 multiply, kept in FP32
            codes[i * ld + j] = gf8o_fp8_from_float(fmt, y);
        }
    *scale_inv_out = scale_inv;
}

void gf8o_quantize(int fmt, int scaling, const float* x, int64_t m, int64_t n, uint8_t* codes,
                   float* scale_inv) {
    if (scaling == 0) { quantize_region(fmt, x, n, 0, m, 0, n, codes, scale_inv); return; }
    const int64_t bm = (m + 127) / 128, bn = (n + 127) / 128;
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < bm * bn; ++b) {
        const int64_t bi = b / bn, bj = b % bn;
        quantize_region(fmt, x, n, bi * 128, std::min(m, bi * 128 + 128), bj * 128,
                        std::min(n, bj * 128 + 128), codes, scale_inv + b);
    }
}

// ------------------------------------------------------------------------------------------------
// O5.  Reduce (Eq. 1; Alg. 1 l.20-21; S8: every payload carries its own scale and is
// dequantised to FP32 before summation).  FP32, rank order, fused multiply-add, then * (1/R).
// ------------------------------------------------------------------------------------------------
void gf8o_reduce(int fmt, int scaling, const uint8_t* const* codes, const float* const* scale_inv,
                 int R, int average, int64_t m, int64_t n, float* out) {
    const int64_t bn = (n + 127) / 128;
    const float invR = 1.0f / (float)R;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < m; ++i)
        for (int64_t j = 0; j < n; ++j) {
            const int64_t sidx = scaling == 0 ? 0 : (i / 128) * bn + (j / 128);
            float acc = 0.0f;
            for (int r = 0; r < R; ++r)
                acc = std::fmaf((float)gf8o_fp8_to_double(fmt, codes[r][i * n + j]), scale_inv[r][sidx], acc);
            if (average) { volatile float t = acc * invR; acc = t; }
            out[i * n + j] = acc;
        }
}

// ------------------------------------------------------------------------------------------------
// O8.  Error feedback in the transformed coordinates (PAPER.md:318 Alg. 1 l.11-15; :354; S10).
// Per tensor and per rank a residual buffer R (same shape as the gradient, FP32, zero at start):
//     U~   = U + R                         (l.11; U is the whitened gradient, the FP32 tensor O4 would quantize)
//     s    = Scale(U~), Q~ = Q(U~; s)      (l.12-13: O4 on U~)
//     deq  = Dequantize(Q~; s)             (l.14: val(code) * scale_inv)
//     R   <- U~ - deq                      (l.15)
// Each line is ONE IEEE FP32 operation per element (add; O4; multiply; subtract), no contraction -- the
// residual is state carried from step to step, so both sides have to round it the same way.
// ------------------------------------------------------------------------------------------------
void gf8o_ef_quantize(int fmt, int scaling, const float* u, float* resid, int64_t m, int64_t n, uint8_t* codes,
                      float* scale_inv) {
    std::vector<float> ut((size_t)(m * n));
    for (int64_t i = 0; i < m * n; ++i) { volatile float t = u[i] + resid[i]; ut[(size_t)i] = t; }
    gf8o_quantize(fmt, scaling, ut.data(), m, n, codes, scale_inv);
    const int64_t bn = (n + 127) / 128;
    for (int64_t i = 0; i < m; ++i)
        for (int64_t j = 0; j < n; ++j) {
            const int64_t sidx = scaling == 0 ? 0 : (i / 128) * bn + (j / 128);
            volatile float deq = (float)gf8o_fp8_to_double(fmt, codes[i * n + j]) * scale_inv[sidx];
            volatile float r = ut[(size_t)(i * n + j)] - deq;
            resid[i * n + j] = r;
        }
}

// ------------------------------------------------------------------------------------------------
// O9.  Synchronised scales and the vulnerability profile (f2, f3).
//   f2 (Alg. 1 l.4-5 "s <- Scale(Wg); s <- AllReduce_MAX(s)"; l.17-19 scale-synchronisation steps): the
//   amax is taken on its own (gf8o_amax), the ranks exchange it (max), and the cast uses the agreed value:
//       scale = fmax / amax_sync, scale_inv = amax_sync / fmax     (O4's rule, same degenerate cases), code = Q(x * scale).
//   f3 ("count how often encoded values hit the upper and lower FP8 boundaries"): with the codes of such a cast,
//       upper hit: the code is +-(largest finite value)                      (the value saturated or rounded up to fmax)
//       lower hit: x != 0 and the code is +-0 or +-(smallest subnormal)      (the value fell to the bottom of the format)
//   (S16: the paper does not define "boundary"; the ratio of hits to elements is the layer's vulnerability score.)
// ------------------------------------------------------------------------------------------------
void gf8o_amax(int scaling, const float* x, int64_t m, int64_t n, float* amax) {
    const int64_t bm = scaling == 0 ? 1 : (m + 127) / 128, bn = scaling == 0 ? 1 : (n + 127) / 128;
    for (int64_t b = 0; b < bm * bn; ++b) {
        const int64_t r0 = scaling == 0 ? 0 : (b / bn) * 128, r1 = scaling == 0 ? m : std::min(m, r0 + 128);
        const int64_t c0 = scaling == 0 ? 0 : (b % bn) * 128, c1 = scaling == 0 ? n : std::min(n, c0 + 128);
        uint32_t ab = 0;
        for (int64_t i = r0; i < r1; ++i)
            for (int64_t j = c0; j < c1; ++j) ab = std::max(ab, f2u(x[i * n + j]) & 0x7FFFFFFFu);
        amax[b] = u2f(ab);
    }
}

void gf8o_quantize_scaled(int fmt, int scaling, const float* x, int64_t m, int64_t n, const float* amax_sync,
                          uint8_t* codes, float* scale_inv, uint64_t* hits2) {
    const int64_t bn = (n + 127) / 128;
    const float fmax = (float)gf8o_fp8_max(fmt);
    const uint8_t top = gf8o_fp8_from_float(fmt, fmax);      // code of the largest finite value
    uint64_t upper = 0, lower = 0;
    const int64_t ns = scaling == 0 ? 1 : ((m + 127) / 128) * bn;
    std::vector<float> scale((size_t)ns);
    for (int64_t b = 0; b < ns; ++b) {
        const float amax = amax_sync[b];
        float sc = fmax / amax, si = amax / fmax;
        if (amax == 0.0f || !std::isfinite(amax) || !std::isfinite(sc)) { sc = 1.0f; si = 1.0f; }
        scale[(size_t)b] = sc;
        scale_inv[b] = si;
    }
    for (int64_t i = 0; i < m; ++i)
        for (int64_t j = 0; j < n; ++j) {
            const int64_t sidx = scaling == 0 ? 0 : (i / 128) * bn + (j / 128);
            volatile float y = x[i * n + j] * scale[(size_t)sidx];
            const uint8_t c = gf8o_fp8_from_float(fmt, y);
            codes[i * n + j] = c;
            const uint8_t mag = c & 0x7F;
            if (mag == (top & 0x7F)) ++upper;
            if (x[i * n + j] != 0.0f && mag <= 1) ++lower;
        }
    if (hits2) { hits2[0] = upper; hits2[1] = lower; }
}

// ------------------------------------------------------------------------------------------------
// O1.  Factor accumulate (Eq. 4: A = E[a a^T], G = E[delta delta^T]; S3, S4).
//   C = (1/T) sum_t x_t x_t^T by the triple loop; first call A = C, later A = beta A + (1-beta) C.
//   Damping is not stored in the accumulator.
// ------------------------------------------------------------------------------------------------
void gf8o_factor_accumulate(double* A, int first, double beta, const double* X, int64_t T, int64_t d) {
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t i = 0; i < d; ++i)
        for (int64_t j = 0; j < d; ++j) {
            double c = 0.0;
            for (int64_t t = 0; t < T; ++t) c += X[t * d + i] * X[t * d + j];
            c /= (double)T;
            A[i * d + j] = first ? c : beta * A[i * d + j] + (1.0 - beta) * c;
        }
}

// ------------------------------------------------------------------------------------------------
// Cyclic Jacobi eigensolver for a symmetric n x n matrix (the k x k Rayleigh-Ritz solve of O2 and
// the brute-force d x d eigenbasis).  Golub & Van Loan Alg. 8.5 rotations, row-cyclic sweeps until
// off(B) <= 1e-14 ||B||_F.  Returns eigenvalues sorted descending in M, eigenvectors in the
// columns of Z (n x n row-major).
// ------------------------------------------------------------------------------------------------
void gf8o_jacobi_eig(const double* Bin, int n, double* Z, double* M) {
    std::vector<double> B(Bin, Bin + (size_t)n * n), Zw((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i) Zw[(size_t)i * n + i] = 1.0;
    double fro = 0.0;
    for (size_t i = 0; i < (size_t)n * n; ++i) fro += B[i] * B[i];
    fro = std::sqrt(fro);
    for (int sweep = 0; sweep < 200; ++sweep) {
        double off = 0.0;
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j) if (i != j) off += B[(size_t)i * n + j] * B[(size_t)i * n + j];
        if (std::sqrt(off) <= 1e-14 * fro) break;
        for (int p = 0; p < n - 1; ++p)
            for (int q = p + 1; q < n; ++q) {
                const double bpq = B[(size_t)p * n + q];
                if (bpq == 0.0) continue;
                const double tau = (B[(size_t)q * n + q] - B[(size_t)p * n + p]) / (2.0 * bpq);
                const double t = (tau >= 0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
                const double c = 1.0 / std::sqrt(1.0 + t * t), s = t * c;
                for (int i = 0; i < n; ++i) {                 // B <- B J  (columns p, q)
                    const double bip = B[(size_t)i * n + p], biq = B[(size_t)i * n + q];
                    B[(size_t)i * n + p] = c * bip - s * biq;
                    B[(size_t)i * n + q] = s * bip + c * biq;
                }
                for (int j = 0; j < n; ++j) {                 // B <- J^T B  (rows p, q)
                    const double bpj = B[(size_t)p * n + j], bqj = B[(size_t)q * n + j];
                    B[(size_t)p * n + j] = c * bpj - s * bqj;
                    B[(size_t)q * n + j] = s * bpj + c * bqj;
                }
                for (int i = 0; i < n; ++i) {                 // Z <- Z J
                    const double zip = Zw[(size_t)i * n + p], ziq = Zw[(size_t)i * n + q];
                    Zw[(size_t)i * n + p] = c * zip - s * ziq;
                    Zw[(size_t)i * n + q] = s * zip + c * ziq;
                }
            }
    }
    std::vector<int> idx(n);
    for (int i = 0; i < n; ++i) idx[i] = i;
    std::stable_sort(idx.begin(), idx.end(),
                     [&](int a, int b) { return B[(size_t)a * n + a] > B[(size_t)b * n + b]; });
    for (int jn = 0; jn < n; ++jn) {
        M[jn] = B[(size_t)idx[jn] * n + idx[jn]];
        for (int i = 0; i < n; ++i) Z[(size_t)i * n + jn] = Zw[(size_t)i * n + idx[jn]];
    }
}

// Twice-applied modified Gram-Schmidt on the columns of V (d x k row-major), in place.
static void mgs2(double* V, int64_t d, int k) {
    for (int j = 0; j < k; ++j) {
        for (int pass = 0; pass < 2; ++pass)
            for (int i = 0; i < j; ++i) {
                double dot = 0.0;
                for (int64_t r = 0; r < d; ++r) dot += V[r * k + i] * V[r * k + j];
                for (int64_t r = 0; r < d; ++r) V[r * k + j] -= dot * V[r * k + i];
            }
        double nrm = 0.0;
        for (int64_t r = 0; r < d; ++r) nrm += V[r * k + j] * V[r * k + j];
        nrm = std::sqrt(nrm);
        for (int64_t r = 0; r < d; ++r) V[r * k + j] /= nrm;
    }
}

// Multipliers from Ritz values (S2, S3): model A_bar = U (M + lam) U^T + rho (I - U U^T),
//   rho = max(0, (tr A - sum mu) / (d - k)) + lam   (k == d: rho = mu_d + lam)
//   D_i = sqrt(rho / (mu_i + lam)),  e_i = D_i - 1 (T = I + U diag(e) U^T = sqrt(rho) A_bar^-1/2),
//   ebar_i = 1/D_i - 1 (T^-1).
void gf8o_multipliers(const double* mu, int k, int64_t d, double trace, double lam, double* rho_out,
                      double* e, double* ebar) {
    double s = 0.0;
    for (int i = 0; i < k; ++i) s += mu[i];
    double rho = (k < d) ? std::max(0.0, (trace - s) / (double)(d - k)) + lam : mu[k - 1] + lam;
    for (int i = 0; i < k; ++i) {
        const double D = std::sqrt(rho / (mu[i] + lam));
        e[i] = D - 1.0;
        ebar[i] = 1.0 / D - 1.0;
    }
    *rho_out = rho;
}

// ------------------------------------------------------------------------------------------------
// O2.  Basis refresh (Eq. 24: A ~ U_r Lambda_r U_r^T; method = S5):
//   V <- orth(V0); q times { Y = A V; V <- orth(Y) }; B = V^T A V; Jacobi B = Z M Z^T (sorted);
//   U = V Z; mu_i = max(M_ii, 0); sign rule: largest-magnitude entry of each column positive.
// ------------------------------------------------------------------------------------------------
void gf8o_refresh_basis(const double* A, int64_t d, int k, const double* V0, int q, double lam,
                        double* U, double* mu, double* rho, double* e, double* ebar) {
    std::vector<double> V(V0, V0 + (size_t)d * k), Y((size_t)d * k);
    mgs2(V.data(), d, k);
    auto matmulAV = [&]() {
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < d; ++i)
            for (int j = 0; j < k; ++j) {
                double acc = 0.0;
                for (int64_t l = 0; l < d; ++l) acc += A[i * d + l] * V[l * k + j];
                Y[i * k + j] = acc;
            }
    };
    for (int it = 0; it < q; ++it) {
        matmulAV();
        V = Y;
        mgs2(V.data(), d, k);
    }
    matmulAV();                                      // Y = A V
    std::vector<double> B((size_t)k * k), Z((size_t)k * k), M(k);
    for (int i = 0; i < k; ++i)
        for (int j = 0; j < k; ++j) {
            double acc = 0.0;
            for (int64_t r = 0; r < d; ++r) acc += V[r * k + i] * Y[r * k + j];
            B[(size_t)i * k + j] = acc;
        }
    for (int i = 0; i < k; ++i)                       // symmetrise the rounding noise
        for (int j = i + 1; j < k; ++j) {
            const double s = 0.5 * (B[(size_t)i * k + j] + B[(size_t)j * k + i]);
            B[(size_t)i * k + j] = B[(size_t)j * k + i] = s;
        }
    gf8o_jacobi_eig(B.data(), k, Z.data(), M.data());
    for (int64_t r = 0; r < d; ++r)
        for (int j = 0; j < k; ++j) {
            double acc = 0.0;
            for (int l = 0; l < k; ++l) acc += V[r * k + l] * Z[(size_t)l * k + j];
            U[r * k + j] = acc;
        }
    for (int j = 0; j < k; ++j) {
        int64_t big = 0;
        for (int64_t r = 1; r < d; ++r) if (std::fabs(U[r * k + j]) > std::fabs(U[big * k + j])) big = r;
        if (U[big * k + j] < 0) for (int64_t r = 0; r < d; ++r) U[r * k + j] = -U[r * k + j];
        mu[j] = std::max(M[j], 0.0);
    }
    double tr = 0.0;
    for (int64_t i = 0; i < d; ++i) tr += A[i * d + i];
    gf8o_multipliers(mu, k, d, tr, lam, rho, e, ebar);
}

// Brute force (tiny inputs only): full d x d cyclic Jacobi, keep the top k; same sign rule.
void gf8o_brute_basis(const double* A, int64_t d, int k, double lam, double* U, double* mu, double* rho,
                      double* e, double* ebar) {
    std::vector<double> Z((size_t)d * d), M(d);
    gf8o_jacobi_eig(A, (int)d, Z.data(), M.data());
    for (int j = 0; j < k; ++j) {
        int64_t big = 0;
        for (int64_t r = 1; r < d; ++r) if (std::fabs(Z[r * d + j]) > std::fabs(Z[big * d + j])) big = r;
        const double sg = Z[big * d + j] < 0 ? -1.0 : 1.0;
        for (int64_t r = 0; r < d; ++r) U[r * k + j] = sg * Z[r * d + j];
        mu[j] = std::max(M[j], 0.0);
    }
    double tr = 0.0;
    for (int64_t i = 0; i < d; ++i) tr += A[i * d + i];
    gf8o_multipliers(mu, k, d, tr, lam, rho, e, ebar);
}

// T = I + U diag(e) U^T  (d x d, S2).
void gf8o_build_T(const double* U, const double* e, int64_t d, int k, double* T) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < d; ++i)
        for (int64_t j = 0; j < d; ++j) {
            double acc = (i == j) ? 1.0 : 0.0;
            for (int l = 0; l < k; ++l) acc += U[i * k + l] * e[l] * U[j * k + l];
            T[i * d + j] = acc;
        }
}

// ------------------------------------------------------------------------------------------------
// O3 / O6, dense form (tiny inputs).  out = T_G W T_A (Eq. 14 with the symmetric
// roots of S1; :180 Eq. 18 when TG == NULL; :172 Eq. 17 / :184 Eq. 19 when called with T^-1).
// ------------------------------------------------------------------------------------------------
void gf8o_whiten_dense(const double* W, int64_t m, int64_t n, const double* TG, const double* TA,
                       double* out) {
    std::vector<double> Y((size_t)m * n);
    for (int64_t i = 0; i < m; ++i)                    // Y = W T_A
        for (int64_t j = 0; j < n; ++j) {
            if (!TA) { Y[i * n + j] = W[i * n + j]; continue; }
            double acc = 0.0;
            for (int64_t l = 0; l < n; ++l) acc += W[i * n + l] * TA[l * n + j];
            Y[i * n + j] = acc;
        }
    for (int64_t i = 0; i < m; ++i)                    // out = T_G Y
        for (int64_t j = 0; j < n; ++j) {
            if (!TG) { out[i * n + j] = Y[i * n + j]; continue; }
            double acc = 0.0;
            for (int64_t l = 0; l < m; ++l) acc += TG[i * m + l] * Y[l * n + j];
            out[i * n + j] = acc;
        }
}

// ------------------------------------------------------------------------------------------------
// O3 / O6, low-rank form (Eq. 22 W~ = W T_A with T_A built from Eq. 24's U_r; S2):
//   P = W U_A (m x kA), Q = U_G^T W (kG x n), S = U_G^T P (kG x kA)
//   out = W + P E_A U_A^T + U_G E_G Q + U_G E_G S E_A U_A^T
// UG == NULL (kG = 0): input side only (Eq. 18).  UA == NULL: output side only.  Both NULL: copy.
// Unwhitening (Eq. 17 / 19) is the same call with the ebar multipliers.
// ------------------------------------------------------------------------------------------------
void gf8o_whiten_lowrank(const double* W, int64_t m, int64_t n, const double* UG, const double* eG,
                         int kG, const double* UA, const double* eA, int kA, double* out) {
    if (!UG) kG = 0;
    if (!UA) kA = 0;
    std::vector<double> P((size_t)m * std::max(kA, 1)), Q((size_t)std::max(kG, 1) * n),
        S((size_t)std::max(kG, 1) * std::max(kA, 1));
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < m; ++i)
        for (int a = 0; a < kA; ++a) {
            double acc = 0.0;
            for (int64_t j = 0; j < n; ++j) acc += W[i * n + j] * UA[j * kA + a];
            P[i * kA + a] = acc;
        }
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < n; ++j)
        for (int g = 0; g < kG; ++g) {
            double acc = 0.0;
            for (int64_t i = 0; i < m; ++i) acc += UG[i * kG + g] * W[i * n + j];
            Q[(size_t)g * n + j] = acc;
        }
    for (int g = 0; g < kG; ++g)
        for (int a = 0; a < kA; ++a) {
            double acc = 0.0;
            for (int64_t i = 0; i < m; ++i) acc += UG[i * kG + g] * P[i * kA + a];
            S[(size_t)g * kA + a] = acc;
        }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < m; ++i)
        for (int64_t j = 0; j < n; ++j) {
            double t1 = 0.0, t2 = 0.0, t3 = 0.0;
            for (int a = 0; a < kA; ++a) t1 += P[i * kA + a] * eA[a] * UA[j * kA + a];
            for (int g = 0; g < kG; ++g) t2 += UG[i * kG + g] * eG[g] * Q[(size_t)g * n + j];
            for (int g = 0; g < kG; ++g) {
                double sa = 0.0;
                for (int a = 0; a < kA; ++a) sa += S[(size_t)g * kA + a] * eA[a] * UA[j * kA + a];
                t3 += UG[i * kG + g] * eG[g] * sa;
            }
            out[i * n + j] = W[i * n + j] + t1 + t2 + t3;
        }
}

// ------------------------------------------------------------------------------------------------
// Conversions.  double -> bf16 is ONE round-to-nearest-even of the double value (O6).
// ------------------------------------------------------------------------------------------------
uint16_t gf8o_double_to_bf16(double v) {
    if (std::isnan(v)) return 0x7FC0;
    const uint16_t sign = std::signbit(v) ? 0x8000 : 0;
    double a = std::fabs(v);
    if (a == 0.0) return sign;
    if (std::isinf(a)) return sign | 0x7F80;
    int e;
    (void)std::frexp(a, &e);
    int E = e - 1;
    if (E < -126) E = -126;
    const double quantum = std::ldexp(1.0, E - 7);
    const double r = rne_int(a / quantum) * quantum;
    if (r >= std::ldexp(1.0, 128)) return sign | 0x7F80;
    const float f = (float)r;                        // exact: r has <= 8 significant bits
    return (uint16_t)(sign | (f2u(f) >> 16));
}
void gf8o_to_bf16(const double* in, int64_t n, uint16_t* out) {
    for (int64_t i = 0; i < n; ++i) out[i] = gf8o_double_to_bf16(in[i]);
}
void gf8o_from_bf16(const uint16_t* in, int64_t n, double* out) {
    for (int64_t i = 0; i < n; ++i) out[i] = (double)u2f((uint32_t)in[i] << 16);
}
void gf8o_to_f32(const double* in, int64_t n, float* out) {
    for (int64_t i = 0; i < n; ++i) out[i] = (float)in[i];
}

// ------------------------------------------------------------------------------------------------
// O7.  Reconstruction metrics (Eq. 21): RelL2, Cos, MaxErr, MSE.
// ------------------------------------------------------------------------------------------------
void gf8o_metrics(const double* ghat, const double* g, int64_t n, double* out4) {
    double d2 = 0, g2 = 0, h2 = 0, dot = 0, mx = 0;
    for (int64_t i = 0; i < n; ++i) {
        const double d = ghat[i] - g[i];
        d2 += d * d; g2 += g[i] * g[i]; h2 += ghat[i] * ghat[i]; dot += ghat[i] * g[i];
        mx = std::max(mx, std::fabs(d));
    }
    out4[0] = std::sqrt(d2) / std::sqrt(g2);
    out4[1] = dot / (std::sqrt(h2) * std::sqrt(g2));
    out4[2] = mx;
    out4[3] = d2 / (double)n;
}

// ------------------------------------------------------------------------------------------------
// Sampled outputs (parity at BASELINE.json's full sizes, where the whole-matrix routines above are too slow):
// each is the plain definition of ONE output element.
//
// O1 at (i, j): A[i][j] = (1/T) sum_t x_t[i] x_t[j]                        (Eq. 4), no EMA.
// O3 / O6 at (i, j): (T_G W T_A)[i][j] = sum_r sum_c T_G[i][r] W[r][c] T_A[c][j] with the DENSE rows / columns of
//   T = I + U diag(e) U^T formed on the fly (Eq. 14 in the dense form; pass ebar for Eq. 17).
// ------------------------------------------------------------------------------------------------
void gf8o_factor_entries(const double* X, int64_t T, int64_t d, const int64_t* ii, const int64_t* jj, int64_t ns, double* out) {
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t s = 0; s < ns; ++s) {
        double c = 0.0;
        for (int64_t t = 0; t < T; ++t) c += X[t * d + ii[s]] * X[t * d + jj[s]];
        out[s] = c / (double)T;
    }
}

void gf8o_whiten_samples(const double* W, int64_t m, int64_t n, const double* UG, const double* eG, int kG, const double* UA,
                         const double* eA, int kA, const int64_t* ii, const int64_t* jj, int64_t ns, double* out) {
    if (!UG) kG = 0;
    if (!UA) kA = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t s = 0; s < ns; ++s) {
        const int64_t i = ii[s], j = jj[s];
        std::vector<double> tg((size_t)m), ta((size_t)n);
        for (int64_t r = 0; r < m; ++r) {                 // row i of T_G
            double acc = r == i ? 1.0 : 0.0;
            for (int g = 0; g < kG; ++g) acc += UG[i * kG + g] * eG[g] * UG[r * kG + g];
            tg[(size_t)r] = acc;
        }
        for (int64_t c = 0; c < n; ++c) {                 // column j of T_A
            double acc = c == j ? 1.0 : 0.0;
            for (int a = 0; a < kA; ++a) acc += UA[c * kA + a] * eA[a] * UA[j * kA + a];
            ta[(size_t)c] = acc;
        }
        double v = 0.0;
        for (int64_t r = 0; r < m; ++r) {
            double row = 0.0;
            for (int64_t c = 0; c < n; ++c) row += W[r * n + c] * ta[(size_t)c];
            v += tg[(size_t)r] * row;
        }
        out[s] = v;
    }
}

// Threads the OpenMP loops use from now on (bench.py's single-thread baseline figure); no effect without OpenMP.
void gf8o_set_num_threads(int n) {
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int gf8o_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
