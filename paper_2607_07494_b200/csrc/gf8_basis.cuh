// gf8_basis.cuh -- the small dense pieces of a2 basis refresh (Eq. 24; S5):
//   CholeskyQR orthonormalisation in FP64, the single-CTA Jacobi eigensolve of the k x k Rayleigh-Ritz
//   matrix, and the multipliers (rho, e, ebar).  No host eigensolver, no host synchronisation.
#pragma once
#include "gf8_common.cuh"

namespace gf8 {

// ---- Cholesky of a k x k SPD Gram matrix, in place, upper factor R (G = R^T R), one CTA -----------
// G row-major in global memory (k <= 512); only the upper triangle is read and written.  With use_smem the matrix is staged in
// dynamic shared memory (k * (k | 1) doubles: an odd leading dimension keeps column walks off one bank), which turns the
// three global round trips of every pivot step into shared-memory ones.
__device__ __forceinline__ void cholesky_upper_body(double* __restrict__ Gg, int k, int use_smem) {
    extern __shared__ double s_chol[];
    __shared__ double s_diag, s_dmax;
    const int ld = use_smem ? (k | 1) : k;
    double* G = use_smem ? s_chol : Gg;
    if (use_smem) {
        for (int idx = threadIdx.x; idx < k * k; idx += blockDim.x) {
            const int i = idx / k, l = idx % k;
            if (l >= i) G[i * ld + l] = Gg[idx];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        double mx = 0.0;
        for (int j = 0; j < k; ++j) mx = fmax(mx, G[(int64_t)j * ld + j]);
        s_dmax = mx;
    }
    __syncthreads();
    if (use_smem) {
        // One phase and one barrier per pivot: row j of the working copy stays unscaled (R_jl = G_jl / sqrt(G_jj) goes straight to
        // global memory), and the trailing update uses G_ji G_jl / G_jj, every thread forming the reciprocal itself.
        const double dmax = s_dmax;
        for (int j = 0; j < k; ++j) {
            const double d = G[j * ld + j];
            const bool good = d > 1e-26 * dmax && d > 0.0;        // (breakdown guard, see below)
            const double rs = good ? rsqrt(d) : 1e-150;
            const double inv_d = good ? rs * rs : 0.0;
            for (int l = j + threadIdx.x; l < k; l += blockDim.x) Gg[(int64_t)j * k + l] = l == j ? (good ? d * rs : 1e150) : G[j * ld + l] * rs;
            const int rem = k - j - 1;
            for (int idx = threadIdx.x; idx < rem * rem; idx += blockDim.x) {
                const int i = j + 1 + idx / rem, l = j + 1 + idx % rem;
                if (l >= i) G[i * ld + l] = fma(-(G[j * ld + i] * inv_d), G[j * ld + l], G[i * ld + l]);
            }
            __syncthreads();
        }
        return;
    }
    for (int j = 0; j < k; ++j) {
        if (threadIdx.x == 0) {
            const double d = G[(int64_t)j * ld + j];
            // Breakdown guard: a pivot that has cancelled to (FP64) rounding level against the largest diagonal entry means the
            // column lies in the span of the earlier ones (rank-deficient A V).  It is DEFLATED: a huge R_jj sends the column
            // of V to ~0 (it then carries Ritz value 0 and contributes nothing to T) instead of blowing it up by 1 / sqrt(tiny).
            s_diag = (d > 1e-26 * s_dmax && d > 0.0) ? sqrt(d) : 1e150;
            G[(int64_t)j * ld + j] = s_diag;
        }
        __syncthreads();
        const double rjj = s_diag;
        for (int l = j + 1 + threadIdx.x; l < k; l += blockDim.x) G[(int64_t)j * ld + l] /= rjj;
        __syncthreads();
        // trailing update of the upper triangle: G[i][l] -= R[j][i] * R[j][l], j < i <= l
        const int rem = k - j - 1;
        for (int idx = threadIdx.x; idx < rem * rem; idx += blockDim.x) {
            const int i = j + 1 + idx / rem, l = j + 1 + idx % rem;
            if (l >= i) G[(int64_t)i * ld + l] -= G[(int64_t)j * ld + i] * G[(int64_t)j * ld + l];
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(1024) cholesky_upper_kernel(double* __restrict__ Gg, int k, int use_smem) {
    cholesky_upper_body(Gg, k, use_smem);
}

// ---- V <- V R^-1 (R upper triangular), V d x k FP64, in place -------------------------------------------
// Row by row x R = v, column-oriented: once x_j = v_j / R_jj is known, v_l -= x_j R_jl for every l > j.
// A warp takes TRI_ROWS rows at once (independent chains hide the shuffle / FMA latency of each other); a lane holds the
// elements l = lane, lane + 32 of each (k <= 64).  R and the reciprocals of its diagonal are staged in shared memory once
// per CTA, which then walks TRI_GROUPS groups of rows.
constexpr int TRI_ROWS = 4, TRI_WARPS = 8, TRI_GROUPS = 8, TRI_MAXK = 64;      // a CTA takes TRI_ROWS * TRI_WARPS * TRI_GROUPS = 256 rows
__device__ __forceinline__ void trisolve_rows_warp_body(double* __restrict__ V, const double* __restrict__ Rm, int d, int k, int blk) {
    __shared__ double s_R[TRI_MAXK * TRI_MAXK];
    __shared__ double s_inv[TRI_MAXK];
    for (int idx = threadIdx.x; idx < k * k; idx += blockDim.x) s_R[idx] = Rm[idx];
    for (int j = threadIdx.x; j < k; j += blockDim.x) s_inv[j] = 1.0 / Rm[(int64_t)j * k + j];
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int g = 0; g < TRI_GROUPS; ++g) {
        const int r0 = ((blk * TRI_GROUPS + g) * TRI_WARPS + warp) * TRI_ROWS;
        if (r0 >= d) return;
        double x[TRI_ROWS][2];
#pragma unroll
        for (int t = 0; t < TRI_ROWS; ++t)
#pragma unroll
            for (int u = 0; u < 2; ++u)
                x[t][u] = (r0 + t < d && lane + 32 * u < k) ? V[(int64_t)(r0 + t) * k + lane + 32 * u] : 0.0;
        for (int j = 0; j < k; ++j) {
            const double inv = s_inv[j];
            const double rl0 = lane < k ? s_R[j * k + lane] : 0.0, rl1 = lane + 32 < k ? s_R[j * k + lane + 32] : 0.0;
#pragma unroll
            for (int t = 0; t < TRI_ROWS; ++t) {
                const double xj = __shfl_sync(0xFFFFFFFFu, j < 32 ? x[t][0] : x[t][1], j & 31) * inv;
                if (lane == j) x[t][0] = xj; else if (lane > j) x[t][0] = fma(-xj, rl0, x[t][0]);
                if (lane + 32 == j) x[t][1] = xj; else if (lane + 32 > j) x[t][1] = fma(-xj, rl1, x[t][1]);
            }
        }
#pragma unroll
        for (int t = 0; t < TRI_ROWS; ++t)
#pragma unroll
            for (int u = 0; u < 2; ++u)
                if (r0 + t < d && lane + 32 * u < k) V[(int64_t)(r0 + t) * k + lane + 32 * u] = x[t][u];
    }
}

__global__ void __launch_bounds__(32 * TRI_WARPS) trisolve_rows_warp_kernel(double* __restrict__ V, const double* __restrict__ Rm,
                                                                            int d, int k) {
    trisolve_rows_warp_body(V, Rm, d, k, blockIdx.x);
}

// One thread per row (any k).
__global__ void __launch_bounds__(128) trisolve_rows_kernel(double* __restrict__ V, const double* __restrict__ Rm,
                                                            int d, int k) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= d) return;
    double* v = V + (int64_t)r * k;
    for (int j = 0; j < k; ++j) {
        double x = v[j];
        for (int i = 0; i < j; ++i) x -= v[i] * Rm[(int64_t)i * k + j];
        v[j] = x / Rm[(int64_t)j * k + j];
    }
}

// ---- Single-CTA parallel-order two-sided Jacobi on a symmetric k x k matrix (FP64) ----------------
// B (k x k) is overwritten; Z receives the eigenvectors (columns).  If the two matrices fit in
// dynamic shared memory (use_smem) they are staged there, otherwise the CTA works on global / L2.
// Round-robin ordering: k-1 rounds of k/2 disjoint rotations per sweep.  Output: mu sorted
// descending, Zs = Z with its columns permuted into that order.
__device__ __forceinline__ void jacobi_body(double* __restrict__ Bg, double* __restrict__ Zg, int k, int use_smem,
                                            double* __restrict__ mu_sorted, double* __restrict__ Zs, int max_sweeps) {
    extern __shared__ double s_dyn[];
    __shared__ double s_c[256], s_s[256];
    __shared__ int s_p[256], s_q[256];
    __shared__ double s_red[64];
    __shared__ int s_done;
    const int tid = threadIdx.x, nt = blockDim.x;
    double* B = use_smem ? s_dyn : Bg;
    const int ld = use_smem ? (k | 1) : k;        // odd leading dimension in shared memory: column walks spread over the banks
    double* Z = use_smem ? s_dyn + (size_t)k * ld : Zg;
    // load + symmetrise; Z = I
    for (int idx = tid; idx < k * k; idx += nt) {
        const int i = idx / k, j = idx % k;
        if (use_smem) B[i * ld + j] = 0.5 * (Bg[(int64_t)i * k + j] + Bg[(int64_t)j * k + i]);
        Z[i * ld + j] = (i == j) ? 1.0 : 0.0;
    }
    __syncthreads();
    if (!use_smem) {                    // in-place symmetrisation on global memory
        for (int idx = tid; idx < k * k; idx += nt) {
            const int i = idx / k, j = idx % k;
            if (i < j) {
                const double v = 0.5 * (B[(int64_t)i * ld + j] + B[(int64_t)j * ld + i]);
                B[(int64_t)i * ld + j] = v;
                B[(int64_t)j * ld + i] = v;
            }
        }
        __syncthreads();
    }
    const int ke = (k + 1) & ~1;        // players (one dummy when k is odd)
    const int half = ke / 2;
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
        // convergence: off(B) <= 1e-14 ||B||_F
        double off = 0.0, fro = 0.0;
        for (int idx = tid; idx < k * k; idx += nt) {
            const double v = B[(idx / k) * ld + idx % k];
            fro += v * v;
            if (idx / k != idx % k) off += v * v;
        }
        for (int o = 16; o > 0; o >>= 1) {
            off += __shfl_xor_sync(0xFFFFFFFFu, off, o);
            fro += __shfl_xor_sync(0xFFFFFFFFu, fro, o);
        }
        if ((tid & 31) == 0) { s_red[tid >> 5] = off; s_red[32 + (tid >> 5)] = fro; }
        __syncthreads();
        if (tid == 0) {
            double o2 = 0, f2 = 0;
            for (int w = 0; w < (nt + 31) / 32; ++w) { o2 += s_red[w]; f2 += s_red[32 + w]; }
            s_done = (sqrt(o2) <= 1e-14 * sqrt(f2)) ? 1 : 0;
        }
        __syncthreads();
        if (s_done) break;
        for (int round = 0; round < ke - 1; ++round) {
            // pairs of this round + rotation angles
            for (int i = tid; i < half; i += nt) {
                int p, q;
                if (i == 0) { p = ke - 1; q = round; }
                else { p = (round + i) % (ke - 1); q = (round - i + (ke - 1)) % (ke - 1); }
                if (p > q) { const int t = p; p = q; q = t; }
                double c = 1.0, s = 0.0;
                if (q < k) {
                    const double bpq = B[(int64_t)p * ld + q];
                    if (bpq != 0.0) {
                        // tan of the rotation angle, t = sign(a) b / (|a| + sqrt(a^2 + b^2)) with a = (B_qq - B_pp) / 2, b = B_pq
                        // (the textbook 1 / (tau + sign(tau) sqrt(1 + tau^2)), tau = a / b, without the division by b);
                        // reciprocal square roots instead of sqrt + divide keep the dependent FP64 chain short
                        const double a = 0.5 * (B[(int64_t)q * ld + q] - B[(int64_t)p * ld + p]);
                        const double h2 = fma(a, a, bpq * bpq);
                        const double h = h2 * rsqrt(h2);
                        const double t = (a >= 0 ? bpq : -bpq) / (fabs(a) + h);
                        c = rsqrt(fma(t, t, 1.0));
                        s = t * c;
                    }
                } else { q = -1; }
                s_p[i] = p; s_q[i] = q; s_c[i] = c; s_s[i] = s;
            }
            __syncthreads();
            // B <- J^T B J in ONE phase: the thread of pair (i, i') owns the 2 x 2 block rows {p, q} x columns {p', q'}; every element
            // of B lies in exactly one block, so the update is in place without a barrier between the column and the row rotation
            for (int idx = tid; idx < half * half; idx += nt) {
                const int i = idx / half, i2 = idx % half;
                const int p = s_p[i], q = s_q[i], p2 = s_p[i2], q2 = s_q[i2];
                const double c = s_c[i], sn = s_s[i], c2 = s_c[i2], sn2 = s_s[i2];
                const bool rq = q >= 0, cq = q2 >= 0;
                const double b00 = B[(int64_t)p * ld + p2];
                const double b01 = cq ? B[(int64_t)p * ld + q2] : 0.0;
                const double b10 = rq ? B[(int64_t)q * ld + p2] : 0.0;
                const double b11 = (rq && cq) ? B[(int64_t)q * ld + q2] : 0.0;
                const double x00 = c2 * b00 - sn2 * b01, x01 = sn2 * b00 + c2 * b01;      // columns
                const double x10 = c2 * b10 - sn2 * b11, x11 = sn2 * b10 + c2 * b11;
                B[(int64_t)p * ld + p2] = c * x00 - sn * x10;                                // rows
                if (cq) B[(int64_t)p * ld + q2] = c * x01 - sn * x11;
                if (rq) B[(int64_t)q * ld + p2] = sn * x00 + c * x10;
                if (rq && cq) B[(int64_t)q * ld + q2] = sn * x01 + c * x11;
            }
            // Z <- Z J  (columns p, q of every row)
            for (int idx = tid; idx < half * k; idx += nt) {
                const int i = idx / k, r = idx % k;
                const int p = s_p[i], q = s_q[i];
                if (q < 0) continue;
                const double c = s_c[i], sn = s_s[i];
                const double zp = Z[(int64_t)r * ld + p], zq = Z[(int64_t)r * ld + q];
                Z[(int64_t)r * ld + p] = c * zp - sn * zq;
                Z[(int64_t)r * ld + q] = sn * zp + c * zq;
            }
            __syncthreads();
        }
    }
    // rank sort (descending, ties by index) and permuted eigenvector output
    for (int i = tid; i < k; i += nt) {
        const double mi = B[(int64_t)i * ld + i];
        int rank = 0;
        for (int j = 0; j < k; ++j) {
            const double mj = B[(int64_t)j * ld + j];
            rank += (mj > mi) || (mj == mi && j < i);
        }
        mu_sorted[rank] = mi;
        // column i of Z goes to column `rank` of Zs
        for (int r = 0; r < k; ++r) Zs[(int64_t)r * k + rank] = Z[(int64_t)r * ld + i];
    }
}

__global__ void __launch_bounds__(1024) jacobi_kernel(double* __restrict__ Bg, double* __restrict__ Zg, int k,
                                                      int use_smem, double* __restrict__ mu_sorted,
                                                      double* __restrict__ Zs, int max_sweeps) {
    jacobi_body(Bg, Zg, k, use_smem, mu_sorted, Zs, max_sweeps);
}

// ---- trace(A) in FP64 and the multipliers (S2, S3) ---------------------------------------
//   rho = max(0, (tr A - sum mu) / (d - k)) + lam   (k == d: rho = mu_k + lam)
//   D_i = sqrt(rho / (mu_i + lam)),  e_i = D_i - 1,  ebar_i = 1/D_i - 1
// One CTA.  If `trace_from` is null, rho_in is used as given (gf8_set_basis).
__device__ __forceinline__ void multipliers_body(const float* __restrict__ factor, int d, int k,
                                                 const double* __restrict__ mu64, const float* __restrict__ mu32,
                                                 double lam, double rho_in, float* __restrict__ mu_out,
                                                 float* __restrict__ e, float* __restrict__ ebar,
                                                 float* __restrict__ rho_out) {
    __shared__ double s_part[256], s_tr[256];
    __shared__ double s_rho, s_floor;
    double tr = 0.0, sm = 0.0;
    if (factor) for (int i = threadIdx.x; i < d; i += blockDim.x) tr += (double)factor[(int64_t)i * d + i];
    for (int i = threadIdx.x; i < k; i += blockDim.x) {
        const double m = mu64 ? fmax(mu64[i], 0.0) : (double)mu32[i];
        sm += m;
    }
    s_part[threadIdx.x] = tr - sm;
    s_tr[threadIdx.x] = factor ? tr : sm;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0, scale = 0.0;
        for (int i = 0; i < blockDim.x; ++i) { t += s_part[i]; scale += s_tr[i]; }
        double rho;
        if (!factor) rho = rho_in;
        else if (k < d) rho = fmax(0.0, t / (double)(d - k)) + lam;
        else rho = (mu64 ? fmax(mu64[k - 1], 0.0) : (double)mu32[k - 1]) + lam;
        // Guard outside the paper's domain (damping 0 with a rank-deficient factor, S13): rho and mu_i + lambda are
        // floored at 2^-23 of the mean eigenvalue, so D = sqrt(rho / (mu + lambda)) and 1 / D stay finite and positive.
        const double fl = fmax(scale / (double)(factor ? d : k), 1e-300) * 1.1920928955078125e-7;
        s_floor = fl;
        rho = fmax(rho, fl);
        s_rho = rho;
        *rho_out = (float)rho;
    }
    __syncthreads();
    const double rho = s_rho;
    for (int i = threadIdx.x; i < k; i += blockDim.x) {
        const double m = mu64 ? fmax(mu64[i], 0.0) : (double)mu32[i];
        const double D = sqrt(rho / fmax(m + lam, s_floor));
        mu_out[i] = (float)m;
        e[i] = (float)(D - 1.0);
        ebar[i] = (float)(1.0 / D - 1.0);
    }
}

__global__ void __launch_bounds__(256) multipliers_kernel(const float* __restrict__ factor, int d, int k,
                                                          const double* __restrict__ mu64, const float* __restrict__ mu32,
                                                          double lam, double rho_in, float* __restrict__ mu_out,
                                                          float* __restrict__ e, float* __restrict__ ebar,
                                                          float* __restrict__ rho_out) {
    multipliers_body(factor, d, k, mu64, mu32, lam, rho_in, mu_out, e, ebar, rho_out);
}

}  // namespace gf8
