// gf8_refresh.cuh -- a2 basis refresh for MANY factor sides at once (Eq. 24; S5).
//
// gf8_refresh_basis_many used to walk one chain of ~35 small launches per side on a handful of streams; the chains are
// latency-bound (single-CTA Cholesky / Jacobi steps, split-K GEMMs with a few hundred CTAs), so a 336-side refresh took
// 0.33 s.  Here every step of the algorithm is ONE launch over all sides of the call: the launch's grid carries the
// side (blockIdx.y, or a prefix table of row blocks for the heavy product), so the single-CTA steps of different sides
// fill the machine together and A V needs no split-K (each CTA runs a whole K loop: fixed summation order).
//
// The arithmetic is that of the per-side path (gf8_basis.cuh bodies, FP64 throughout):
//   V <- U (start basis), orthonormalise (CholeskyQR twice), n_iter times { V <- A V, orthonormalise },
//   Y = A V, B = V^T Y, Jacobi eigensolve of B, U <- V Z (sorted), multipliers (rho, e, ebar).
// Ranks k <= 64 only (the triangular solve and the product tile hold a 64-wide panel); other sides take the per-side path.
#pragma once
#include "gf8_basis.cuh"

namespace gf8 {
namespace rb {

constexpr int RB_MAXK = 64;
constexpr int RB_CHUNK = 256;            // rows of V per partial Gram product
constexpr int AV_BM = 128, AV_BK = 32;   // A V tile: 128 rows of A, K in steps of 32
constexpr int AV_LDA = AV_BM + 8;        // leading dimension of the K-major A tile (floats): 8 banks per K row, fragment loads conflict-free
constexpr int AV_LDV = RB_MAXK + 8;      // leading dimension of the V tile (doubles): K rows 16 banks apart, the two-wavefront minimum
constexpr int AV_SMEM = AV_BK * AV_LDV * 8 + AV_BK * AV_LDA * 4;

struct RefreshJob {
    const float* factor;     // d x d FP32
    float* U;                // d x k FP32: start basis in, refreshed basis out
    double* buf[2];          // d x k FP64 each: V and Y take turns
    double* part;            // ceil(d / RB_CHUNK) partial k x k products
    double* Gm;              // k x k: Gram matrix / its Cholesky factor
    double* Bm;              // k x k: Rayleigh-Ritz matrix (destroyed by the eigensolve)
    double* Zm;              // k x k scratch of the eigensolve (unused when it runs in shared memory)
    double* Zs;              // k x k eigenvectors, columns sorted by descending eigenvalue
    double* mu64;            // k
    float *mu, *e, *ebar, *rho;
    double lam;
    int32_t d, k;
    int32_t blk0;            // first AV_BM-row block of this side in the launch-wide list
    int32_t n_chunks;
    // FAST path: BF16 copies of the refreshed basis for the tensor-core engine (null: the side has none), rank padded to kp
    __nv_bfloat16 *U16, *Ut16, *U16_lo, *Ut16_lo;
    int32_t kp, pad_;
};

// ---- V <- (double) U ----------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) rb_widen_kernel(const RefreshJob* __restrict__ jobs, int flip) {
    const RefreshJob& j = jobs[blockIdx.y];
    const int64_t n = (int64_t)j.d * j.k;
    double* V = j.buf[flip];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) V[i] = (double)j.U[i];
}

// ---- partial products  part[c] = X[chunk c]^T W[chunk c]  (k x k, FP64), X = buf[xa], W = buf[xb] --------------
// FP64 tensor-core path (mma.sync m8n8k4): warp w owns rows 8 w .. 8 w + 7 of the product and all 64 columns (8 MMA tiles);
// 32 rows of the chunk are staged per step.  Leading dimension 72 doubles: the four K rows of a fragment load fall 16 banks
// apart, the two-wavefront minimum of a 64-bit warp load.
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
constexpr int RB_LD = RB_MAXK + 8;
__global__ void __launch_bounds__(256) rb_gram_kernel(const RefreshJob* __restrict__ jobs, int xa, int xb) {
    const RefreshJob& j = jobs[blockIdx.y];
    const int c = blockIdx.x;
    if (c >= j.n_chunks) return;
    const int d = j.d, k = j.k;
    const double* X = j.buf[xa];
    const double* W = j.buf[xb];
    __shared__ double Xs[32][RB_LD], Ws[32][RB_LD];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, fr = lane >> 2, fk = lane & 3;
    double acc[8][2] = {};
    const int r_begin = c * RB_CHUNK, r_end = min(d, r_begin + RB_CHUNK);
    for (int r0 = r_begin; r0 < r_end; r0 += 32) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int idx = tid + 256 * u, l = idx >> 6, col = idx & 63;
            const bool ok = r0 + l < r_end && col < k;
            Xs[l][col] = ok ? X[(int64_t)(r0 + l) * k + col] : 0.0;
            Ws[l][col] = ok ? W[(int64_t)(r0 + l) * k + col] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            const double a = Xs[4 * ks + fk][8 * warp + fr];
#pragma unroll
            for (int nb = 0; nb < 8; ++nb) dmma884(acc[nb][0], acc[nb][1], a, Ws[4 * ks + fk][8 * nb + fr]);
        }
        __syncthreads();
    }
    double* P = j.part + (int64_t)c * k * k;
    const int i = 8 * warp + fr;
#pragma unroll
    for (int nb = 0; nb < 8; ++nb) {
        const int l = 8 * nb + 2 * fk;
        if (i < k && l < k) P[(int64_t)i * k + l] = acc[nb][0];
        if (i < k && l + 1 < k) P[(int64_t)i * k + l + 1] = acc[nb][1];
    }
}

// ---- out = sum over chunks of part[c], in chunk order (fixed summation order); to_B: into Bm, else into Gm --------
__global__ void __launch_bounds__(256) rb_sum_kernel(const RefreshJob* __restrict__ jobs, int to_B) {
    const RefreshJob& j = jobs[blockIdx.y];
    const int kk = j.k * j.k;
    double* out = to_B ? j.Bm : j.Gm;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < kk; i += gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int c = 0; c < j.n_chunks; ++c) s += j.part[(int64_t)c * kk + i];
        out[i] = s;
    }
}

// Cholesky factor R of Gm (upper, in place) and then Zs <- R^-1 (upper triangular, zero below the diagonal): the panel is
// orthonormalised as the product V R^-1 (rb_rightmul_kernel), a register-tiled GEMM, instead of d triangular solves.
// 16 threads share a column of the inverse: x_c = 1 / R_cc, x_i = -(sum_{i < l <= c} R_il x_l) / R_ii for i = c-1 .. 0.
__global__ void __launch_bounds__(1024) rb_chol_kernel(const RefreshJob* __restrict__ jobs) {
    const RefreshJob& j = jobs[blockIdx.x];
    const int k = j.k;
    cholesky_upper_body(j.Gm, k, 1);
    __syncthreads();
    extern __shared__ double s_inv_dyn[];             // (the Cholesky working copy is dead: its shared memory holds the inverse)
    double (*s_x)[RB_MAXK + 1] = reinterpret_cast<double (*)[RB_MAXK + 1]>(s_inv_dyn);      // s_x[c][i]: column c of the inverse
    const int c = threadIdx.x >> 4, sub = threadIdx.x & 15;
    const double* R = j.Gm;                           // (written by this CTA above; the barrier makes it visible CTA-wide)
    // (the two columns of a warp run loops of different lengths: every warp-level primitive names its own half-warp)
    const unsigned hmask = 0xFFFFu << (16 * ((threadIdx.x >> 4) & 1));
    if (c < k) {
        for (int i = sub; i < k; i += 16) s_x[c][i] = 0.0;
        __syncwarp(hmask);
        if (sub == 0) s_x[c][c] = 1.0 / R[(int64_t)c * k + c];
        __syncwarp(hmask);
        for (int i = c - 1; i >= 0; --i) {
            double part = 0.0;
            for (int l = i + 1 + sub; l <= c; l += 16) part = fma(R[(int64_t)i * k + l], s_x[c][l], part);
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) part += __shfl_xor_sync(hmask, part, o, 16);
            if (sub == 0) s_x[c][i] = -part / R[(int64_t)i * k + i];
            __syncwarp(hmask);
        }
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < k * k; idx += blockDim.x) {
        const int i = idx / k, cc = idx % k;
        j.Zs[idx] = s_x[cc][i];
    }
}

// ---- buf[flip] <- buf[flip] * Zs   (to_U = 0: FP64, in place)   or   U <- (float)(buf[flip] * Zs)   (to_U = 1) ------------
// One CTA per 64 rows, FP64 tensor-core path: warp w owns rows 8 w .. 8 w + 7 and all 64 columns; K = k <= 64.  The row panel
// stays row-major in shared memory (leading dimension 68 doubles: the eight rows of an A fragment load fall 8 banks apart).
constexpr int RM_LDV = RB_MAXK + 4;
constexpr int RM_SMEM = (64 * RM_LDV + RB_MAXK * RB_LD) * 8;
__global__ void __launch_bounds__(256) rb_rightmul_kernel(const RefreshJob* __restrict__ jobs, int flip, int to_U) {
    const RefreshJob& j = jobs[blockIdx.y];
    const int d = j.d, k = j.k;
    const int r0 = blockIdx.x * 64;
    if (r0 >= d) return;
    extern __shared__ __align__(16) double s_rm[];             // RM_SMEM bytes
    double (*Vsh)[RM_LDV] = reinterpret_cast<double (*)[RM_LDV]>(s_rm);                       // Vsh[r][l]
    double (*Zsh)[RB_LD] = reinterpret_cast<double (*)[RB_LD]>(s_rm + 64 * RM_LDV);          // Zsh[l][c]
    double* V = j.buf[flip];
    for (int idx = threadIdx.x; idx < RB_MAXK * RB_MAXK; idx += 256) {
        const int l = idx >> 6, c = idx & 63;
        Zsh[l][c] = (l < k && c < k) ? j.Zs[(int64_t)l * k + c] : 0.0;
    }
    for (int idx = threadIdx.x; idx < 64 * RB_MAXK; idx += 256) {
        const int r = idx >> 6, l = idx & 63;
        Vsh[r][l] = (r0 + r < d && l < k) ? V[(int64_t)(r0 + r) * k + l] : 0.0;
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, fr = lane >> 2, fk = lane & 3;
    double acc[8][2] = {};
#pragma unroll
    for (int ks = 0; ks < RB_MAXK / 4; ++ks) {
        const double a = Vsh[8 * warp + fr][4 * ks + fk];
#pragma unroll
        for (int nb = 0; nb < 8; ++nb) dmma884(acc[nb][0], acc[nb][1], a, Zsh[4 * ks + fk][8 * nb + fr]);
    }
    const int gi = r0 + 8 * warp + fr;
    if (gi < d) {
#pragma unroll
        for (int nb = 0; nb < 8; ++nb) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int c = 8 * nb + 2 * fk + e;
                if (c >= k) continue;
                if (to_U) j.U[(int64_t)gi * k + c] = (float)acc[nb][e];
                else V[(int64_t)gi * k + c] = acc[nb][e];
            }
        }
    }
}

__global__ void __launch_bounds__(1024) rb_jacobi_kernel(const RefreshJob* __restrict__ jobs, int max_sweeps) {
    const RefreshJob& j = jobs[blockIdx.x];
    jacobi_body(j.Bm, j.Zm, j.k, 1, j.mu64, j.Zs, max_sweeps);
}

__global__ void __launch_bounds__(256) rb_multipliers_kernel(const RefreshJob* __restrict__ jobs) {
    const RefreshJob& j = jobs[blockIdx.x];
    multipliers_body(j.factor, j.d, j.k, j.mu64, nullptr, j.lam, 0.0, j.mu, j.e, j.ebar, j.rho);
}

// ---- Y = A V: buf[flip ^ 1] <- factor (d x d FP32) * buf[flip] (d x k FP64), FP64 accumulate -----------------------
// One CTA per 128-row block of one side (blockIdx.x walks the launch-wide block list), the whole K = d loop inside it.
// The product runs on the FP64 tensor-core path (mma.sync m8n8k4, DMMA): a warp owns 16 rows x 64 columns = 2 x 8 MMA
// tiles, so one K = 4 step is 2 + 8 fragment loads for 16 MMAs.  The CUDA-core version of this kernel (8 x 4 register tiles)
// was bound by shared-memory wavefronts at 47 % of the FP64 pipe (ncu: a 128-bit shared load costs four wavefronts per warp
// whatever it broadcasts); the fragments need a fifth of that traffic.  The A tile stays FP32 in shared memory (K-major)
// and is widened in registers; a warp of the loader takes 32 consecutive rows, so the transposing stores are
// conflict-free.  The next tile's global loads are in flight while the current one is multiplied.
__global__ void __launch_bounds__(256, 2) rb_av_kernel(const RefreshJob* __restrict__ jobs, int n_jobs, int flip) {
    extern __shared__ __align__(16) double s_av[];                  // AV_SMEM bytes
    double (*Vs)[AV_LDV] = reinterpret_cast<double (*)[AV_LDV]>(s_av);
    float (*As)[AV_LDA] = reinterpret_cast<float (*)[AV_LDA]>(s_av + AV_BK * AV_LDV);
    int lo = 0, hi = n_jobs - 1;
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (jobs[mid].blk0 <= (int)blockIdx.x) lo = mid; else hi = mid - 1; }
    const RefreshJob& j = jobs[lo];
    const int d = j.d, k = j.k;
    const int i0 = ((int)blockIdx.x - j.blk0) * AV_BM;
    const float* __restrict__ A = j.factor;
    const double* __restrict__ V = j.buf[flip];
    double* __restrict__ Y = j.buf[flip ^ 1];
    const int tid = threadIdx.x;
    // loader roles: A tile 128 rows x 32 floats = 1024 float4 (4 per thread: row = idx % 128, quad = idx / 128);
    //               V tile 32 rows x 64 doubles = 1024 double2 (4 per thread: row = idx / 32, pair = idx % 32)
    float4 pa[4];
    double2 pv[4];
    const bool vec_ok = (d & 3) == 0 && (k & 1) == 0;
    auto fetch = [&](int k0) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int idx = tid + 256 * u, row = idx & 127, quad = idx >> 7;
            const int gi = i0 + row, gl = k0 + 4 * quad;
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (gi < d) {
                const float* p = A + (int64_t)gi * d + gl;
                if (vec_ok && gl + 3 < d) v = __ldg(reinterpret_cast<const float4*>(p));
                else {
                    if (gl < d) v.x = p[0];
                    if (gl + 1 < d) v.y = p[1];
                    if (gl + 2 < d) v.z = p[2];
                    if (gl + 3 < d) v.w = p[3];
                }
            }
            pa[u] = v;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int idx = tid + 256 * u, row = idx >> 5, pair = idx & 31;
            const int gl = k0 + row, col = 2 * pair;
            double2 v = make_double2(0.0, 0.0);
            if (gl < d) {
                const double* p = V + (int64_t)gl * k + col;
                if (vec_ok && col + 1 < k) v = *reinterpret_cast<const double2*>(p);
                else {
                    if (col < k) v.x = p[0];
                    if (col + 1 < k) v.y = p[1];
                }
            }
            pv[u] = v;
        }
    };
    auto stash = [&]() {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int idx = tid + 256 * u, row = idx & 127, quad = idx >> 7;
            As[4 * quad][row] = pa[u].x; As[4 * quad + 1][row] = pa[u].y;
            As[4 * quad + 2][row] = pa[u].z; As[4 * quad + 3][row] = pa[u].w;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int idx = tid + 256 * u, row = idx >> 5, pair = idx & 31;
            *reinterpret_cast<double2*>(&Vs[row][2 * pair]) = pv[u];
        }
    };
    const int warp = tid >> 5, lane = tid & 31, fr = lane >> 2, fk = lane & 3;      // fragment row / column group, K index
    double acc[2][8][2] = {};
    fetch(0);
    for (int k0 = 0; k0 < d; k0 += AV_BK) {
        stash();
        __syncthreads();
        if (k0 + AV_BK < d) fetch(k0 + AV_BK);
#pragma unroll
        for (int ks = 0; ks < AV_BK / 4; ++ks) {
            const int kk = 4 * ks + fk;
            double a[2], b[8];
#pragma unroll
            for (int mb = 0; mb < 2; ++mb) a[mb] = (double)As[kk][16 * warp + 8 * mb + fr];
#pragma unroll
            for (int nb = 0; nb < 8; ++nb) b[nb] = Vs[kk][8 * nb + fr];
#pragma unroll
            for (int mb = 0; mb < 2; ++mb)
#pragma unroll
                for (int nb = 0; nb < 8; ++nb)
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                                 : "+d"(acc[mb][nb][0]), "+d"(acc[mb][nb][1]) : "d"(a[mb]), "d"(b[nb]));
        }
        __syncthreads();
    }
#pragma unroll
    for (int mb = 0; mb < 2; ++mb) {
        const int gi = i0 + 16 * warp + 8 * mb + fr;
        if (gi >= d) continue;
#pragma unroll
        for (int nb = 0; nb < 8; ++nb) {
            const int col = 8 * nb + 2 * fk;
            if (col < k) Y[(int64_t)gi * k + col] = acc[mb][nb][0];
            if (col + 1 < k) Y[(int64_t)gi * k + col + 1] = acc[mb][nb][1];
        }
    }
}

// ---- U (d x k FP32) -> U16 (d x kp BF16, zero-padded), its transpose Ut16 (kp x d) and the residuals U - bf16(U) --------
// (the per-side pack_basis_kernel of gf8_fast.cuh, for all sides of the call in one launch)
__global__ void __launch_bounds__(256) rb_pack_kernel(const RefreshJob* __restrict__ jobs) {
    const RefreshJob& j = jobs[blockIdx.y];
    if (!j.U16) return;
    const int d = j.d, k = j.k, kp = j.kp;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < (int64_t)d * kp; idx += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(idx / kp), col = (int)(idx % kp);
        const float x = col < k ? j.U[(int64_t)i * k + col] : 0.0f;
        const __nv_bfloat16 v = __float2bfloat16_rn(x);
        const __nv_bfloat16 lo = __float2bfloat16_rn(x - __bfloat162float(v));
        j.U16[idx] = v;
        j.Ut16[(int64_t)col * d + i] = v;
        j.U16_lo[idx] = lo;
        j.Ut16_lo[(int64_t)col * d + i] = lo;
    }
}

}  // namespace rb
}  // namespace gf8
