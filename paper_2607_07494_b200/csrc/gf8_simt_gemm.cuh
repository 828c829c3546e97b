// gf8_simt_gemm.cuh -- a plain strided CUDA-core GEMM.
//
// It is the FP32 / FP64 reference arithmetic of the library: the EXACT transform path at small
// rank, every k x k and d x k product of the basis refresh (FP64 accumulate), and the yardstick the
// tensor-core kernels are debugged against on the GPU.  Operands are addressed by strides so the
// transposes of Eq. 14 / Eq. 4 (U_G^T Wg, X^T X) need no copies.
//
//   C[i][j] = rowscale[i] * ( alpha * sum_l A(i,l) * lscale[l] * B(l,j) + beta * C[i][j] )
//   A(i,l) = A[i*sa_i + l*sa_l],  B(l,j) = B[l*sb_l + j*sb_j],  C row-major with leading dim ldc.
// gridDim.z > 1 splits K; each split writes its partial product to the workspace g.ws and splitk_sum_kernel adds them up in
// split order (deterministic); without a workspace the partial sums are added into C atomically (caller pre-sets C).
#pragma once
#include "gf8_common.cuh"

namespace gf8 {

template <typename TA, typename TB, typename TC, typename TAcc>
struct GemmArgs {
    const TA* A; int64_t sa_i, sa_l;
    const TB* B; int64_t sb_l, sb_j;
    TC* C; int64_t ldc;
    int M, N, K;
    const float* lscale;    // length K or nullptr
    const float* rowscale;  // length M or nullptr
    TAcc alpha, beta;
    TAcc* ws;               // split-K workspace [gridDim.z][M][N] (deterministic: summed in split order by splitk_sum_kernel),
                            // or nullptr: partial sums are added into C atomically
};

template <typename TC, typename TAcc> __device__ __forceinline__ void store_c(TC* p, TAcc v);
template <> __device__ __forceinline__ void store_c<float, float>(float* p, float v) { *p = v; }
template <> __device__ __forceinline__ void store_c<float, double>(float* p, double v) { *p = (float)v; }
template <> __device__ __forceinline__ void store_c<double, double>(double* p, double v) { *p = v; }

constexpr int SG_BM = 64, SG_BN = 64, SG_BK = 16;

template <typename TA, typename TB, typename TC, typename TAcc>
__global__ void __launch_bounds__(256) simt_gemm_kernel(const GemmArgs<TA, TB, TC, TAcc> g) {
    __shared__ TAcc As[SG_BK][SG_BM + 4];
    __shared__ TAcc Bs[SG_BK][SG_BN + 4];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int i0 = blockIdx.y * SG_BM, j0 = blockIdx.x * SG_BN;
    // K range of this split
    const int nsplit = gridDim.z;
    const int kchunks = (g.K + SG_BK - 1) / SG_BK;
    const int cps = (kchunks + nsplit - 1) / nsplit;
    const int kbeg = blockIdx.z * cps * SG_BK, kend = min(g.K, (int)(blockIdx.z + 1) * cps * SG_BK);

    TAcc acc[4][4];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[r][c] = (TAcc)0;

    const bool a_kcontig = (g.sa_l == 1);
    const bool b_jcontig = (g.sb_j == 1);
    for (int k0 = kbeg; k0 < kend; k0 += SG_BK) {
        // A tile: 64 x 16 -> As[l][i]
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            int li, ii;
            if (a_kcontig) { ii = tid >> 2; li = (tid & 3) * 4 + u; }
            else { li = tid >> 4; ii = (tid & 15) * 4 + u; }
            const int gi = i0 + ii, gl = k0 + li;
            TAcc v = (TAcc)0;
            if (gi < g.M && gl < kend) {
                v = ld_as<TAcc, TA>(g.A, (int64_t)gi * g.sa_i + (int64_t)gl * g.sa_l);
                if (g.lscale) v *= (TAcc)g.lscale[gl];
            }
            As[li][ii] = v;
        }
        // B tile: 16 x 64 -> Bs[l][j]
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            int li, ji;
            if (b_jcontig) { li = tid >> 4; ji = (tid & 15) * 4 + u; }
            else { ji = tid >> 2; li = (tid & 3) * 4 + u; }
            const int gj = j0 + ji, gl = k0 + li;
            TAcc v = (TAcc)0;
            if (gj < g.N && gl < kend) v = ld_as<TAcc, TB>(g.B, (int64_t)gl * g.sb_l + (int64_t)gj * g.sb_j);
            Bs[li][ji] = v;
        }
        __syncthreads();
#pragma unroll
        for (int l = 0; l < SG_BK; ++l) {
            TAcc a[4], b[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) a[r] = As[l][ty * 4 + r];
#pragma unroll
            for (int c = 0; c < 4; ++c) b[c] = Bs[l][tx * 4 + c];
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[r][c] = fma(a[r], b[c], acc[r][c]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int gi = i0 + ty * 4 + r;
        if (gi >= g.M) continue;
        const TAcc rs = g.rowscale ? (TAcc)g.rowscale[gi] : (TAcc)1;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int gj = j0 + tx * 4 + c;
            if (gj >= g.N) continue;
            TC* p = g.C + (int64_t)gi * g.ldc + gj;
            if (nsplit > 1 && g.ws) {
                g.ws[((int64_t)blockIdx.z * g.M + gi) * g.N + gj] = rs * g.alpha * acc[r][c];
            } else if (nsplit > 1) {
                atomicAdd(p, (TC)(rs * g.alpha * acc[r][c]));
            } else {
                TAcc v = g.alpha * acc[r][c];
                if (g.beta != (TAcc)0) v += g.beta * (TAcc)(*p);
                store_c<TC, TAcc>(p, rs * v);
            }
        }
    }
}

// C[i][j] = (beta != 0 ? rowscale[i] * beta * C[i][j] : 0) + sum over splits z = 0, 1, ... of ws[z][i][j]  (fixed order)
template <typename TC, typename TAcc>
__global__ void __launch_bounds__(256) splitk_sum_kernel(const TAcc* __restrict__ ws, int splits, int M, int N, TC* __restrict__ C,
                                                         int64_t ldc, TAcc beta, const float* __restrict__ rowscale) {
    const int64_t total = (int64_t)M * N;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(idx / N), j = (int)(idx % N);
        TC* p = C + (int64_t)i * ldc + j;
        TAcc s = (TAcc)0;
        if (beta != (TAcc)0) s = (rowscale ? (TAcc)rowscale[i] : (TAcc)1) * beta * (TAcc)(*p);
        for (int z = 0; z < splits; ++z) s += ws[(int64_t)z * total + idx];
        store_c<TC, TAcc>(p, s);
    }
}

}  // namespace gf8
