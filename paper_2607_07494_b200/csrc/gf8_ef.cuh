// gf8_ef.cuh -- f1: error feedback in the transformed coordinates (PAPER.md:318 Alg. 1 l.11-15; :354; S10).
//   U~ = U + R;  s = Scale(U~);  Q~ = Q(U~; s);  R <- U~ - Dequantize(Q~; s)
// U is the whitened gradient (FP32, written by the codec's tap path) or, for a Euclidean tensor, the gradient itself;
// R is a caller-owned FP32 buffer of the tensor's shape (one per tensor and rank, zero before the first step).
// Streaming kernels, HBM-bound: the amax pass reads U and R (8 B / element for FP32 U), the cast pass reads both again
// and writes the code and the new residual (8 + 1 + 4).  Every element sees exactly the FP32 operations of the oracle
// (O8), one rounding each -- add, multiply by scale, cast, multiply by scale_inv, subtract -- so codes, scales and the
// residual are bit-identical to it on the same U.
#pragma once
#include "gf8_common.cuh"
#include "gf8_quant.cuh"

namespace gf8 {

template <typename T>
__device__ __forceinline__ void ef_load16(const T* __restrict__ u, const float* __restrict__ resid, int64_t e0, float* ut) {
    float f[16];
    if (sizeof(T) == 2) {
        const uint4* p = reinterpret_cast<const uint4*>(u + e0);
        const uint4 a = ld_stream(p), b = ld_stream(p + 1);
        unpack_bf16x8(a, f);
        unpack_bf16x8(b, f + 8);
    } else {
        const uint4* p = reinterpret_cast<const uint4*>(u + e0);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint4 a = ld_stream(p + q);
            f[4 * q] = __uint_as_float(a.x); f[4 * q + 1] = __uint_as_float(a.y);
            f[4 * q + 2] = __uint_as_float(a.z); f[4 * q + 3] = __uint_as_float(a.w);
        }
    }
    const uint4* pr = reinterpret_cast<const uint4*>(resid + e0);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const uint4 a = ld_stream(pr + q);
        ut[4 * q] = __fadd_rn(f[4 * q], __uint_as_float(a.x)); ut[4 * q + 1] = __fadd_rn(f[4 * q + 1], __uint_as_float(a.y));
        ut[4 * q + 2] = __fadd_rn(f[4 * q + 2], __uint_as_float(a.z)); ut[4 * q + 3] = __fadd_rn(f[4 * q + 3], __uint_as_float(a.w));
    }
}

// amax of U + R.  scaling == 0: one slot (zero on entry), grid-stride, one atomic per CTA.  scaling == 1: the grid is
// (column blocks, row blocks), one CTA per 128 x 128 block, no atomics.  Each thread takes 16 consecutive elements of a row.
template <typename T>
__global__ void __launch_bounds__(256) ef_amax_kernel(const T* __restrict__ u, const float* __restrict__ resid, int64_t m,
                                                      int64_t n, int scaling, uint32_t* __restrict__ amax_bits) {
    uint32_t loc = 0;
    float ut[16];
    if (scaling == 0) {
        const int64_t ngroups = m * n / 16;
        for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < ngroups; g += (int64_t)gridDim.x * blockDim.x) {
            ef_load16<T>(u, resid, g * 16, ut);
#pragma unroll
            for (int q = 0; q < 16; ++q) loc = max(loc, __float_as_uint(ut[q]) & 0x7FFFFFFFu);
        }
        block_atomic_max_bits(loc, amax_bits);
        return;
    }
    const int64_t r0 = (int64_t)blockIdx.y * 128, c0 = (int64_t)blockIdx.x * 128;
    const int rows = (int)min((int64_t)128, m - r0), cols = (int)min((int64_t)128, n - c0);
    const int gpr = cols / 16;
    for (int idx = threadIdx.x; idx < rows * gpr; idx += blockDim.x) {
        ef_load16<T>(u, resid, (r0 + idx / gpr) * n + c0 + 16 * (idx % gpr), ut);
#pragma unroll
        for (int q = 0; q < 16; ++q) loc = max(loc, __float_as_uint(ut[q]) & 0x7FFFFFFFu);
    }
    __shared__ uint32_t s_warp[8];
    loc = warp_max_u32(loc);
    if ((threadIdx.x & 31) == 0) s_warp[threadIdx.x >> 5] = loc;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t v = 0;
        for (int w = 0; w < 8; ++w) v = max(v, s_warp[w]);
        amax_bits[(int64_t)blockIdx.y * gridDim.x + blockIdx.x] = v;
    }
}

// code = cast((U + R) * scale);  R <- (U + R) - val(code) * scale_inv
template <typename T, int FMT>
__global__ void __launch_bounds__(256) ef_cast_kernel(const T* __restrict__ u, float* __restrict__ resid, int64_t m, int64_t n,
                                                      int scaling, const float* __restrict__ scale,
                                                      const float* __restrict__ scale_inv, uint8_t* __restrict__ codes) {
    const int64_t ngroups = m * n / 16;
    const int64_t bn = (n + 127) / 128;
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < ngroups; g += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e0 = g * 16;
        int64_t sidx = 0;
        if (scaling != 0) { const int64_t r = e0 / n, c = e0 % n; sidx = (r / 128) * bn + c / 128; }
        const float s = __ldg(scale + sidx), si = __ldg(scale_inv + sidx);
        float ut[16], y[16];
        ef_load16<T>(u, resid, e0, ut);
#pragma unroll
        for (int q = 0; q < 16; ++q) y[q] = __fmul_rn(ut[q], s);
        uint4 o;
        o.x = f32x4_to_fp8x4<FMT>(y[0], y[1], y[2], y[3]);
        o.y = f32x4_to_fp8x4<FMT>(y[4], y[5], y[6], y[7]);
        o.z = f32x4_to_fp8x4<FMT>(y[8], y[9], y[10], y[11]);
        o.w = f32x4_to_fp8x4<FMT>(y[12], y[13], y[14], y[15]);
        st_stream(reinterpret_cast<uint4*>(codes + e0), o);
        const uint32_t w[4] = {o.x, o.y, o.z, o.w};
        float r[16];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            float v[4];
            fp8x4_to_f32x4<FMT>(w[q], v);
#pragma unroll
            for (int t = 0; t < 4; ++t) r[4 * q + t] = __fsub_rn(ut[4 * q + t], __fmul_rn(v[t], si));
        }
        uint4* pr = reinterpret_cast<uint4*>(resid + e0);
#pragma unroll
        for (int q = 0; q < 4; ++q)
            st_stream(pr + q, make_uint4(__float_as_uint(r[4 * q]), __float_as_uint(r[4 * q + 1]), __float_as_uint(r[4 * q + 2]),
                                         __float_as_uint(r[4 * q + 3])));
    }
}

}  // namespace gf8

// ---- f2 / f3: cast with an externally agreed amax, boundary-hit counters fused into it ------------------------------------
// (Alg. 1 l.4-5 and l.17-19: s <- AllReduce_MAX(s); "count how often encoded values hit the
//  upper and lower FP8 boundaries".)  scale / scale_inv follow from amax_sync by the quantizer's rule (scales_kernel);
//  upper hit: |code| is the largest finite value; lower hit: x != 0 and |code| is zero or the smallest subnormal.
//  hits (nullable): two 64-bit counters, accumulated with one atomic pair per CTA.
namespace gf8 {

template <typename T, int FMT>
__global__ void __launch_bounds__(256) cast_scaled_kernel(const T* __restrict__ x, int64_t m, int64_t n, int scaling,
                                                          const float* __restrict__ scale, uint8_t* __restrict__ codes,
                                                          unsigned long long* __restrict__ hits) {
    constexpr uint32_t TOP = FMT == 0 ? 0x7Eu : 0x7Bu;        // E4M3 448 = S.1111.110, E5M2 57344 = S.11110.11
    const int64_t ngroups = m * n / 16;
    const int64_t bn = (n + 127) / 128;
    uint32_t up = 0, lo = 0;
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < ngroups; g += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e0 = g * 16;
        float s;
        if (scaling == 0) s = __ldg(scale);
        else { const int64_t r = e0 / n, c = e0 % n; s = __ldg(scale + (r / 128) * bn + c / 128); }
        float f[16];
        if (sizeof(T) == 2) {
            const uint4* p = reinterpret_cast<const uint4*>(x + e0);
            const uint4 a = ld_stream(p), b = ld_stream(p + 1);
            unpack_bf16x8(a, f);
            unpack_bf16x8(b, f + 8);
        } else {
            const uint4* p = reinterpret_cast<const uint4*>(x + e0);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint4 a = ld_stream(p + u);
                f[4 * u] = __uint_as_float(a.x); f[4 * u + 1] = __uint_as_float(a.y);
                f[4 * u + 2] = __uint_as_float(a.z); f[4 * u + 3] = __uint_as_float(a.w);
            }
        }
        uint32_t w[4];
#pragma unroll
        for (int q = 0; q < 4; ++q)
            w[q] = f32x4_to_fp8x4<FMT>(__fmul_rn(f[4 * q], s), __fmul_rn(f[4 * q + 1], s), __fmul_rn(f[4 * q + 2], s), __fmul_rn(f[4 * q + 3], s));
        st_stream(reinterpret_cast<uint4*>(codes + e0), make_uint4(w[0], w[1], w[2], w[3]));
        if (hits) {
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const uint32_t mag = (w[q >> 2] >> (8 * (q & 3))) & 0x7Fu;
                up += mag == TOP;
                lo += (mag <= 1u) && (f[q] != 0.0f);
            }
        }
    }
    if (hits) {
        __shared__ uint32_t s_up[8], s_lo[8];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { up += __shfl_xor_sync(0xFFFFFFFFu, up, o); lo += __shfl_xor_sync(0xFFFFFFFFu, lo, o); }
        if ((threadIdx.x & 31) == 0) { s_up[threadIdx.x >> 5] = up; s_lo[threadIdx.x >> 5] = lo; }
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned long long u = 0, l = 0;
            for (int q = 0; q < 8; ++q) { u += s_up[q]; l += s_lo[q]; }
            if (u) atomicAdd(hits, u);
            if (l) atomicAdd(hits + 1, l);
        }
    }
}

__global__ void amax_bits_to_float_kernel(const uint32_t* __restrict__ bits, int n, float* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = __uint_as_float(bits[i]);
}
__global__ void scales_from_float_kernel(const float* __restrict__ amax, int n, float fmax, float* __restrict__ scale,
                                         float* __restrict__ scale_inv) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float s, si;
    scales_from_amax(__float_as_uint(amax[i]) & 0x7FFFFFFFu, fmax, s, si);
    scale[i] = s;
    scale_inv[i] = si;
}

}  // namespace gf8
