// gf8_quant.cuh -- streaming kernels of the shared FP8 communication core (Fig. 4):
//   a5 amax + scale, a6 cast (Alg. 1 l.12-13), a7 reduce (Eq. 1; Alg. 1 l.20-21).
// All HBM-bound: 16-byte vectorised BF16 / FP32 / FP8 traffic, warp shuffle + one atomic per CTA.
#pragma once
#include "gf8_common.cuh"

namespace gf8 {

// ---- a5: per-tensor amax over a contiguous tensor ------------------------------------------------
// amax_bits must be zero on entry.  numel % 16 == 0, 16-byte aligned.
template <typename T>
__global__ void __launch_bounds__(256) amax_tensor_kernel(const T* __restrict__ x, int64_t numel,
                                                          uint32_t* __restrict__ amax_bits) {
    const uint4* xv = reinterpret_cast<const uint4*>(x);
    const int64_t nvec = numel * (int64_t)sizeof(T) / 16;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    uint32_t loc = 0;
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < nvec; i += 4 * stride) {            // 4 independent 16-byte loads in flight
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = ld_stream(xv + i + u * stride);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (sizeof(T) == 2) {
                const uint32_t w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
#pragma unroll
                for (int k = 0; k < 4; ++k) loc = max(loc, max((w[k] << 16) & 0x7FFF0000u, w[k] & 0x7FFF0000u));
            } else {
                loc = max(max(loc, v[u].x & 0x7FFFFFFFu), max(v[u].y & 0x7FFFFFFFu,
                          max(v[u].z & 0x7FFFFFFFu, v[u].w & 0x7FFFFFFFu)));
            }
        }
    }
    for (; i < nvec; i += stride) {
        const uint4 v = ld_stream(xv + i);
        if (sizeof(T) == 2) {
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) loc = max(loc, max((w[k] << 16) & 0x7FFF0000u, w[k] & 0x7FFF0000u));
        } else {
            loc = max(max(loc, v.x & 0x7FFFFFFFu), max(v.y & 0x7FFFFFFFu, max(v.z & 0x7FFFFFFFu, v.w & 0x7FFFFFFFu)));
        }
    }
    block_atomic_max_bits(loc, amax_bits);
}

// ---- a5: per-128x128-block amax; one CTA per block, no atomics ------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) amax_block_kernel(const T* __restrict__ x, int64_t m, int64_t n,
                                                         uint32_t* __restrict__ amax_bits) {
    constexpr int VEC = 16 / sizeof(T);
    const int64_t r0 = (int64_t)blockIdx.y * 128, c0 = (int64_t)blockIdx.x * 128;
    const int rows = (int)min((int64_t)128, m - r0), cols = (int)min((int64_t)128, n - c0);
    const int vpr = cols / VEC;                                    // vectors per row (cols % 16 == 0)
    uint32_t loc = 0;
    for (int idx = threadIdx.x; idx < rows * vpr; idx += blockDim.x) {
        const int r = idx / vpr, cv = idx % vpr;
        const uint4 v = ld_stream(reinterpret_cast<const uint4*>(x + (r0 + r) * n + c0) + cv);
        if (sizeof(T) == 2) {
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) loc = max(loc, max((w[k] << 16) & 0x7FFF0000u, w[k] & 0x7FFF0000u));
        } else {
            loc = max(max(loc, v.x & 0x7FFFFFFFu), max(v.y & 0x7FFFFFFFu, max(v.z & 0x7FFFFFFFu, v.w & 0x7FFFFFFFu)));
        }
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

// ---- scale = fmax / amax, scale_inv = amax / fmax (one IEEE FP32 division each; S6) ------
// amax == 0, amax not finite or scale not finite => both 1 (S13).
__device__ __forceinline__ void scales_from_amax(uint32_t bits, float fmax, float& scale, float& scale_inv) {
    const float amax = __uint_as_float(bits);
    scale = __fdiv_rn(fmax, amax);
    scale_inv = __fdiv_rn(amax, fmax);
    if (bits == 0u || bits >= 0x7F800000u || !(fabsf(scale) <= 3.402823466e38f)) { scale = 1.0f; scale_inv = 1.0f; }
}

__global__ void scales_kernel(const uint32_t* __restrict__ amax_bits, int n, float fmax, float* __restrict__ scale,
                              float* __restrict__ scale_inv) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float s, si;
    scales_from_amax(amax_bits[i], fmax, s, si);
    scale[i] = s;
    scale_inv[i] = si;
}

// ---- a6: cast.  Each thread handles 16 consecutive elements of one row (n % 16 == 0) -------------
template <typename T, int FMT>
__global__ void __launch_bounds__(256) cast_kernel(const T* __restrict__ x, int64_t m, int64_t n, int scaling,
                                                   const float* __restrict__ scale, uint8_t* __restrict__ codes) {
    const int64_t ngroups = m * n / 16;
    const int64_t bn = (n + 127) / 128;
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
#pragma unroll
        for (int u = 0; u < 16; ++u) f[u] = __fmul_rn(f[u], s);
        uint4 o;
        o.x = f32x4_to_fp8x4<FMT>(f[0], f[1], f[2], f[3]);
        o.y = f32x4_to_fp8x4<FMT>(f[4], f[5], f[6], f[7]);
        o.z = f32x4_to_fp8x4<FMT>(f[8], f[9], f[10], f[11]);
        o.w = f32x4_to_fp8x4<FMT>(f[12], f[13], f[14], f[15]);
        st_stream(reinterpret_cast<uint4*>(codes + e0), o);
    }
}

// ---- a7: reduce R payloads in FP32, rank order, fused multiply-add, then * (1/R) -------------------
struct ReducePtrs {
    const uint8_t* codes[64];
    const float* sinv[64];
};

// OutT = float (scratch / FP32 output) or bf16 (Euclidean tensors decoded straight to BF16).
template <int FMT, typename OutT>
__global__ void __launch_bounds__(256) reduce_kernel(const __grid_constant__ ReducePtrs p, int R, int average,
                                                     int64_t m, int64_t n, int scaling, OutT* __restrict__ out,
                                                     bf16* __restrict__ out16 = nullptr, bf16* __restrict__ out16_lo = nullptr) {
    const int64_t ngroups = m * n / 16;
    const int64_t bn = (n + 127) / 128;
    const float invR = __fdiv_rn(1.0f, (float)R);
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < ngroups; g += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e0 = g * 16;
        int64_t sidx = 0;
        if (scaling != 0) { const int64_t r = e0 / n, c = e0 % n; sidx = (r / 128) * bn + c / 128; }
        float acc[16];
#pragma unroll
        for (int u = 0; u < 16; ++u) acc[u] = 0.0f;
        for (int r = 0; r < R; ++r) {
            const uint4 c = ld_stream(reinterpret_cast<const uint4*>(p.codes[r] + e0));
            const float s = __ldg(p.sinv[r] + sidx);
            float v[16];
            fp8x4_to_f32x4<FMT>(c.x, v); fp8x4_to_f32x4<FMT>(c.y, v + 4);
            fp8x4_to_f32x4<FMT>(c.z, v + 8); fp8x4_to_f32x4<FMT>(c.w, v + 12);
#pragma unroll
            for (int u = 0; u < 16; ++u) acc[u] = __fmaf_rn(v[u], s, acc[u]);
        }
        if (average) {
#pragma unroll
            for (int u = 0; u < 16; ++u) acc[u] = __fmul_rn(acc[u], invR);
        }
        if (sizeof(OutT) == 4) {
            if (out) {
                uint4* o = reinterpret_cast<uint4*>(reinterpret_cast<float*>(out) + e0);
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    st_stream(o + u, make_uint4(__float_as_uint(acc[4 * u]), __float_as_uint(acc[4 * u + 1]),
                                                __float_as_uint(acc[4 * u + 2]), __float_as_uint(acc[4 * u + 3])));
            }
            if (out16) {      // BF16 copy: the tensor-core operand of the unwhitening projections (FAST path)
                uint32_t w[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const __nv_bfloat162 h = __floats2bfloat162_rn(acc[2 * u], acc[2 * u + 1]);
                    w[u] = *reinterpret_cast<const uint32_t*>(&h);
                }
                uint4* o2 = reinterpret_cast<uint4*>(out16 + e0);
                o2[0] = make_uint4(w[0], w[1], w[2], w[3]);
                o2[1] = make_uint4(w[4], w[5], w[6], w[7]);
                if (out16_lo) {   // residual acc - bf16(acc): hi + lo carries ~16 mantissa bits into the MMAs
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const float2 hi = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&w[u]));
                        const __nv_bfloat162 h = __floats2bfloat162_rn(acc[2 * u] - hi.x, acc[2 * u + 1] - hi.y);
                        w[u] = *reinterpret_cast<const uint32_t*>(&h);
                    }
                    uint4* o3 = reinterpret_cast<uint4*>(out16_lo + e0);
                    o3[0] = make_uint4(w[0], w[1], w[2], w[3]);
                    o3[1] = make_uint4(w[4], w[5], w[6], w[7]);
                }
            }
        } else {
            uint32_t w[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const __nv_bfloat162 h = __floats2bfloat162_rn(acc[2 * u], acc[2 * u + 1]);
                w[u] = *reinterpret_cast<const uint32_t*>(&h);
            }
            uint4* o = reinterpret_cast<uint4*>(reinterpret_cast<bf16*>(out) + e0);
            st_stream(o, make_uint4(w[0], w[1], w[2], w[3]));
            st_stream(o + 1, make_uint4(w[4], w[5], w[6], w[7]));
        }
    }
}

// Grouped form of the reduction for the FAST decode path: up to 22 tensors per launch (the jobs travel as kernel
// parameters), R <= 8 payloads each, result written as hi + lo BF16 (the operands of the unwhitening MMAs).
// Block b covers 1024 16-element groups of its job; a thread keeps all R 16-byte loads of a group in flight.
// Same arithmetic as reduce_kernel: acc = fma(value_r, scale_inv_r, acc) in rank order, then * (1/R).
constexpr int REDUCE_MAX_JOBS = 22, REDUCE_GROUPS_PER_BLOCK = 1024;
struct ReduceJob {
    const uint8_t* codes[8];
    const float* sinv[8];
    bf16* out16;
    bf16* out16_lo;
    int64_t n_groups;             // m * n / 16
    int64_t n;                    // columns (block scaling only)
    int64_t first_block;          // first block of this job in the launch
};
struct ReduceBatch {
    int32_t n_jobs, R, average, scaling;
    ReduceJob job[REDUCE_MAX_JOBS];
};

template <int FMT>
__global__ void __launch_bounds__(256) reduce_many_kernel(const __grid_constant__ ReduceBatch b) {
    int j = 0;
    while (j + 1 < b.n_jobs && (int64_t)blockIdx.x >= b.job[j + 1].first_block) ++j;
    const ReduceJob& jb = b.job[j];
    const int R = b.R;
    const float invR = __fdiv_rn(1.0f, (float)R);
    const int64_t g0 = ((int64_t)blockIdx.x - jb.first_block) * REDUCE_GROUPS_PER_BLOCK;
    const int64_t bn = (jb.n + 127) / 128;
#pragma unroll 1
    for (int it = 0; it < REDUCE_GROUPS_PER_BLOCK / 256; ++it) {
        const int64_t g = g0 + it * 256 + threadIdx.x;
        if (g >= jb.n_groups) break;
        const int64_t e0 = g * 16;
        int64_t sidx = 0;
        if (b.scaling != 0) { const int64_t r = e0 / jb.n, c = e0 % jb.n; sidx = (r / 128) * bn + c / 128; }
        uint4 c[8];
        float s[8];
#pragma unroll
        for (int r = 0; r < 8; ++r)
            if (r < R) { c[r] = ld_stream(reinterpret_cast<const uint4*>(jb.codes[r] + e0)); s[r] = __ldg(jb.sinv[r] + sidx); }
        float acc[16];
#pragma unroll
        for (int u = 0; u < 16; ++u) acc[u] = 0.0f;
#pragma unroll
        for (int r = 0; r < 8; ++r)
            if (r < R) {
                float v[16];
                fp8x4_to_f32x4<FMT>(c[r].x, v); fp8x4_to_f32x4<FMT>(c[r].y, v + 4);
                fp8x4_to_f32x4<FMT>(c[r].z, v + 8); fp8x4_to_f32x4<FMT>(c[r].w, v + 12);
#pragma unroll
                for (int u = 0; u < 16; ++u) acc[u] = __fmaf_rn(v[u], s[r], acc[u]);
            }
        if (b.average) {
#pragma unroll
            for (int u = 0; u < 16; ++u) acc[u] = __fmul_rn(acc[u], invR);
        }
        uint32_t w[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const __nv_bfloat162 h = __floats2bfloat162_rn(acc[2 * u], acc[2 * u + 1]);
            w[u] = *reinterpret_cast<const uint32_t*>(&h);
        }
        uint4* o2 = reinterpret_cast<uint4*>(jb.out16 + e0);
        o2[0] = make_uint4(w[0], w[1], w[2], w[3]);
        o2[1] = make_uint4(w[4], w[5], w[6], w[7]);
        if (jb.out16_lo) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const float2 hi = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&w[u]));
                const __nv_bfloat162 h = __floats2bfloat162_rn(acc[2 * u] - hi.x, acc[2 * u + 1] - hi.y);
                w[u] = *reinterpret_cast<const uint32_t*>(&h);
            }
            uint4* o3 = reinterpret_cast<uint4*>(jb.out16_lo + e0);
            o3[0] = make_uint4(w[0], w[1], w[2], w[3]);
            o3[1] = make_uint4(w[4], w[5], w[6], w[7]);
        }
    }
}

// Grouped plain FP8 encode of BF16 tensors with a per-tensor scale (the Euclidean tensors of a batched call): one amax
// launch and one cast launch for up to 22 tensors instead of three launches per tensor.  Non-persistent grids (a block
// = 4096 16-byte vectors), so on SMs that hold a tensor-core CTA their blocks fill in one at a time as room allows.
// Same arithmetic as amax_tensor_kernel + scales_kernel + cast_kernel.
constexpr int QUANT_MAX_JOBS = 22, QUANT_VEC_PER_BLOCK = 4096;
struct QuantJob {
    const bf16* x;
    uint8_t* codes;
    float* scale_inv;
    uint32_t* amax_bits;          // zero before the amax launch
    int64_t nvec;                 // numel / 8 (16-byte vectors of BF16)
    int64_t first_block;
};
struct QuantBatch {
    int32_t n_jobs, pad;
    QuantJob job[QUANT_MAX_JOBS];
};

__global__ void __launch_bounds__(256) amax_many_kernel(const __grid_constant__ QuantBatch b) {
    int j = 0;
    while (j + 1 < b.n_jobs && (int64_t)blockIdx.x >= b.job[j + 1].first_block) ++j;
    const QuantJob& jb = b.job[j];
    const uint4* xv = reinterpret_cast<const uint4*>(jb.x);
    const int64_t v0 = ((int64_t)blockIdx.x - jb.first_block) * QUANT_VEC_PER_BLOCK;
    uint32_t loc = 0;
#pragma unroll 1
    for (int it = 0; it < QUANT_VEC_PER_BLOCK / 1024; ++it) {
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int64_t i = v0 + it * 1024 + u * 256 + threadIdx.x;
            v[u] = i < jb.nvec ? ld_stream(xv + i) : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
#pragma unroll
            for (int k = 0; k < 4; ++k) loc = max(loc, max((w[k] << 16) & 0x7FFF0000u, w[k] & 0x7FFF0000u));
        }
    }
    block_atomic_max_bits(loc, jb.amax_bits);
}

template <int FMT>
__global__ void __launch_bounds__(256) cast_many_kernel(const __grid_constant__ QuantBatch b) {
    int j = 0;
    while (j + 1 < b.n_jobs && (int64_t)blockIdx.x >= b.job[j + 1].first_block) ++j;
    const QuantJob& jb = b.job[j];
    float s, si;
    scales_from_amax(*jb.amax_bits, FMT == 0 ? 448.0f : 57344.0f, s, si);
    if ((int64_t)blockIdx.x == jb.first_block && threadIdx.x == 0) *jb.scale_inv = si;
    const int64_t ngroups = jb.nvec / 2;                          // 16 elements = two 16-byte vectors in, one out
    const int64_t g0 = ((int64_t)blockIdx.x - jb.first_block) * (QUANT_VEC_PER_BLOCK / 2);
#pragma unroll 1
    for (int it = 0; it < QUANT_VEC_PER_BLOCK / 2 / 512; ++it) {
        uint4 a[2] = {make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0)}, c[2] = {make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0)};
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int64_t g = g0 + it * 512 + u * 256 + threadIdx.x;
            if (g < ngroups) {
                const uint4* p = reinterpret_cast<const uint4*>(jb.x + g * 16);
                a[u] = ld_stream(p); c[u] = ld_stream(p + 1);
            }
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int64_t g = g0 + it * 512 + u * 256 + threadIdx.x;
            if (g >= ngroups) continue;
            float f[16];
            unpack_bf16x8(a[u], f);
            unpack_bf16x8(c[u], f + 8);
#pragma unroll
            for (int k = 0; k < 16; ++k) f[k] = __fmul_rn(f[k], s);
            uint4 o;
            o.x = f32x4_to_fp8x4<FMT>(f[0], f[1], f[2], f[3]);
            o.y = f32x4_to_fp8x4<FMT>(f[4], f[5], f[6], f[7]);
            o.z = f32x4_to_fp8x4<FMT>(f[8], f[9], f[10], f[11]);
            o.w = f32x4_to_fp8x4<FMT>(f[12], f[13], f[14], f[15]);
            st_stream(reinterpret_cast<uint4*>(jb.codes + g * 16), o);
        }
    }
}

// FP32 -> BF16 (RNE) / FP32 copy of a contiguous tensor, and BF16 -> FP32 widening.
template <typename TI, typename TO>
__global__ void __launch_bounds__(256) convert_kernel(const TI* __restrict__ in, int64_t numel, TO* __restrict__ out) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < numel; i += (int64_t)gridDim.x * blockDim.x) {
        const float v = ldf<TI>(in, i);
        if (sizeof(TO) == 4) reinterpret_cast<float*>(out)[i] = v;
        else reinterpret_cast<bf16*>(out)[i] = __float2bfloat16_rn(v);
    }
}

}  // namespace gf8
