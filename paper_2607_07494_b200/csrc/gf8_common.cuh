// gf8_common.cuh -- small device helpers shared by the gf8 kernels (sm_100a).
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_fp8.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gf8 {

typedef __nv_bfloat16 bf16;

// ---- streaming 16-byte global access (Guideline 13/14: read-once data bypasses L1) ---------------
__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream(uint4* p, const uint4& v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// ---- element loads as float / double --------------------------------------------------------------
template <typename T> __device__ __forceinline__ float ldf(const T* p, int64_t i);
template <> __device__ __forceinline__ float ldf<float>(const float* p, int64_t i) { return p[i]; }
template <> __device__ __forceinline__ float ldf<bf16>(const bf16* p, int64_t i) { return __bfloat162float(p[i]); }
template <> __device__ __forceinline__ float ldf<double>(const double* p, int64_t i) { return (float)p[i]; }

template <typename TAcc, typename T> __device__ __forceinline__ TAcc ld_as(const T* p, int64_t i);
template <> __device__ __forceinline__ float ld_as<float, float>(const float* p, int64_t i) { return p[i]; }
template <> __device__ __forceinline__ float ld_as<float, bf16>(const bf16* p, int64_t i) { return __bfloat162float(p[i]); }
template <> __device__ __forceinline__ double ld_as<double, float>(const float* p, int64_t i) { return (double)p[i]; }
template <> __device__ __forceinline__ double ld_as<double, bf16>(const bf16* p, int64_t i) { return (double)__bfloat162float(p[i]); }
template <> __device__ __forceinline__ double ld_as<double, double>(const double* p, int64_t i) { return p[i]; }

// ---- unpack 16 bytes of input into floats ----------------------------------------------------------
// bf16: 8 values per uint4; f32: 4 values per uint4.
__device__ __forceinline__ void unpack_bf16x8(const uint4& v, float* f) {
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        f[2 * i] = __uint_as_float(w[i] << 16);
        f[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
}

// ---- FP8 casts (a6): round-to-nearest-even, saturate to +-max finite, NaN -> NaN code --------------
template <int FMT>
__device__ __forceinline__ uint32_t f32x4_to_fp8x4(float a, float b, float c, float d) {
    constexpr __nv_fp8_interpretation_t I = (FMT == 0) ? __NV_E4M3 : __NV_E5M2;
    const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(a, b), __NV_SATFINITE, I);
    const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(c, d), __NV_SATFINITE, I);
    return lo | (hi << 16);
}
// Exact FP8 -> FP32 (every E4M3 / E5M2 value is representable in FP16).
template <int FMT>
__device__ __forceinline__ void fp8x4_to_f32x4(uint32_t w, float* f) {
    constexpr __nv_fp8_interpretation_t I = (FMT == 0) ? __NV_E4M3 : __NV_E5M2;
    const __half2_raw lo = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)(w & 0xFFFFu), I);
    const __half2_raw hi = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)(w >> 16), I);
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&lo));
    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&hi));
    f[0] = a.x; f[1] = a.y; f[2] = b.x; f[3] = b.y;
}

__device__ __forceinline__ uint32_t warp_max_u32(uint32_t v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(0xFFFFFFFFu, v, o));
    return v;
}

// Block-wide max of non-negative-float bit patterns, then ONE atomicMax per CTA (a5).
__device__ __forceinline__ void block_atomic_max_bits(uint32_t loc, uint32_t* dst) {
    __shared__ uint32_t s_warp[32];
    loc = warp_max_u32(loc);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) s_warp[wid] = loc;
    __syncthreads();
    if (wid == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        uint32_t v = lane < nw ? s_warp[lane] : 0u;
        v = warp_max_u32(v);
        if (lane == 0 && v != 0u) atomicMax(dst, v);
    }
}

}  // namespace gf8
