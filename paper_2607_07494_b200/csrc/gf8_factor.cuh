// gf8_factor.cuh -- a1 factor accumulate on the tensor cores (sm_100a):  F <- beta F + alpha X^T X  for BF16 samples X [T][d]
// (Eq. 4; alpha = (1 - beta) / T).  One persistent, warp-specialised kernel runs the jobs of a whole
// gf8_factor_update_many call: only the tiles that touch the UPPER triangle are computed (128 x 256 tiles, one
// tcgen05.mma of N = 256 per K = 16 step, FP32 accumulators double-buffered in TMEM), the lower triangle is written by
// mirroring, and the EMA is folded into the epilogue.  Both MMA operands are MN-major views of X through ONE tensor map per job
// (64 x 64 boxes of K = 64 samples x 64 columns), so X is read as it lies in memory.  BF16 products are exact in FP32: only
// the accumulation order differs from an FP32 reference (gate G6).
// Roles: warp 0 TMA producer, warp 1 MMA issuer (+ TMEM allocation), warps 2-5 epilogue (thread = accumulator row).
#pragma once
#include "gf8_tc.cuh"

namespace gf8 {
namespace fac {

using namespace gf8::tc;

constexpr int F_STAGES = 4;
constexpr int F_STAGE_BYTES = 49152;              // A: 128 columns x 64 samples (16 KB), B: 256 columns x 64 samples (32 KB)
constexpr int F_SMEM = F_STAGES * F_STAGE_BYTES + 1024;
constexpr int F_THREADS = 192;

struct __align__(128) FactorJob {
    CUtensorMap map;          // X [T][d] BF16, boxes of 64 columns x 64 rows, 128 B swizzle
    float* F;                 // d x d FP32, row-major (in / out)
    int32_t d, T;
    float alpha, beta;        // F <- beta F + alpha X^T X   (beta = 0: F is not read)
    int32_t tile0, n_tiles;   // this job's range in the launch's tile list
    int32_t nI, nJ;           // 128-row blocks, 256-column blocks
    int32_t pad[6];
};
static_assert(sizeof(FactorJob) == 256, "job record size");

// tiles of a job, column-block-major: column block j (256 wide) needs the row blocks i (128 high) with 128 i <= 256 j + 255
__host__ __device__ inline int factor_tiles(int nI, int nJ) {
    int n = 0;
    for (int j = 0; j < nJ; ++j) n += min(nI, 2 * j + 2);
    return n;
}

__global__ void __launch_bounds__(F_THREADS, 1) factor_gemm_kernel(const FactorJob* __restrict__ jobs, int n_jobs, int n_tiles, int* err) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t smem0 = smem_u32(smem_raw);
    if (smem0 & 1023u) { if (threadIdx.x == 0) atomicExch(err, 3); return; }
    const uint32_t bars = smem0 + F_STAGES * F_STAGE_BYTES;
    auto full_bar = [&](uint32_t s) { return bars + 8u * s; };
    auto empty_bar = [&](uint32_t s) { return bars + 8u * (F_STAGES + s); };
    auto tfull_bar = [&](uint32_t a) { return bars + 8u * (2 * F_STAGES + a); };
    auto tempty_bar = [&](uint32_t a) { return bars + 8u * (2 * F_STAGES + 2 + a); };
    const uint32_t drain_bar = bars + 8u * (2 * F_STAGES + 4);
    uint32_t* s_tmem = reinterpret_cast<uint32_t*>(smem_raw + F_STAGES * F_STAGE_BYTES + 128);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < F_STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), 4); }
        mbar_init(drain_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tmem)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(s_tmem);

    // tile g of the launch -> (job, row block ti, column block tj); every role walks the same static sequence g = b, b + grid, ...
    auto locate = [&](int g, int& job, int& ti, int& tj) {
        int lo = 0, hi = n_jobs - 1;
        while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (jobs[mid].tile0 <= g) lo = mid; else hi = mid - 1; }
        job = lo;
        int l = g - jobs[lo].tile0;
        const int nI = jobs[lo].nI;
        int j = 0;
        for (;; ++j) { const int c = min(nI, 2 * j + 2); if (l < c) break; l -= c; }
        tj = j; ti = l;
    };

    if (warp == 0) {
        // ===== TMA producer =====
        uint32_t stage = 0, phase = 0;
        bool ok = true;
        const CUtensorMap* last = nullptr;
        for (int g = blockIdx.x; g < n_tiles && ok; g += gridDim.x) {
            int job, ti, tj;
            locate(g, job, ti, tj);
            const CUtensorMap* mp = &jobs[job].map;
            if (mp != last) { if (elect_one()) tmap_acquire(mp); __syncwarp(); last = mp; }
            const int atoms = (jobs[job].T + 63) >> 6;
            for (int t = 0; t < atoms && ok; ++t) {
                if (!(ok = mbar_wait(empty_bar(stage), phase ^ 1u, err))) break;
                const uint32_t sa = smem0 + stage * F_STAGE_BYTES, fb = full_bar(stage);
                if (elect_one()) {
                    mbar_expect_tx(fb, (uint32_t)F_STAGE_BYTES);
#pragma unroll
                    for (int h = 0; h < 2; ++h) tma_load_2d(sa + 8192u * h, mp, 128 * ti + 64 * h, 64 * t, fb);
#pragma unroll
                    for (int h = 0; h < 4; ++h) tma_load_2d(sa + 16384u + 8192u * h, mp, 256 * tj + 64 * h, 64 * t, fb);
                }
                __syncwarp();
                if (++stage == F_STAGES) { stage = 0; phase ^= 1u; }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: D[128][256] += A_t^T-view [128][64] * B_t [256][64]^T, both MN-major =====
        uint32_t stage = 0, phase = 0, n = 0;
        bool ok = true;
        const uint32_t idesc = instr_desc(256, 1, 1);
        for (int g = blockIdx.x; g < n_tiles && ok; g += gridDim.x, ++n) {
            int job, ti, tj;
            locate(g, job, ti, tj);
            const int atoms = (jobs[job].T + 63) >> 6;
            const uint32_t acc = n & 1u;
            if (!(ok = mbar_wait(tempty_bar(acc), ((n >> 1) & 1u) ^ 1u, err))) break;
            tc_fence_after();
            const uint32_t d = tmem_base + acc * 256u;
            for (int t = 0; t < atoms && ok; ++t) {
                if (!(ok = mbar_wait(full_bar(stage), phase, err))) break;
                tc_fence_after();
                const uint32_t sa = smem0 + stage * F_STAGE_BYTES, sb = sa + 16384u;
                if (elect_one()) {
#pragma unroll
                    for (int kk = 0; kk < 4; ++kk)
                        tc_mma_bf16(d, smem_desc(sa + 2048u * kk, 8192u, 1024u), smem_desc(sb + 2048u * kk, 8192u, 1024u), idesc, (t | kk) ? 1u : 0u);
                    tc_commit(empty_bar(stage));
                }
                __syncwarp();
                if (++stage == F_STAGES) { stage = 0; phase ^= 1u; }
            }
            if (ok && elect_one()) tc_commit(tfull_bar(acc));
            __syncwarp();
        }
        if (ok) {
            if (elect_one()) tc_commit(drain_bar);
            __syncwarp();
            mbar_wait(drain_bar, 0u, err);
        }
    } else {
        // ===== epilogue warps 2..5 (TMEM lane quarter = warp & 3): scale, EMA, store the upper part and its mirror image =====
        const int q4 = warp & 3;
        const int r = q4 * 32 + lane;
        uint32_t n = 0;
        bool ok = true;
        for (int g = blockIdx.x; g < n_tiles && ok; g += gridDim.x, ++n) {
            int job, ti, tj;
            locate(g, job, ti, tj);
            const FactorJob& jb = jobs[job];
            const int d = jb.d;
            const float alpha = jb.alpha, beta = jb.beta;
            float* F = jb.F;
            const uint32_t acc = n & 1u;
            if (!(ok = mbar_wait(tfull_bar(acc), (n >> 1) & 1u, err))) break;
            tc_fence_after();
            const int row = 128 * ti + r;
            const uint32_t taddr = tmem_base + acc * 256u + ((uint32_t)(q4 * 32) << 16);
#pragma unroll 1
            for (int c0 = 0; c0 < 256; c0 += 32) {
                uint32_t a[32];
                tmem_ld32_nowait(taddr + (uint32_t)c0, a);
                tmem_wait();
                const int col0 = 256 * tj + c0;
                if (row >= d || col0 >= d || col0 + 31 < row) continue;      // nothing of this chunk lies on or above the diagonal
                float v[32];
#pragma unroll
                for (int e = 0; e < 32; ++e) v[e] = alpha * __uint_as_float(a[e]);
                float* frow = F + (int64_t)row * d + col0;
                if (beta != 0.0f) {
#pragma unroll
                    for (int e = 0; e < 32; e += 4) {
                        if (col0 + e < d) {
                            const float4 o = __ldcg(reinterpret_cast<const float4*>(frow + e));
                            v[e] = fmaf(beta, o.x, v[e]); v[e + 1] = fmaf(beta, o.y, v[e + 1]);
                            v[e + 2] = fmaf(beta, o.z, v[e + 2]); v[e + 3] = fmaf(beta, o.w, v[e + 3]);
                        }
                    }
                }
                // elements left of the diagonal inside this chunk belong to the mirror image of another element: not stored from here
#pragma unroll
                for (int e = 0; e < 32; e += 4) {
                    const int c = col0 + e;
                    if (c >= d) break;
                    if (c >= row) {
                        *reinterpret_cast<float4*>(frow + e) = make_float4(v[e], v[e + 1], v[e + 2], v[e + 3]);
                    } else if (c + 3 >= row) {
#pragma unroll
                        for (int u = 0; u < 4; ++u) if (c + u >= row) frow[e + u] = v[e + u];
                    }
                }
#pragma unroll
                for (int e = 0; e < 32; ++e) {
                    const int c = col0 + e;
                    if (c < d && c > row) F[(int64_t)c * d + row] = v[e];       // mirror: F[c][row] = F[row][c]
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(acc));
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
    }
}

}  // namespace fac
}  // namespace gf8
