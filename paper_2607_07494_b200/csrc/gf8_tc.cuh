// gf8_tc.cuh -- the tensor-core engine of the FAST path (sm_100a): one persistent, warp-specialised
// kernel that runs a list of "items", each a 128 x N BF16 contraction with FP32 accumulation in TMEM
//
//     acc[128][N] = sum over K-atoms t of  A_t[128][64] * B_t[N][64]^T          (tcgen05.mma, kind::f16)
//
// followed by a fused epilogue (add the streamed base tile, column multipliers, amax, FP8 cast ...).
// Every dense contraction of the codec is an instance (PAPER.md:158 Eq. 14, :250 Eq. 22, :172 Eq. 17 in the
// low-rank form of DESIGN.md "Transform"):
//     P' = (Wg U_A) E_A        A = Wg   (K-major),  B = U_A^T        -> BF16 panel
//     Q^T = Wg^T U_G           A = Wg   (MN-major), B = U_G^T        -> FP32 / BF16 panel
//     (S E_A)^T = P'^T U_G     A = P'   (MN-major), B = U_G^T        -> BF16, stored transposed
//     Q'^T = (Q^T + U_A (S E_A)^T) E_G                               -> BF16 panel
//     W~ = Wg + [P' | U_G] [U_A | Q'^T]^T   (rank-2k update)         -> amax / FP8 codes / BF16 / FP32
// Operands are staged by TMA (cp.async.bulk.tensor, 64 x 64 BF16 boxes, 128-byte swizzle) through an
// mbarrier ring of 32 KB stages; one elected thread issues the MMAs; accumulators are double-buffered in
// TMEM so the epilogue of item i overlaps the MMAs of item i+1.  The streamed base tile of the rank-2k
// update (the gradient itself: the HBM-bound traffic) is also fetched by TMA, double-buffered, and the
// FP8 / BF16 output tile leaves through a TMA store, so every HBM access is a full-line bulk transfer.
// Warps 0-7: epilogue (TMEM lane quarter = warp & 3, column half = warp >> 2), warp 8: item fetch + base-tile
// TMA producer, warps 9 / 10: A / B operand TMA producers, warp 11: TMEM allocation + MMA issue.
#pragma once
#include <cuda.h>

#include "gf8_common.cuh"
#include "gf8_quant.cuh"

namespace gf8 {
namespace tc {

constexpr int MAX_STAGES = 7;
constexpr int A_BYTES = 128 * 64 * 2;            // one K-atom of A: 128 x 64 BF16
constexpr int B_BYTES = 128 * 64 * 2;            // one K-atom of B: up to 128 x 64 BF16
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;   // 32 KB
constexpr int TILE_BYTES = 128 * 128 * 2;        // one streamed 128 x 128 BF16 base tile (two 64-column halves)
constexpr int DATA_BYTES = MAX_STAGES * STAGE_BYTES;   // 224 KB, split at launch into ring stages + base tiles
constexpr int MISC_BYTES = 2048;                 // barriers, TMEM address, reductions, parked-tile info, item ring
// 226 KB: the dynamic shared memory is declared 1024-byte aligned (checked at kernel entry), so no alignment slack is
// needed, and 2 KB of the SM's 228 KB stay free: one block of a streaming kernel (1 KB system slice + <= 1 KB of its own)
// fits beside a tensor-core CTA, which is what lets the auxiliary stream's kernels overlap the stages.
constexpr int SMEM_BYTES = DATA_BYTES + MISC_BYTES;
constexpr int EPI_WARPS = 8, PRODUCER_WARP = 8, OPERAND_WARP = 9, MMA_WARP = 11, SYNC_WARP = 12;
constexpr int THREADS = 32 * (EPI_WARPS + 5);
constexpr int ITEM_SLOTS = 4;                    // shared-memory ring of item descriptors
constexpr int MAX_BASE_SLOTS = 4;                // streamed base tiles in flight (ring, decoupled from TMEM)
constexpr int TMEM_COLS = 512;                   // four 128-column accumulator slots
constexpr int FUSE_LAG = 2;                      // fused update: tiles parked in TMEM while the tensor amax completes
                                                 // (2 parked + 1 in the epilogue + 1 under the MMAs = 4 slots)
constexpr int CODE_TILE_BYTES = 128 * 128;       // staging of one 128 x 128 FP8 code tile
constexpr int STRIP_L_BYTES = 4 * A_BYTES;       // strip mode: resident A tiles, [row block 0/1][K-atom 0/1]
constexpr int STRIP_RING = 2;                    // strip mode: ring of column-tile stages, each the (up to two) 16 KB B K-atoms of a column tile
constexpr int NSEG = 6;                          // operand segments per item (hi/lo split products)

enum Epi : int32_t {
    EPI_STORE = 0,       // out = (base + acc) * colscale           (BF16 or FP32)
    EPI_STORE_T = 1,     // out[c][r] = acc * colscale  (BF16, transposed store; the small S matrix)
    EPI_AMAX = 2,        // atomicMax(amax, max |base + acc|)        (a5, per-tensor scale)
    EPI_CAST = 3,        // codes = fp8((base + acc) * scale(amax))  (a6)
    EPI_BLOCKCAST = 4,   // per-128x128-block amax + scale + cast in one pass (a5 + a6)
    EPI_END = -1         // written into the item ring by the fetch warp: no more items for this CTA
};
enum Ty : int32_t { TY_NONE = 0, TY_BF16 = 1, TY_F32 = 2 };

struct __align__(16) Item {
    int32_t map_a[NSEG], map_b[NSEG];   // tensor-map indices (into the plan's CUtensorMap array) per segment
    int32_t atoms[NSEG];                // K-atoms (64 wide) per segment; 0 = unused
    int32_t a_c0[NSEG], a_r0[NSEG];     // first box of A: (col, row) in its matrix
    int32_t b_c0[NSEG], b_r0[NSEG];     // first box of B
    int32_t a_mn;                 // 1: A is MN-major (the 128 "M" elements are contiguous in memory)
    int32_t N;                    // accumulator columns: multiple of 64, <= 128
    int32_t mode, fmt;
    int32_t row0, col0, rows, cols;   // output tile origin and valid extent (rows <= 128, cols <= N)
    int32_t base_type, out_type;
    int32_t write_scale, out_map; // out_map >= 0: the output tile leaves through a TMA store from shared memory
    int32_t base_map[2];          // >= 0: the base tile (hi [+ lo]) is streamed by TMA into shared memory
    int32_t b_mn;                 // 1: B is MN-major too (the factor GEMM X^T X reads both operands from X)
    int32_t strip;                // 1: strip item of the update (up to 256 rows x all columns; see tc_items_kernel)
    int32_t tri;                  // 1: segments 0..2 are the split products hi*hi, lo*hi, hi*lo of one operand pair: in a kmode 5
    int32_t sync;                 //    launch every K-atom brings A_hi, A_lo, B_hi, B_lo in once and feeds all three
                                  // sync (pair launches, kmode 6): 1 = amax item, counts itself done in *(uint32_t*)base once per
                                  // epilogue warp; 2 = cast item, starts when that counter has reached base_ld
    int64_t base_ld, out_ld;
    const void* base;
    void* out;
    void* out_lo;                 // EPI_STORE / EPI_STORE_T with BF16 output: optional residual v - bf16(v) (split operands)
    const float* colscale;        // indexed by tile column c (already offset), or null
    uint32_t* amax;               // EPI_AMAX: target; EPI_CAST: source
    float* scale_inv_out;         // EPI_CAST (write_scale) / EPI_BLOCKCAST: where scale_inv goes
};

// What the fused update keeps about a tile parked in TMEM until its tensor's amax is complete.
struct Parked {
    int32_t out_map, col0, row0, fmt, write_scale, total;
    uint32_t* amax;
    float* scale_inv_out;
    uint32_t* done;
};

constexpr int ITEM_BYTES = (int)sizeof(Item);
static_assert(ITEM_BYTES % 16 == 0 && 656 + ITEM_SLOTS * ITEM_BYTES <= MISC_BYTES, "item ring must fit its shared-memory slice");

// ---- PTX wrappers ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(bar), "r"(bytes)
                 : "memory");
}
// Bounded spin: a broken pipeline sets *err and lets the kernel drain instead of hanging the GPU.
__device__ __forceinline__ bool mbar_wait(uint32_t bar, uint32_t parity, int* err) {
    uint32_t done = 0;
    for (uint32_t spin = 0; spin < (1u << 26); ++spin) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        if (done) return true;
        if ((spin & 0xFFFF) == 0xFFFF && *(volatile int*)err) return false;
    }
    atomicExch(err, 1);
    return false;
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c, int r, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c), "r"(r) : "memory");
}
// One lane of a converged warp (the role loops stay warp-uniform, so their operands live in uniform registers
// and the TMA / MMA issues need no per-thread waterfall).
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tmap_acquire(const CUtensorMap* map) {
    asm volatile("fence.proxy.tensormap::generic.acquire.gpu [%0], 128;" ::"l"(map) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_mma_bf16(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                            uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// 32 columns of this thread's TMEM lane; the caller waits (tmem_wait) before using v.
__device__ __forceinline__ void tmem_ld32_nowait(uint32_t taddr, uint32_t* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
        "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
        ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
          "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]),
          "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]), "r"(v[20]), "r"(v[21]), "r"(v[22]), "r"(v[23]),
          "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]), "r"(v[31])
        : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor (SWIZZLE_128B, version 1).  lbo / sbo in bytes.
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((addr >> 4) & 0x3FFFu) | ((uint64_t)((lbo >> 4) & 0x3FFFu) << 16) |
           ((uint64_t)((sbo >> 4) & 0x3FFFu) << 32) | (1ull << 46) | (2ull << 61);
}
// Instruction descriptor: D = F32, A = B = BF16, M = 128, N, A / B major-ness (0 = K-major, 1 = MN-major).
__device__ __forceinline__ uint32_t instr_desc(int N, int a_mn, int b_mn) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_mn << 15) | ((uint32_t)b_mn << 16) | ((uint32_t)(N >> 3) << 17) |
           ((128u >> 4) << 24);
}

// ---- epilogue helpers ---------------------------------------------------------------------------------
// Eight epilogue warps: warp w reads TMEM lanes 32 (w & 3) .. +31 (one accumulator row per thread) and the
// column half (w >> 2) of the tile, so every SM sub-partition holds two epilogue warps.
// 16 consecutive elements of the base tile row as floats (zero when there is no base).
__device__ __forceinline__ void load_base16(const Item& it, int64_t off, float* b) {
    if (it.base_type == TY_BF16) {
        const uint4* p = reinterpret_cast<const uint4*>(reinterpret_cast<const bf16*>(it.base) + off);
        const uint4 x = __ldg(p), y = __ldg(p + 1);
        unpack_bf16x8(x, b);
        unpack_bf16x8(y, b + 8);
    } else if (it.base_type == TY_F32) {
        const float4* p = reinterpret_cast<const float4*>(reinterpret_cast<const float*>(it.base) + off);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float4 x = __ldg(p + u);
            b[4 * u] = x.x; b[4 * u + 1] = x.y; b[4 * u + 2] = x.z; b[4 * u + 3] = x.w;
        }
    } else {
#pragma unroll
        for (int u = 0; u < 16; ++u) b[u] = 0.0f;
    }
}

// (v0, v1) * s with one packed multiply (FMUL2); the same IEEE products as two FMULs
__device__ __forceinline__ void mul2(float v0, float v1, float s, float& x0, float& x1) {
    uint64_t a, ss;
    asm("mov.b64 %0, {%1, %1};" : "=l"(ss) : "f"(s));
    asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(v0), "f"(v1));
    asm("mul.rn.f32x2 %0, %0, %1;" : "+l"(a) : "l"(ss));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x0), "=f"(x1) : "l"(a));
}
template <int FMT>
__device__ __forceinline__ uint4 codes16(const float* v, float s) {
    float x[16];
#pragma unroll
    for (int u = 0; u < 16; u += 2) mul2(v[u], v[u + 1], s, x[u], x[u + 1]);
    uint4 q;
    q.x = f32x4_to_fp8x4<FMT>(x[0], x[1], x[2], x[3]);
    q.y = f32x4_to_fp8x4<FMT>(x[4], x[5], x[6], x[7]);
    q.z = f32x4_to_fp8x4<FMT>(x[8], x[9], x[10], x[11]);
    q.w = f32x4_to_fp8x4<FMT>(x[12], x[13], x[14], x[15]);
    return q;
}
template <int FMT>
__device__ __forceinline__ uint4 codes16_scalar(const float* v, float s) {
    uint4 o;
    o.x = f32x4_to_fp8x4<FMT>(__fmul_rn(v[0], s), __fmul_rn(v[1], s), __fmul_rn(v[2], s), __fmul_rn(v[3], s));
    o.y = f32x4_to_fp8x4<FMT>(__fmul_rn(v[4], s), __fmul_rn(v[5], s), __fmul_rn(v[6], s), __fmul_rn(v[7], s));
    o.z = f32x4_to_fp8x4<FMT>(__fmul_rn(v[8], s), __fmul_rn(v[9], s), __fmul_rn(v[10], s), __fmul_rn(v[11], s));
    o.w = f32x4_to_fp8x4<FMT>(__fmul_rn(v[12], s), __fmul_rn(v[13], s), __fmul_rn(v[14], s), __fmul_rn(v[15], s));
    return o;
}

__device__ __forceinline__ void epi_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }

__device__ __forceinline__ uint32_t epi_block_max(uint32_t loc, int warp, int lane, uint32_t* s_red) {
    loc = warp_max_u32(loc);
    if (lane == 0) s_red[warp] = loc;
    epi_sync();
    uint32_t bits = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) bits = max(bits, s_red[w]);
    epi_sync();
    return bits;
}

// One accumulator tile -> global memory with the base (if any) read straight from global memory: the small
// panels (P', Q^T, S, Q'^T) and FP32 gradients.  Thread = one row, 16 columns per tcgen05.ld.
__device__ __forceinline__ void epilogue(const Item& it, uint32_t tmem_acc, int warp, int lane, uint32_t* s_red, int rblk = 0, int dbgx = 0) {
    // rblk = 1: the second row block of a 256-row panel item (rows 128.., accumulator 64 columns further on)
    const int r = rblk * 128 + (warp & 3) * 32 + lane, half = warp >> 2;
    const bool row_ok = r < it.rows;
    const int64_t grow = it.row0 + r;
    const uint32_t taddr = tmem_acc + ((uint32_t)((warp & 3) * 32) << 16) + 64u * (uint32_t)rblk;
    const int nch = it.cols >> 4;
    const int cb = half ? ((nch + 1) >> 1) << 4 : 0, ce = half ? nch << 4 : ((nch + 1) >> 1) << 4;
    uint32_t a[16];
    float v[16];
    float scale = 1.0f;
    if (it.mode == EPI_BLOCKCAST) {
        uint32_t loc = 0;
        for (int c0 = cb; c0 < ce; c0 += 16) {
            tmem_ld16(taddr + c0, a);
            if (row_ok) {
                load_base16(it, grow * it.base_ld + it.col0 + c0, v);
#pragma unroll
                for (int u = 0; u < 16; ++u) loc = max(loc, __float_as_uint(v[u] + __uint_as_float(a[u])) & 0x7FFFFFFFu);
            }
        }
        const uint32_t bits = epi_block_max(loc, warp, lane, s_red);
        float si;
        scales_from_amax(bits, it.fmt == 0 ? 448.0f : 57344.0f, scale, si);
        if (r == 0 && half == 0) *it.scale_inv_out = si;
    } else if (it.mode == EPI_CAST) {
        float si;
        scales_from_amax(*reinterpret_cast<volatile uint32_t*>(it.amax), it.fmt == 0 ? 448.0f : 57344.0f, scale, si);
        if (it.write_scale && r == 0 && half == 0) *it.scale_inv_out = si;
    }
    uint32_t loc = 0;
    for (int c0 = cb; c0 < ce; c0 += 16) {
        tmem_ld16(taddr + c0, a);                 // warp-collective: every lane executes it
        if (!row_ok) continue;
        if (it.mode == EPI_STORE_T) {
            bf16* o = reinterpret_cast<bf16*>(it.out);
#pragma unroll
            for (int u = 0; u < 16; ++u) {
                const float cs = it.colscale ? __ldg(it.colscale + c0 + u) : 1.0f;
                const float x = __uint_as_float(a[u]) * cs;
                const bf16 hi = __float2bfloat16_rn(x);
                o[(int64_t)(it.col0 + c0 + u) * it.out_ld + grow] = hi;
                if (it.out_lo)
                    reinterpret_cast<bf16*>(it.out_lo)[(int64_t)(it.col0 + c0 + u) * it.out_ld + grow] =
                        __float2bfloat16_rn(x - __bfloat162float(hi));
            }
            continue;
        }
        if (dbgx & 4096) {
#pragma unroll
            for (int u = 0; u < 16; ++u) v[u] = 0.0f;
        } else load_base16(it, grow * it.base_ld + it.col0 + c0, v);
#pragma unroll
        for (int u = 0; u < 16; ++u) v[u] += __uint_as_float(a[u]);
        if (it.mode == EPI_AMAX) {
#pragma unroll
            for (int u = 0; u < 16; ++u) loc = max(loc, __float_as_uint(v[u]) & 0x7FFFFFFFu);
        } else if (it.mode == EPI_CAST || it.mode == EPI_BLOCKCAST) {
            uint8_t* p = reinterpret_cast<uint8_t*>(it.out) + grow * it.out_ld + it.col0 + c0;
            *reinterpret_cast<uint4*>(p) = it.fmt == 0 ? codes16<0>(v, scale) : codes16<1>(v, scale);
        } else {   // EPI_STORE
            if (it.colscale && !(dbgx & 8192)) {
#pragma unroll
                for (int u = 0; u < 16; ++u) v[u] *= __ldg(it.colscale + c0 + u);
            }
            const int64_t off = grow * it.out_ld + it.col0 + c0;
            if ((dbgx & 16384) && v[0] != 12345.0f) continue;
            if (it.out_type == TY_F32) {
                float4* o = reinterpret_cast<float4*>(reinterpret_cast<float*>(it.out) + off);
#pragma unroll
                for (int u = 0; u < 4; ++u) o[u] = make_float4(v[4 * u], v[4 * u + 1], v[4 * u + 2], v[4 * u + 3]);
            } else {
                uint32_t w[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const __nv_bfloat162 h = __floats2bfloat162_rn(v[2 * u], v[2 * u + 1]);
                    w[u] = *reinterpret_cast<const uint32_t*>(&h);
                }
                uint4* o = reinterpret_cast<uint4*>(reinterpret_cast<bf16*>(it.out) + off);
                o[0] = make_uint4(w[0], w[1], w[2], w[3]);
                o[1] = make_uint4(w[4], w[5], w[6], w[7]);
                if (it.out_lo) {
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const float2 hi = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&w[u]));
                        const __nv_bfloat162 h = __floats2bfloat162_rn(v[2 * u] - hi.x, v[2 * u + 1] - hi.y);
                        w[u] = *reinterpret_cast<const uint32_t*>(&h);
                    }
                    uint4* o2 = reinterpret_cast<uint4*>(reinterpret_cast<bf16*>(it.out_lo) + off);
                    o2[0] = make_uint4(w[0], w[1], w[2], w[3]);
                    o2[1] = make_uint4(w[4], w[5], w[6], w[7]);
                }
            }
        }
    }
    if (it.mode == EPI_AMAX) {
        loc = warp_max_u32(loc);
        if (lane == 0 && loc != 0u) atomicMax(it.amax, loc);
    }
}

// ---- tile epilogue: base tile(s) in shared memory (TMA, 128 B swizzle), output through a TMA store ------------
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, uint32_t src, int c, int r) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];"
                 ::"l"(map), "r"(src), "r"(c), "r"(r) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, const uint4& v) {
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// v[16] = base(hi [+ lo]) columns [c0, c0+16) of row r of the staged tile + accumulator.
// Tile layout: half h (64 columns) at h * 16 KB, row r at r * 128 B, 16-byte chunk q at (q ^ (r & 7)) * 16.
__device__ __forceinline__ void tile_values16(uint32_t tile, int n_base, int r, int c0, const uint32_t* a, float* v) {
    const uint32_t row = tile + (uint32_t)(c0 >> 6) * 16384u + (uint32_t)r * 128u;
    const uint32_t q = (uint32_t)(c0 & 63) >> 3;
    const uint4 x = lds128(row + (((q) ^ (uint32_t)(r & 7)) << 4));
    const uint4 y = lds128(row + (((q + 1) ^ (uint32_t)(r & 7)) << 4));
    unpack_bf16x8(x, v);
    unpack_bf16x8(y, v + 8);
    if (n_base > 1) {
        float w[16];
        const uint4 x2 = lds128(row + TILE_BYTES + (((q) ^ (uint32_t)(r & 7)) << 4));
        const uint4 y2 = lds128(row + TILE_BYTES + (((q + 1) ^ (uint32_t)(r & 7)) << 4));
        unpack_bf16x8(x2, w);
        unpack_bf16x8(y2, w + 8);
#pragma unroll
        for (int u = 0; u < 16; ++u) v[u] += w[u];
    }
#pragma unroll
    for (int u = 0; u < 16; ++u) v[u] += __uint_as_float(a[u]);
}

// v[32] = base(hi [+ lo]) + accumulator for columns [32 g, 32 g + 32) of this warp's 64-column half: the TMEM
// load and the shared-memory loads are all issued before the single wait.  `row` = this row's 128 B of the half.
__device__ __forceinline__ void tile_values32(uint32_t taddr, uint32_t row, int n_base, int r, int g, float* v) {
    uint32_t a[32];
    tmem_ld32_nowait(taddr + 32u * g, a);
    uint4 b[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) b[j] = lds128(row + (((uint32_t)(4 * g + j) ^ (uint32_t)(r & 7)) << 4));
    if (n_base == 1) {
        // one BF16 base: v = float(base) + acc in ONE instruction per element (FHADD.BF16: exact widening, one FP32 rounding --
        // bit-identical to unpack-then-add, at a third of the instructions)
        tmem_wait();
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t w[4] = {b[j].x, b[j].y, b[j].z, b[j].w};
#pragma unroll
            for (int e = 0; e < 4; ++e)
                asm("{\n\t.reg .b16 lo, hi;\n\tmov.b32 {lo, hi}, %2;\n\tadd.rn.f32.bf16 %0, lo, %3;\n\tadd.rn.f32.bf16 %1, hi, %4;\n\t}"
                    : "=f"(v[8 * j + 2 * e]), "=f"(v[8 * j + 2 * e + 1])
                    : "r"(w[e]), "f"(__uint_as_float(a[8 * j + 2 * e])), "f"(__uint_as_float(a[8 * j + 2 * e + 1])));
        }
        return;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) unpack_bf16x8(b[j], v + 8 * j);
    if (n_base > 1) {
#pragma unroll
        for (int j = 0; j < 4; ++j) b[j] = lds128(row + TILE_BYTES + (((uint32_t)(4 * g + j) ^ (uint32_t)(r & 7)) << 4));
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            float w[8];
            unpack_bf16x8(b[j], w);
#pragma unroll
            for (int u = 0; u < 8; ++u) v[8 * j + u] += w[u];
        }
    }
    tmem_wait();
#pragma unroll
    for (int u = 0; u < 32; ++u) v[u] += __uint_as_float(a[u]);
}

// Returns true if a TMA store was issued from `tile` (the caller waits for its smem reads before reuse).
// All eight warps share the tile: warp w covers rows 32 (w & 3) .. +31 of the 64-column half w >> 2.
// ---- error feedback (f1; Alg. 1 l.11-15) fused into the update epilogue --------------------------------------
// An EPI_AMAX / EPI_CAST / EPI_BLOCKCAST item whose out_lo is non-null carries the tensor's FP32 residual R there: the epilogue
// quantizes U~ = W~ + R and, in the cast, writes R <- U~ - val(code) * scale_inv.  One FP32 rounding per operation, like oracle
// O8.  R lives in the EPILOGUE'S OWN LAYOUT ("tiled", EF_TILE floats per 128 x 128 tile, tiles row-major over the padded
// tensor): element (r, 64 h + 32 g + 4 q + e) of a tile sits at (((2 h + g) 8 + q) 128 + r) 4 + e, so that the 32 lanes of a
// warp -- 32 consecutive rows -- read one contiguous 512 B per load instruction.  (With a row-major R every lane touches its
// own 128 B line: the load/store unit then serialises 32 lines per instruction and the two update passes take 15 + 30 ms
// instead of 2 + 3.3, measured.)  gf8_resid_export converts to row-major.
// `valid` = columns of this 32-column group inside the tensor (multiple of 4).
constexpr int EF_TILE = 128 * 128;
__device__ __forceinline__ void ef_add32(const float* __restrict__ grp /* tile + ((2h+g) 8 * 128 + r) * 4 */, int valid, float* v) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        if (4 * q < valid) {
            const float4 t = __ldcg(reinterpret_cast<const float4*>(grp + q * 512));
            v[4 * q] = __fadd_rn(v[4 * q], t.x); v[4 * q + 1] = __fadd_rn(v[4 * q + 1], t.y);
            v[4 * q + 2] = __fadd_rn(v[4 * q + 2], t.z); v[4 * q + 3] = __fadd_rn(v[4 * q + 3], t.w);
        }
    }
}
template <int FMT>
__device__ __forceinline__ void ef_store32(float* __restrict__ grp, int valid, const float* ut, const uint4& c0, const uint4& c1, float si) {
    const uint32_t w[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        if (4 * q < valid) {
            float val[4];
            fp8x4_to_f32x4<FMT>(w[q], val);
            float4 o;
            o.x = __fsub_rn(ut[4 * q], __fmul_rn(val[0], si)); o.y = __fsub_rn(ut[4 * q + 1], __fmul_rn(val[1], si));
            o.z = __fsub_rn(ut[4 * q + 2], __fmul_rn(val[2], si)); o.w = __fsub_rn(ut[4 * q + 3], __fmul_rn(val[3], si));
            __stcg(reinterpret_cast<float4*>(grp + q * 512), o);
        }
    }
}

template <bool EF>
__device__ __forceinline__ bool epilogue_tile(const Item& it, uint32_t tmem_acc, uint32_t tile, int n_base, int warp,
                                              int lane, uint32_t* s_red, const CUtensorMap* maps, float cast_scale, float cast_si,
                                              int row0, int col0, bool write_scale, float* sinv_out, uint32_t* run_max) {
    // (row0, col0) = the tile's origin: the item's own for tile items, a tile of the strip for strip items;
    // run_max != null: EPI_AMAX accumulates into the caller's per-thread running maximum (one atomic per strip)
    const int r = (warp & 3) * 32 + lane;
    const int h0 = warp >> 2, h1 = h0 + 1;
    const uint32_t taddr0 = tmem_acc + ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t row_lo = tile + (uint32_t)r * 128u;
    const bool lead = r == 0 && h0 == 0;
    const int mode = it.mode, fmt = it.fmt;
    float v[32];
    float scale = 1.0f, si_cast = cast_si;
    // error feedback: the tensor's residual row segment under this tile (null: plain codec)
    float* resid = (EF && (mode == EPI_AMAX || mode == EPI_CAST || mode == EPI_BLOCKCAST)) ? reinterpret_cast<float*>(it.out_lo) : nullptr;
    const bool ef_row_ok = row0 + r < it.row0 + it.rows;
    // (this thread's first group in the tile: h = 0, g = 0, q = 0)
    float* resid_row = resid ? resid + ((int64_t)(row0 >> 7) * ((it.out_ld + 127) >> 7) + (col0 >> 7)) * EF_TILE + r * 4 : nullptr;
    const int ef_cols = it.col0 + it.cols - col0;            // columns of the tensor from this tile's origin on
    if (mode == EPI_BLOCKCAST || mode == EPI_AMAX) {
        uint32_t loc = 0;
        for (int h = h0; h < h1; ++h)
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                tile_values32(taddr0 + 64u * h, row_lo + 16384u * h, n_base, r, g, v);
                if (resid && ef_row_ok) ef_add32(resid_row + (2 * h + g) * 4096, ef_cols - 64 * h - 32 * g, v);
                // max |v| two elements per instruction (FMNMX3, NaN-propagating: a NaN amax orders above every finite value
                // as an integer, like the bit-pattern maximum it replaces)
                float mx = __uint_as_float(loc);
#pragma unroll
                for (int u = 0; u < 32; u += 2)
                    asm("max.NaN.f32 %0, %1, %2, %0;" : "+f"(mx) : "f"(fabsf(v[u])), "f"(fabsf(v[u + 1])));
                loc = __float_as_uint(mx);
            }
        if (mode == EPI_AMAX) {
            if (run_max) { *run_max = max(*run_max, loc); return false; }
            loc = warp_max_u32(loc);
            if (lane == 0 && loc != 0u) atomicMax(it.amax, loc);
            return false;
        }
        const uint32_t bits = epi_block_max(loc, warp, lane, s_red);
        float si;
        scales_from_amax(bits, fmt == 0 ? 448.0f : 57344.0f, scale, si);
        si_cast = si;
        if (lead) *sinv_out = si;
    } else if (mode == EPI_CAST) {
        scale = cast_scale;                       // (from the tensor's amax, once per item by the caller)
        if (write_scale && lead) *sinv_out = cast_si;
    }
    if (mode == EPI_CAST || mode == EPI_BLOCKCAST) {
        // 64 codes per row half and thread.  Written straight from registers, a warp's store instruction would touch 32 different
        // 128 B lines with 16 bytes each, and L1TEX takes them one line per cycle: 1024 cycles per tile, more than the rest of
        // the cast epilogue (measured: 1757 cycles per tile against 685 for the amax epilogue).  So the warp transposes its
        // 32 x 64 B through the 4 KB of the base tile that only it reads (its 32 rows of this column half, dead once the values
        // are in registers): afterwards four lanes hold the 64 contiguous bytes of a row and an instruction touches 8 lines.
        // No CTA-level barrier and no proxy fence are involved, so the base slot still goes back to the producer at once.
        const int q4 = warp & 3, l_row = lane >> 2, l_chk = lane & 3;
        for (int h = h0; h < h1; ++h) {
            uint4 cd[4];
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                tile_values32(taddr0 + 64u * h, row_lo + 16384u * h, n_base, r, g, v);
                if (resid && ef_row_ok) ef_add32(resid_row + (2 * h + g) * 4096, ef_cols - 64 * h - 32 * g, v);
                cd[2 * g] = fmt == 0 ? codes16<0>(v, scale) : codes16<1>(v, scale);
                cd[2 * g + 1] = fmt == 0 ? codes16<0>(v + 16, scale) : codes16<1>(v + 16, scale);
                if (resid && ef_row_ok) {
                    if (fmt == 0) ef_store32<0>(resid_row + (2 * h + g) * 4096, ef_cols - 64 * h - 32 * g, v, cd[2 * g], cd[2 * g + 1], si_cast);
                    else ef_store32<1>(resid_row + (2 * h + g) * 4096, ef_cols - 64 * h - 32 * g, v, cd[2 * g], cd[2 * g + 1], si_cast);
                }
            }
            // staging: row l of the warp keeps its chunk q at 16-byte slot 4 l + (q ^ ((l >> 1) & 3)) (4 wavefronts per
            // instruction both ways: the minimum for 512 bytes)
            const uint32_t stg = tile + 16384u * (uint32_t)h + 4096u * (uint32_t)q4;
            __syncwarp();                                     // (every lane has read its base values)
#pragma unroll
            for (int q = 0; q < 4; ++q) sts128(stg + (uint32_t)(4 * lane + (q ^ ((lane >> 1) & 3))) * 16u, cd[q]);
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int lr = 8 * j + l_row;                 // row of the warp this lane stores a piece of
                const uint4 piece = lds128(stg + (uint32_t)(4 * lr + (l_chk ^ ((lr >> 1) & 3))) * 16u);
                const int grow = row0 + 32 * q4 + lr, gcol = col0 + 64 * h + 16 * l_chk;
                if (grow < it.row0 + it.rows && gcol < it.col0 + it.cols)
                    *reinterpret_cast<uint4*>(reinterpret_cast<uint8_t*>(it.out) + (int64_t)grow * it.out_ld + gcol) = piece;
            }
            __syncwarp();                                     // (the staging area is read before the next half overwrites... its own)
        }
        return false;
    }
    // EPI_STORE: BF16 output in place of the hi tile (same layout) and out through a TMA
    // store, or FP32 output straight to global memory
    const int half = h0, cbase = half * 64;
    const uint32_t taddr = taddr0 + (uint32_t)cbase, row = row_lo + 16384u * half;
    if (it.out_type == TY_BF16) {
#pragma unroll
        for (int g = 0; g < 2; ++g) {
            tile_values32(taddr, row, n_base, r, g, v);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                uint32_t w[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const __nv_bfloat162 h = __floats2bfloat162_rn(v[8 * j + 2 * u], v[8 * j + 2 * u + 1]);
                    w[u] = *reinterpret_cast<const uint32_t*>(&h);
                }
                sts128(row + (((uint32_t)(4 * g + j) ^ (uint32_t)(r & 7)) << 4), make_uint4(w[0], w[1], w[2], w[3]));
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        epi_sync();
        if (threadIdx.x == 0) {
#pragma unroll
            for (int h = 0; h < 2; ++h) tma_store_2d(maps + it.out_map, tile + h * 16384u, col0 + 64 * h, row0);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        return true;
    }
    const bool row_ok = r < it.rows;
#pragma unroll
    for (int g = 0; g < 2; ++g) {
        tile_values32(taddr, row, n_base, r, g, v);
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const int c0 = cbase + 32 * g + 16 * q;
            if (!row_ok || c0 >= it.cols) continue;
            float4* o = reinterpret_cast<float4*>(reinterpret_cast<float*>(it.out) + (int64_t)(row0 + r) * it.out_ld + col0 + c0);
#pragma unroll
            for (int u = 0; u < 4; ++u)
                o[u] = make_float4(v[16 * q + 4 * u], v[16 * q + 4 * u + 1], v[16 * q + 4 * u + 2], v[16 * q + 4 * u + 3]);
        }
    }
    return false;
}

// ---- the kernel ------------------------------------------------------------------------------------------
// Persistent: CTA b runs items b, b + gridDim.x, ...  The 224 KB of data shared memory is split at launch into
// `n_stages` operand ring stages (32 KB) and 2 x `n_base` streamed base tiles (32 KB; double-buffered like the
// TMEM accumulators).  The producer warp copies each item descriptor into a 4-slot shared-memory ring one item
// ahead, so no role waits on a global load.  `err` is set (and the kernel drains) if a barrier wait times out,
// so a pipeline bug cannot hang the GPU.
// EF: the error-feedback epilogue (f1) is compiled into its own instance, so the default kernel keeps its registers.
template <bool EF>
__global__ void __launch_bounds__(THREADS, 1) tc_items_kernel(const Item* __restrict__ items, int n_items,
                                                              const CUtensorMap* __restrict__ maps, int* err,
                                                              int n_stages, int n_base, int n_bslots, int kmode, int dbg_in,
                                                              long long* __restrict__ prof_in, int* ctr) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
#ifndef GF8_DEBUG
    // (release builds: the ablation bits of `dbg_in` and the per-role wait profile are compiled out)
    constexpr int dbg = 0;
    constexpr long long* prof = nullptr;
    (void)dbg_in; (void)prof_in;
#else
    const int dbg = dbg_in;
    long long* const prof = prof_in;
#endif
    const int fuse = kmode == 1 ? 1 : 0;           // kmode: 0 = tile items, 1 = fused update (TMEM-parked), 2 = strip items
    // kmode 6 = strip items in PAIRS (amax item, cast item of the same sub-strip, adjacent in the list): a CTA claims a pair, so
    // the cast pass re-reads its gradient tiles right after the amax pass has brought them in (L2), one launch for both passes
    // (bits 8.. of kmode: claim granularity.  A CTA takes `chunk` consecutive items per claim, so that tile items -- whose ten
    //  tensor maps change with the tensor -- come in runs of the same tensor: every new map costs its TMA instruction a
    //  descriptor fetch, and a CTA that gets one or two tiles per tensor pays that on every item)
    const int chunk = (kmode >> 8) > 0 ? (kmode >> 8) : 1;
    kmode &= 0xFF;
    const bool pair = kmode == 6;
    const bool strip = kmode == 2 || pair;
    // ctr != null: items are handed out dynamically (atomic counter, list order = start order), so item durations may
    // differ without idling CTAs and the planner's ordering decides which items run at the same time (L2 reuse).
    // The fused update keeps the static round-robin (its cast of parked tiles counts on it).
    const bool dyn = ctr != nullptr && !fuse;
    const uint32_t smem0 = smem_u32(smem_raw);                              // 1024-byte aligned (swizzle atoms)
    if (smem0 & 1023u) {                                                    // (never seen; fail loudly rather than corrupt tiles)
        if (threadIdx.x == 0) atomicExch(err, 3);
        return;
    }
    // kmode 3 = tile items with wide operand stages: [A rows 0-127 | A rows 128-255 | B (N <= 64)] = 40 KB, for panel
    // items of up to 256 rows (two accumulators of 64 columns in one TMEM slot share every B atom)
    // (kmode 4: the same with a 16 KB B area, 48 KB stages, when the launch also holds N = 128 items)
    // (kmode 5: wide stages for interleaved split products: [A_hi 32 KB | A_lo 32 KB | B_hi 8 KB | B_lo 8 KB] = 80 KB)
    const bool tri = kmode == 5;
    const bool wide = kmode == 3 || kmode == 4 || tri;
    const uint32_t stage_bytes = kmode == 3 ? 40960u : (kmode == 4 ? 49152u : (tri ? 81920u : (uint32_t)STAGE_BYTES));
    const uint32_t b_off = tri ? 65536u : (wide ? 32768u : (uint32_t)A_BYTES);
    const uint32_t base0 = smem0 + (uint32_t)n_stages * stage_bytes;        // base tiles: [acc][n_base] x 32 KB
    const uint32_t bars = smem0 + DATA_BYTES;
    uint8_t* gen0 = smem_raw + (smem0 - smem_u32(smem_raw));
    uint32_t* s_tmem = reinterpret_cast<uint32_t*>(gen0 + DATA_BYTES + 384);
    uint32_t* s_red = s_tmem + 4;
    Parked* s_park = reinterpret_cast<Parked*>(gen0 + DATA_BYTES + 464);
    uint8_t* s_items = gen0 + DATA_BYTES + 656;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    auto full_bar = [&](int s) { return bars + 8u * s; };
    auto empty_bar = [&](int s) { return bars + 8u * (MAX_STAGES + s); };
    auto tfull_bar = [&](int a) { return bars + 8u * (2 * MAX_STAGES + a); };
    auto tempty_bar = [&](int a) { return bars + 8u * (2 * MAX_STAGES + 4 + a); };
    auto bfull_bar = [&](int a) { return bars + 8u * (2 * MAX_STAGES + 8 + a); };
    auto bempty_bar = [&](int a) { return bars + 8u * (2 * MAX_STAGES + 8 + MAX_BASE_SLOTS + a); };
    auto ifull_bar = [&](int s) { return bars + 8u * (2 * MAX_STAGES + 8 + 2 * MAX_BASE_SLOTS + s); };
    auto iempty_bar = [&](int s) { return bars + 8u * (2 * MAX_STAGES + 8 + 2 * MAX_BASE_SLOTS + ITEM_SLOTS + s); };
    auto parked_bar = [&](int a) { return bars + 8u * (2 * MAX_STAGES + 8 + 2 * MAX_BASE_SLOTS + 2 * ITEM_SLOTS + a); };
    auto sready_bar = [&](int a) { return bars + 8u * (2 * MAX_STAGES + 8 + 2 * MAX_BASE_SLOTS + 2 * ITEM_SLOTS + 4 + a); };
    auto drain_bar = [&](int a) { return bars + 8u * (2 * MAX_STAGES + 8 + 2 * MAX_BASE_SLOTS + 2 * ITEM_SLOTS + 8 + a); };
    float* s_scale = reinterpret_cast<float*>(s_red + 8);     // fused update: scale of each parked tile's tensor
    const uint32_t n_acc = 4u;                       // TMEM accumulator slots in rotation (4 x 128 columns)
    auto base_tile = [&](uint32_t b) { return base0 + b * (uint32_t)n_base * TILE_BYTES; };
    auto item_slot = [&](uint32_t s) { return reinterpret_cast<const Item*>(s_items + s * ITEM_BYTES); };

    if (threadIdx.x == 0) {
        for (int s = 0; s < MAX_STAGES; ++s) { mbar_init(full_bar(s), strip ? 1 : 2); mbar_init(empty_bar(s), strip ? 2 : 1); }
        for (int a = 0; a < 4; ++a) {
            mbar_init(parked_bar(a), strip && a == 1 ? 2 : 1); mbar_init(sready_bar(a), 1);
            mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), EPI_WARPS);
        }
        mbar_init(drain_bar(0), 1); mbar_init(drain_bar(1), 1);
        for (int b = 0; b < MAX_BASE_SLOTS; ++b) { mbar_init(bfull_bar(b), 1); mbar_init(bempty_bar(b), EPI_WARPS); }
        for (int s = 0; s < ITEM_SLOTS; ++s) { mbar_init(ifull_bar(s), 1); mbar_init(iempty_bar(s), EPI_WARPS + (strip ? 4 : 3)); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == MMA_WARP) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tmem)), "r"(TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(s_tmem);

    // Tensor maps live in global memory (the plan's array): every CTA acquires a map through the tensormap proxy before its
    // first use IN THIS LAUNCH (a freed plan's storage may be handed to a new plan, and an SM could otherwise still hold the
    // old descriptor).  Each issuing warp remembers the last four maps it fenced, so a map costs one fence per CTA per run of
    // items that use it, not one per item.  Call from converged code.
    const CUtensorMap *fc0 = nullptr, *fc1 = nullptr, *fc2 = nullptr, *fc3 = nullptr;
    auto acq = [&](const CUtensorMap* mp) {
        if (mp != fc0 && mp != fc1 && mp != fc2 && mp != fc3) {
            if (elect_one()) tmap_acquire(mp);
            __syncwarp();
            fc3 = fc2; fc2 = fc1; fc1 = fc0; fc0 = mp;
        }
    };
    // optional profile (prof != nullptr): cycles each role spends in each kind of wait, per CTA
    long long pw[6] = {0, 0, 0, 0, 0, 0};
    const long long t_start = clock64();
#ifdef GF8_DEBUG
#define TRC(role, item, ev) do { if ((dbg & 2048) && prof && blockIdx.x == 1 && (item) < 48u && lane == 0) prof[8192 + ((role) * 48 + (item)) * 4 + (ev)] = clock64(); } while (0)
#else
#define TRC(role, item, ev) do {} while (0)
#endif
#define TWAIT(slot, expr) ([&]() { const long long _t0 = prof ? clock64() : 0; const bool _r = (expr); if (prof) pw[slot] += clock64() - _t0; return _r; })()
    if (warp == PRODUCER_WARP) {
        // ===== item fetch (whole warp) + TMA producer (lane 0) =====
        constexpr int NCHUNK = ITEM_BYTES / 16;
        uint32_t n_done = 0, b_bs = 0, b_bph = 0;
        int ok = 1;
        uint4 nxt = make_uint4(0, 0, 0, 0);
        auto claim = [&](int after) {          // index of this CTA's next item (claimed one item ahead of its use)
            if (!dyn) return after + (int)gridDim.x;
            int v = 0;
            if (lane == 0) v = atomicAdd(ctr, pair ? 2 : chunk);
            return __shfl_sync(0xFFFFFFFFu, v, 0);
        };
        int i = dyn ? claim(0) : (int)blockIdx.x;
        if (i < n_items && lane < NCHUNK) nxt = __ldg(reinterpret_cast<const uint4*>(items + i) + lane);
        for (; (dyn || i < n_items) && ok; ++n_done) {
            const uint32_t slot = n_done % ITEM_SLOTS, iphase = (n_done / ITEM_SLOTS) & 1u;
            if (lane == 0) ok = TWAIT(0, mbar_wait(iempty_bar(slot), iphase ^ 1u, err)) ? 1 : 0;
            ok = __shfl_sync(0xFFFFFFFFu, ok, 0);
            if (!ok) break;
            if (i >= n_items) {                 // (dynamic only) tell the other roles this CTA is done
                if (lane == 0) reinterpret_cast<Item*>(s_items + slot * ITEM_BYTES)->mode = EPI_END;
                __syncwarp();
                if (lane == 0) mbar_arrive(ifull_bar(slot));
                break;
            }
            if (lane < NCHUNK) reinterpret_cast<uint4*>(s_items + slot * ITEM_BYTES)[lane] = nxt;
            __syncwarp();
            if (lane == 0) mbar_arrive(ifull_bar(slot));
            TRC(0, n_done, 0);
            // pair launches: the amax item (even index) is followed by its cast item; the NEXT pair is claimed only after the
            // cast item's loads have been issued, i.e. after its epilogue has passed the tensor's join (the base ring is shorter
            // than a sub-strip): a pair claimed earlier could hold an amax item that this CTA's own waiting cast item needs
            const bool defer_claim = pair && (i & 1);
            if (pair && !(i & 1)) i = i + 1;
            else if (dyn && !pair && chunk > 1 && (i + 1) % chunk != 0 && i + 1 < n_items) i = i + 1;     // (next item of the claimed run)
            else if (!defer_claim) i = claim(i);
            if (!defer_claim && i < n_items && lane < NCHUNK) nxt = __ldg(reinterpret_cast<const uint4*>(items + i) + lane);
            if (strip) {
                // strip item: one base tile per (column tile, row block), in the order the epilogue consumes them
                const Item& it = *item_slot(slot);
                const int bm0 = it.base_map[0], row0 = it.row0, nrb = (it.rows + 127) >> 7, nct = (it.cols + 127) >> 7;
                const CUtensorMap* mp = maps + bm0;
                acq(mp);
                for (int ct = 0; ct < nct && ok; ++ct)
                    for (int rb = 0; rb < nrb && ok; ++rb) {
                        const uint32_t bs = b_bs, bph = b_bph;
                        if (++b_bs == (uint32_t)n_bslots) { b_bs = 0; b_bph ^= 1u; }
                        ok = TWAIT(1, mbar_wait(bempty_bar(bs), bph ^ 1u, err)) ? 1 : 0;
                        if (ok && elect_one()) {
                            if (dbg & 64) mbar_arrive(bfull_bar(bs));
                            else {
                            mbar_expect_tx(bfull_bar(bs), TILE_BYTES);
#pragma unroll
                            for (int h = 0; h < 2; ++h)
                                tma_load_2d(base_tile(bs) + h * 16384u, mp, it.col0 + 128 * ct + 64 * h, row0 + 128 * rb, bfull_bar(bs));
                            }
                        }
                        __syncwarp();
                    }
                if (defer_claim && ok) {
                    i = claim(i);
                    if (i < n_items && lane < NCHUNK) nxt = __ldg(reinterpret_cast<const uint4*>(items + i) + lane);
                }
            } else if (n_base > 0) {
                // the item's base tile(s): hi [+ lo], each two 64-column halves of 128 rows (converged warp, one
                // elected lane issues)
                const Item& it = *item_slot(slot);
                const uint32_t acc = n_done % (uint32_t)n_bslots, aphase = (n_done / (uint32_t)n_bslots) & 1u;
                ok = TWAIT(1, mbar_wait(bempty_bar(acc), aphase ^ 1u, err)) ? 1 : 0;
                if (ok) {
                    const int bm0 = it.base_map[0], bm1 = it.base_map[1], col0 = it.col0, row0 = it.row0;
                    const int nb = (bm0 >= 0 ? 1 : 0) + (bm1 >= 0 ? 1 : 0);
                    if (bm0 >= 0) acq(maps + bm0);
                    if (bm1 >= 0) acq(maps + bm1);
                    if (elect_one()) {
                        if (nb == 0 || (dbg & 64)) mbar_arrive(bfull_bar(acc));
                        else {
                            mbar_expect_tx(bfull_bar(acc), (uint32_t)nb * TILE_BYTES);
                            for (int b = 0; b < nb; ++b) {
                                const CUtensorMap* mp = maps + (b ? bm1 : bm0);
                                const uint32_t dst = base_tile(acc) + (uint32_t)b * TILE_BYTES;
#pragma unroll
                                for (int h = 0; h < 2; ++h) tma_load_2d(dst + h * 16384u, mp, col0 + 64 * h, row0, bfull_bar(acc));
                            }
                        }
                    }
                    __syncwarp();
                }
                TRC(0, n_done, 1);
            }
            ok = __shfl_sync(0xFFFFFFFFu, ok, 0);
        }
    } else if (warp == OPERAND_WARP || warp == OPERAND_WARP + 1) {
        // ===== operand TMA producers (one lane each): warp 9 streams the A K-atoms, warp 10 the B K-atoms =====
        // (a TMA issue costs ~200 cycles of the issuing thread, so the two operands get a warp each)
        {
            const bool is_b = warp != OPERAND_WARP;
            uint32_t stage = 0, phase = 0, n_done = 0;
            bool ok = true;
            for (int i = blockIdx.x; (dyn || i < n_items) && ok; i += gridDim.x, ++n_done) {
                const uint32_t slot = n_done % ITEM_SLOTS, iphase = (n_done / ITEM_SLOTS) & 1u;
                if (!(ok = TWAIT(3, mbar_wait(ifull_bar(slot), iphase, err)))) break;
                if (dyn && item_slot(slot)->mode == EPI_END) break;
                const Item& it = *item_slot(slot);
                if (strip) {
                    // strip item: warp 9 loads the strip's resident A tiles once ([row block][K-atom]); warp 10 streams
                    // the B K-atoms of every column tile through the 16 KB ring (each serves both row blocks)
                    const int nrb = (it.rows + 127) >> 7, nct = (it.cols + 127) >> 7;
                    const int na = it.atoms[0] + it.atoms[1];
                    for (int seg = 0; seg < 2; ++seg)
                        if (it.atoms[seg] > 0) acq(maps + (is_b ? it.map_b[seg] : it.map_a[seg]));
                    if (!is_b) {
                        if (!(ok = TWAIT(2, mbar_wait(parked_bar(1), (n_done & 1u) ^ 1u, err)))) break;   // L buffer free
                        if (elect_one()) {
                            mbar_expect_tx(parked_bar(0), (uint32_t)(nrb * na) * A_BYTES);
                            for (int rb = 0; rb < nrb; ++rb) {
                                int a = 0;
                                for (int seg = 0; seg < 2; ++seg)
                                    for (int t = 0; t < it.atoms[seg]; ++t, ++a)
                                        tma_load_2d(smem0 + (uint32_t)(rb * 2 + a) * A_BYTES, maps + it.map_a[seg],
                                                    it.a_c0[seg] + 64 * t, it.a_r0[seg] + 128 * rb, parked_bar(0));
                            }
                        }
                        __syncwarp();
                    } else {
                        // one ring stage = the (up to two) B K-atoms of a column tile, under one barrier pair
                        for (int ct = 0; ct < nct && ok; ++ct) {
                            if (!TWAIT(2, mbar_wait(empty_bar(stage), phase ^ 1u, err))) { ok = false; break; }
                            if (elect_one()) {
                                if (dbg & 128) mbar_arrive(full_bar(stage));
                                else {
                                    mbar_expect_tx(full_bar(stage), (uint32_t)na * B_BYTES);
                                    int a = 0;
                                    for (int seg = 0; seg < 2; ++seg)
                                        for (int t = 0; t < it.atoms[seg]; ++t, ++a)
                                            tma_load_2d(smem0 + STRIP_L_BYTES + (stage * 2u + (uint32_t)a) * B_BYTES, maps + it.map_b[seg],
                                                        it.b_c0[seg] + 64 * t, it.b_r0[seg] + 128 * ct, full_bar(stage));
                                }
                            }
                            __syncwarp();
                            if (++stage == (uint32_t)STRIP_RING) { stage = 0; phase ^= 1u; }
                        }
                    }
                    __syncwarp();
                    if (elect_one()) mbar_arrive(iempty_bar(slot));
                    continue;
                }
                const int a_mn = it.a_mn, b_mn = it.b_mn, nbx = it.N >> 6;
                const int nrb = (wide && it.rows > 128) ? 2 : 1;
                const uint32_t tx = is_b ? (uint32_t)it.N * 128u : (uint32_t)(nrb * A_BYTES);
                if (tri) {
                    // interleaved split products: per K-atom the hi and the lo tile of this warp's operand, once each
                    const CUtensorMap* m_hi = maps + (is_b ? it.map_b[0] : it.map_a[0]);
                    const CUtensorMap* m_lo = maps + (is_b ? it.map_b[2] : it.map_a[1]);
                    const int c0 = is_b ? it.b_c0[0] : it.a_c0[0], r0 = is_b ? it.b_r0[0] : it.a_r0[0];
                    acq(m_hi);
                    acq(m_lo);
                    for (int t = 0; t < it.atoms[0]; ++t) {
                        if (!TWAIT(2, mbar_wait(empty_bar(stage), phase ^ 1u, err))) { ok = false; break; }
                        const uint32_t sa = smem0 + stage * stage_bytes;
                        if (elect_one()) {
                            mbar_expect_tx(full_bar(stage), 2u * tx);
                            for (int v = 0; v < 2; ++v) {
                                const CUtensorMap* mp = v ? m_lo : m_hi;
                                if (is_b) {               // N rows x 64 columns, one box (B is K-major in panel items)
                                    tma_load_2d(sa + b_off + (uint32_t)v * 8192u, mp, c0 + 64 * t, r0, full_bar(stage));
                                } else if (a_mn) {
                                    for (int rb = 0; rb < nrb; ++rb) {
                                        const uint32_t d = sa + 32768u * v + 16384u * rb;
                                        tma_load_2d(d, mp, c0 + 128 * rb, r0 + 64 * t, full_bar(stage));
                                        tma_load_2d(d + 8192, mp, c0 + 128 * rb + 64, r0 + 64 * t, full_bar(stage));
                                    }
                                } else {
                                    for (int rb = 0; rb < nrb; ++rb)
                                        tma_load_2d(sa + 32768u * v + 16384u * rb, mp, c0 + 64 * t, r0 + 128 * rb, full_bar(stage));
                                }
                            }
                        }
                        __syncwarp();
                        if (++stage == (uint32_t)n_stages) { stage = 0; phase ^= 1u; }
                    }
                    __syncwarp();
                    if (elect_one()) mbar_arrive(iempty_bar(slot));
                    continue;
                }
                TRC(is_b ? 2 : 1, n_done, 0);
#pragma unroll 1
                for (int seg = 0; seg < NSEG && ok; ++seg) {
                    const int na = it.atoms[seg];
                    if (na <= 0) continue;
                    const CUtensorMap* mp = maps + (is_b ? it.map_b[seg] : it.map_a[seg]);
                    const int c0 = is_b ? it.b_c0[seg] : it.a_c0[seg], r0 = is_b ? it.b_r0[seg] : it.a_r0[seg];
                    acq(mp);
                    for (int t = 0; t < na; ++t) {
                        if (!TWAIT(2, mbar_wait(empty_bar(stage), phase ^ 1u, err))) { ok = false; break; }
                        const uint32_t sa = smem0 + stage * stage_bytes;
                        if (elect_one()) {
                            mbar_expect_tx(full_bar(stage), tx);
                            if (is_b && b_mn) {       // N / 64 boxes of 64 K-rows x 64 contiguous N elements
                                for (int h = 0; h < nbx; ++h)
                                    tma_load_2d(sa + b_off + 8192u * h, mp, c0 + 64 * h, r0 + 64 * t, full_bar(stage));
                            } else if (is_b) {        // N rows x 64 columns, one box
                                tma_load_2d(sa + b_off, mp, c0 + 64 * t, r0, full_bar(stage));
                            } else if (a_mn) {        // per row block two 64 x 64 boxes: 64 K-rows of 128 contiguous M elements
                                for (int rb = 0; rb < nrb; ++rb) {
                                    tma_load_2d(sa + 16384u * rb, mp, c0 + 128 * rb, r0 + 64 * t, full_bar(stage));
                                    tma_load_2d(sa + 16384u * rb + 8192, mp, c0 + 128 * rb + 64, r0 + 64 * t, full_bar(stage));
                                }
                            } else {                  // per row block one 128-row x 64-column box
                                for (int rb = 0; rb < nrb; ++rb)
                                    tma_load_2d(sa + 16384u * rb, mp, c0 + 64 * t, r0 + 128 * rb, full_bar(stage));
                            }
                        }
                        __syncwarp();
                        if (seg == 0 && t == 0) TRC(is_b ? 2 : 1, n_done, 1);
                        if (++stage == (uint32_t)n_stages) { stage = 0; phase ^= 1u; }
                    }
                }
                TRC(is_b ? 2 : 1, n_done, 2);
                __syncwarp();
                if (elect_one()) mbar_arrive(iempty_bar(slot));
            }
        }
    } else if (warp == MMA_WARP || (strip && warp == SYNC_WARP)) {
        // ===== MMA issuer (converged warp, one elected lane issues) =====
        // Strip items have two issuers: warp 11 takes row block 0 of every column tile, warp 12 row block 1.  One
        // issuer's serial stream (barrier waits, fences, 8 MMAs and the commits of a tile) is otherwise what bounds the
        // tile rate (measured: ~1400 cycles per tile with everything else switched off).
        {
            uint32_t stage = 0, phase = 0, n_done = 0, t_count = 0;
            bool ok = true;
            for (int i = blockIdx.x; (dyn || i < n_items) && ok; i += gridDim.x, ++n_done) {
                const uint32_t slot = n_done % ITEM_SLOTS, iphase = (n_done / ITEM_SLOTS) & 1u;
                if (!(ok = TWAIT(0, mbar_wait(ifull_bar(slot), iphase, err)))) break;
                if (dyn && item_slot(slot)->mode == EPI_END) break;
                const Item& it = *item_slot(slot);
                const int a_mn = it.a_mn, b_mn = it.b_mn;
                const uint32_t idesc = instr_desc(it.N, a_mn, b_mn);
                int total = 0;
#pragma unroll
                for (int seg = 0; seg < NSEG; ++seg) total += it.atoms[seg];
                if (strip) {
                    // strip item: A tiles resident, per column tile the B atoms serve both row blocks
                    const int nrb = (it.rows + 127) >> 7, nct = (it.cols + 127) >> 7;
                    const int rb = warp == MMA_WARP ? 0 : 1;
                    const bool mine = rb < nrb;              // (a 128-row strip: the second issuer only keeps the barriers in step)
                    __syncwarp();
                    if (elect_one()) mbar_arrive(iempty_bar(slot));
                    if (!(ok = TWAIT(0, mbar_wait(parked_bar(0), n_done & 1u, err)))) break;       // A tiles landed
                    tc_fence_after();
                    for (int ct = 0; ct < nct && ok; ++ct) {
                        const uint32_t tc_ = t_count + (uint32_t)rb;
                        const uint32_t acc = tc_ % n_acc, aphase = (tc_ / n_acc) & 1u;
                        t_count += (uint32_t)nrb;
                        if (mine) {
                            if (!(ok = TWAIT(1, mbar_wait(tempty_bar(acc), aphase ^ 1u, err)))) break;
                            tc_fence_after();
                        }
                        const uint32_t d = tmem_base + acc * 128u;
                        if (!(ok = TWAIT(2, mbar_wait(full_bar(stage), phase, err)))) break;     // both B atoms of the column tile
                        tc_fence_after();
                        if (elect_one()) {
                            if (mine && !(dbg & 1))
                                for (int a = 0; a < total; ++a) {
                                    const uint32_t sa = smem0 + (uint32_t)(rb * 2 + a) * A_BYTES;
                                    const uint32_t sb = smem0 + STRIP_L_BYTES + (stage * 2u + (uint32_t)a) * B_BYTES;
#pragma unroll
                                    for (int kk = 0; kk < 4; ++kk)
                                        tc_mma_bf16(d, smem_desc(sa + 32u * kk, 16u, 1024u), smem_desc(sb + 32u * kk, 16u, 1024u),
                                                    idesc, (a | kk) ? 1u : 0u);
                                }
                            tc_commit(empty_bar(stage));         // (two arrivals free the ring stage: one per issuer)
                            if (mine) tc_commit(tfull_bar(acc));
                        }
                        __syncwarp();
                        if (++stage == (uint32_t)STRIP_RING) { stage = 0; phase ^= 1u; }
                    }
                    if (ok && elect_one()) tc_commit(parked_bar(1));       // A tiles free once these MMAs retire
                    __syncwarp();
                    continue;
                }
                __syncwarp();
                if (elect_one()) mbar_arrive(iempty_bar(slot));
                TRC(3, n_done, 0);
                const uint32_t acc = n_done % n_acc, aphase = (n_done / n_acc) & 1u;
                if (!(ok = TWAIT(1, mbar_wait(tempty_bar(acc), aphase ^ 1u, err)))) break;
                tc_fence_after();
                TRC(3, n_done, 1);
                const uint32_t d = tmem_base + acc * 128u;
                const bool nrb2 = wide && it.rows > 128;
                if (tri) total = it.atoms[0];              // one ring stage per K-atom carries all three products
                for (int t = 0; t < total; ++t) {
                    if (!(ok = TWAIT(2, mbar_wait(full_bar(stage), phase, err)))) break;
                    tc_fence_after();
                    if (t == 0) TRC(3, n_done, 2);
                    const uint32_t sa = smem0 + stage * stage_bytes, sb = sa + b_off;
                    if (elect_one()) {
#pragma unroll
                        for (int kk = 0; kk < 4; ++kk) {
                            const uint64_t da = a_mn ? smem_desc(sa + 2048u * kk, 8192u, 1024u) : smem_desc(sa + 32u * kk, 16u, 1024u);
                            const uint64_t db = b_mn ? smem_desc(sb + 2048u * kk, 8192u, 1024u) : smem_desc(sb + 32u * kk, 16u, 1024u);
                            if (!(dbg & 1)) tc_mma_bf16(d, da, db, idesc, (t | kk) ? 1u : 0u);
                            if (nrb2 && !(dbg & 1)) {     // second row block: A 16 KB further on, accumulator 64 columns further on
                                const uint64_t da2 = a_mn ? smem_desc(sa + 16384u + 2048u * kk, 8192u, 1024u)
                                                          : smem_desc(sa + 16384u + 32u * kk, 16u, 1024u);
                                tc_mma_bf16(d + 64u, da2, db, idesc, (t | kk) ? 1u : 0u);
                            }
                            if (tri && !(dbg & 1)) {      // + A_lo * B_hi + A_hi * B_lo (A_lo 32 KB, B_lo 8 KB further on)
                                const uint64_t db_lo = smem_desc(sb + 8192u + 32u * kk, 16u, 1024u);
                                for (int rb = 0; rb < (nrb2 ? 2 : 1); ++rb) {
                                    const uint32_t a_hi = sa + 16384u * rb, a_lo = a_hi + 32768u;
                                    const uint64_t dl = a_mn ? smem_desc(a_lo + 2048u * kk, 8192u, 1024u) : smem_desc(a_lo + 32u * kk, 16u, 1024u);
                                    const uint64_t dh = a_mn ? smem_desc(a_hi + 2048u * kk, 8192u, 1024u) : smem_desc(a_hi + 32u * kk, 16u, 1024u);
                                    tc_mma_bf16(d + 64u * rb, dl, db, idesc, 1u);
                                    tc_mma_bf16(d + 64u * rb, dh, db_lo, idesc, 1u);
                                }
                            }
                        }
                        tc_commit(empty_bar(stage));      // frees the smem stage when these MMAs retire
                    }
                    __syncwarp();
                    if (++stage == (uint32_t)n_stages) { stage = 0; phase ^= 1u; }
                }
                if (ok && elect_one()) tc_commit(tfull_bar(acc));   // accumulator complete -> epilogue
                __syncwarp();
                TRC(3, n_done, 3);
            }
            // Drain: commits complete in issue order, so once this last one has arrived no mbarrier arrive of this
            // issuer is still in flight when the CTA exits (a late arrive would land in the shared memory of the
            // next kernel's CTA on this SM).
            if (ok) {
                const uint32_t db = drain_bar(warp == MMA_WARP ? 0 : 1);
                if (elect_one()) tc_commit(db);
                __syncwarp();
                mbar_wait(db, 0u, err);
            }
        }
    } else if (warp == SYNC_WARP) {
        // ===== fused update: grid-level bookkeeping off the epilogue's critical path (one lane) =====
        // add(n): tile n is parked -> bump its tensor's counter.  resolve(n - FUSE_LAG): wait until that tensor's
        // counter is complete, read its amax, publish the scale in shared memory and release cast(n - FUSE_LAG).
        // Lane a serves TMEM slot a (tiles n = a, a + 4, ...): bump (release) then poll (acquire), so the four
        // slots' round trips to L2 overlap and no lane's wait holds back another tile's bump.
        if (fuse && lane < 4) {
            uint32_t my_items = 0;
            for (int i = blockIdx.x; i < n_items; i += gridDim.x) ++my_items;
            for (uint32_t n = (uint32_t)lane; n < my_items; n += 4) {
                const uint32_t acc = n & 3u;
                if (!mbar_wait(parked_bar(acc), (n >> 2) & 1u, err)) break;
                const Parked pk = s_park[acc];
                asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(pk.done) : "memory");
                uint32_t spin = 0, seen = 0;
                bool bad = false;
                for (;;) {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(pk.done) : "memory");
                    if (seen >= (uint32_t)pk.total) break;
                    if (++spin > (1u << 24) || ((spin & 0x3FF) == 0 && *reinterpret_cast<volatile int*>(err))) { bad = true; break; }
                }
                if (bad) { atomicExch(err, 2); break; }
                float scale, si;
                scales_from_amax(*reinterpret_cast<volatile uint32_t*>(pk.amax), pk.fmt == 0 ? 448.0f : 57344.0f, scale, si);
                if (pk.write_scale) *pk.scale_inv_out = si;
                s_scale[acc] = scale;
                mbar_arrive(sready_bar(acc));
            }
        }
    } else if (fuse) {
        // ===== epilogue warps 0..7, FUSED update (a4 + a5 + a6 in one pass over the gradient) =====
        // park(n): W~ tile = base + acc, its amax goes to the tensor's amax word, the FP32 tile is written back into
        // its TMEM slot and the tensor's done-counter is bumped.  cast(n - FUSE_LAG): once the counter says every
        // tile of that tensor is parked (spin on a global word; deadlock-free because a tensor's tiles are contiguous
        // in the item list, all CTAs are co-resident and FUSE_LAG >= ceil(tiles / grid)), the parked tile is read
        // back, scaled, cast and stored.  Four TMEM slots hold three parked tiles plus the one being computed.
        const int r = (warp & 3) * 32 + lane, half = warp >> 2;
        const uint32_t lane_off = ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(half * 64);
        const uint32_t code0 = base0 + (uint32_t)n_bslots * (uint32_t)n_base * TILE_BYTES;   // two code-tile buffers
        uint32_t my_items = 0;
        for (int i = blockIdx.x; i < n_items; i += gridDim.x) ++my_items;
        bool ok = true;
        auto cast_one = [&](uint32_t j) -> bool {
            const uint32_t acc = j & 3u;
            // the sync warp has seen the tensor's last tile parked and left its scale in shared memory
            if (!mbar_wait(sready_bar(acc), (j >> 2) & 1u, err)) return false;
            if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");   // staging buffer j & 1 is free
            epi_sync();
            const Parked pk = s_park[acc];
            const float scale = s_scale[acc];
            const uint32_t taddr = tmem_base + acc * 128u + lane_off;
            uint4 cd[4];
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                uint32_t a[32];
                tmem_ld32_nowait(taddr + 32u * g, a);
                tmem_wait();
                float v[32];
#pragma unroll
                for (int u = 0; u < 32; ++u) v[u] = __uint_as_float(a[u]);
                cd[2 * g] = pk.fmt == 0 ? codes16<0>(v, scale) : codes16<1>(v, scale);
                cd[2 * g + 1] = pk.fmt == 0 ? codes16<0>(v + 16, scale) : codes16<1>(v + 16, scale);
            }
            const uint32_t tile = code0 + (j & 1u) * CODE_TILE_BYTES;
#pragma unroll
            for (int q = 0; q < 4; ++q)
                sts128(tile + (uint32_t)r * 128u + (((uint32_t)(4 * half + q) ^ (uint32_t)(r & 7)) << 4), cd[q]);
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            tc_fence_before();
            epi_sync();
            if (threadIdx.x == 0) {
                tma_store_2d(maps + pk.out_map, tile, pk.col0, pk.row0);
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(acc));
            return true;
        };
        for (uint32_t n = 0; n < my_items && ok; ++n) {
            const uint32_t slot = n % ITEM_SLOTS, iphase = (n / ITEM_SLOTS) & 1u;
            const uint32_t acc = n & 3u, aphase = (n >> 2) & 1u;
            const uint32_t bs = n % (uint32_t)n_bslots, bphase = (n / (uint32_t)n_bslots) & 1u;
            ok = TWAIT(0, mbar_wait(ifull_bar(slot), iphase, err));
            ok = ok && TWAIT(1, mbar_wait(bfull_bar(bs), bphase, err));
            ok = ok && TWAIT(2, mbar_wait(tfull_bar(acc), aphase, err));
            ok = __all_sync(0xFFFFFFFFu, ok);
            if (!ok) break;
            tc_fence_after();
            const long long t_e0 = prof ? clock64() : 0;
            const Item& it = *item_slot(slot);
            const uint32_t taddr = tmem_base + acc * 128u + lane_off;
            const uint32_t row = base_tile(bs) + (uint32_t)half * 16384u + (uint32_t)r * 128u;
            uint32_t loc = 0;
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                float v[32];
                tile_values32(taddr, row, 1, r, g, v);
                uint32_t w[32];
#pragma unroll
                for (int u = 0; u < 32; ++u) { w[u] = __float_as_uint(v[u]); loc = max(loc, w[u] & 0x7FFFFFFFu); }
                tmem_st32(taddr + 32u * g, w);
            }
            tmem_wait_st();
            loc = warp_max_u32(loc);
            if (lane == 0 && loc != 0u) atomicMax(it.amax, loc);
            if (threadIdx.x == 0) {
                Parked pk;
                pk.out_map = it.out_map; pk.col0 = it.col0; pk.row0 = it.row0; pk.fmt = it.fmt;
                pk.write_scale = it.write_scale; pk.total = (int32_t)it.base_ld;
                pk.amax = it.amax; pk.scale_inv_out = it.scale_inv_out;
                pk.done = reinterpret_cast<uint32_t*>(const_cast<void*>(it.base));
                s_park[acc] = pk;
            }
            tc_fence_before();
            epi_sync();                       // base tile consumed, amax atomics issued, parked info visible
            if (threadIdx.x == 0) mbar_arrive(parked_bar(acc));
            if (lane == 0) mbar_arrive(bempty_bar(bs));
            __syncwarp();
            if (lane == 0) mbar_arrive(iempty_bar(slot));
            if (prof) pw[3] += clock64() - t_e0;
            const long long t_p0 = prof ? clock64() : 0;
            if (n >= (uint32_t)FUSE_LAG) ok = cast_one(n - FUSE_LAG);
            if (prof) pw[4] += clock64() - t_p0;
        }
        for (uint32_t j = my_items > (uint32_t)FUSE_LAG ? my_items - FUSE_LAG : 0u; j < my_items && ok; ++j) ok = cast_one(j);
        if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    } else {
        // ===== epilogue warps 0..7 =====
        uint32_t n_done = 0, s_tiles = 0, s_bs = 0, s_bph = 0;
        int pending_slot = -1;
        bool ok = true;
        for (int i = blockIdx.x; (dyn || i < n_items) && ok; i += gridDim.x, ++n_done) {
            const uint32_t slot = n_done % ITEM_SLOTS, iphase = (n_done / ITEM_SLOTS) & 1u;
            const uint32_t acc = n_done % n_acc, aphase = (n_done / n_acc) & 1u;
            const uint32_t bs = n_base > 0 ? n_done % (uint32_t)n_bslots : 0u, bphase = n_base > 0 ? (n_done / (uint32_t)n_bslots) & 1u : 0u;
            ok = TWAIT(0, mbar_wait(ifull_bar(slot), iphase, err));
            if (ok && dyn && item_slot(slot)->mode == EPI_END) break;
            // the tensor's amax (EPI_CAST) is fetched before the data waits, so its latency hides behind them
            float cast_scale = 1.0f, cast_si = 1.0f;
            if (ok && item_slot(slot)->mode == EPI_CAST && item_slot(slot)->sync == 2) {
                // join: every amax item of the tensor has counted itself done (each after its atomicMax and a fence)
                if (lane == 0) {
                    const volatile uint32_t* cnt = reinterpret_cast<const volatile uint32_t*>(item_slot(slot)->base);
                    const uint32_t want = (uint32_t)item_slot(slot)->base_ld;
                    uint32_t spins = 0;
                    while (*cnt < want) {
                        __nanosleep(200);
                        if (++spins > (1u << 23) || *reinterpret_cast<volatile int*>(err)) { atomicExch(err, 2); ok = false; break; }
                    }
                    __threadfence();
                }
                ok = __shfl_sync(0xFFFFFFFFu, ok ? 1 : 0, 0) != 0;
            }
            if (ok && item_slot(slot)->mode == EPI_CAST)
                scales_from_amax(*reinterpret_cast<volatile uint32_t*>(item_slot(slot)->amax), item_slot(slot)->fmt == 0 ? 448.0f : 57344.0f,
                                 cast_scale, cast_si);
            if (strip) {
                // strip item: (column tile, row block) tiles in order; one amax atomic per warp per strip
                ok = __all_sync(0xFFFFFFFFu, ok);
                if (!ok) break;
                const Item& it = *item_slot(slot);
                const int nrb = (it.rows + 127) >> 7, nct = (it.cols + 127) >> 7;
                uint32_t run_max = 0;
                // error feedback: the residual of a tile is asked into L2 two tiles ahead (a warp's share of a tile is 16 chunks
                // of 512 B = 64 lines: two per lane), so the epilogue's loads find it there instead of waiting on DRAM
                const float* ef_base = (EF && (it.mode == EPI_AMAX || it.mode == EPI_CAST || it.mode == EPI_BLOCKCAST))
                                           ? reinterpret_cast<const float*>(it.out_lo) : nullptr;
                auto ef_prefetch = [&](int t) {
                    if (!ef_base || t >= nct * nrb) return;
                    const int pct = t / nrb, prb = t % nrb;
                    const float* tile = ef_base + ((int64_t)((it.row0 >> 7) + prb) * ((it.out_ld + 127) >> 7) + (it.col0 >> 7) + pct) * EF_TILE;
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const int line = 2 * lane + u, chunk = line >> 2, sub = line & 3;      // chunk = g * 8 + q of this warp's half
                        const float* a = tile + (((2 * (warp >> 2) + (chunk >> 3)) * 8 + (chunk & 7)) * 128 + 32 * (warp & 3) + 8 * sub) * 4;
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
                    }
                };
                ef_prefetch(0);
                ef_prefetch(1);
                for (int ct = 0; ct < nct && ok; ++ct)
                    for (int rb = 0; rb < nrb && ok; ++rb, ++s_tiles) {
                        ef_prefetch(ct * nrb + rb + 2);
                        const uint32_t sacc = s_tiles % n_acc, saph = (s_tiles / n_acc) & 1u;
                        const uint32_t sbs = s_bs, sbph = s_bph;       // = s_tiles % n_bslots, (s_tiles / n_bslots) & 1
                        if (++s_bs == (uint32_t)n_bslots) { s_bs = 0; s_bph ^= 1u; }
                        ok = TWAIT(1, mbar_wait(bfull_bar(sbs), sbph, err));
                        ok = ok && TWAIT(2, mbar_wait(tfull_bar(sacc), saph, err));
                        ok = __all_sync(0xFFFFFFFFu, ok);
                        if (!ok) break;
                        tc_fence_after();
                        const long long t_s0 = prof ? clock64() : 0;
                        if (!(dbg & 32))
                            epilogue_tile<EF>(it, tmem_base + sacc * 128u, base_tile(sbs), 1, warp, lane, s_red, maps, cast_scale, cast_si,
                                          it.row0 + 128 * rb, it.col0 + 128 * ct, it.write_scale != 0 && ct == 0 && rb == 0,
                                          it.mode == EPI_BLOCKCAST ? it.scale_inv_out + (size_t)((it.row0 >> 7) + rb) * nct + ct
                                                                   : it.scale_inv_out,
                                          &run_max);
                        tc_fence_before();
                        __syncwarp();
                        // (codes leave through plain stores, so the base slot goes straight back to the producer)
                        if (lane == 0) { mbar_arrive(tempty_bar(sacc)); mbar_arrive(bempty_bar(sbs)); }
                        if (prof) pw[3] += clock64() - t_s0;
                    }
                if (ok && it.mode == EPI_AMAX) {
                    run_max = warp_max_u32(run_max);
                    if (lane == 0) {
                        if (run_max != 0u) atomicMax(it.amax, run_max);
                        if (it.sync == 1) {       // (the maximum is performed before the count: fence between the two atomics)
                            __threadfence();
                            atomicAdd(reinterpret_cast<uint32_t*>(const_cast<void*>(it.base)), 1u);
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(iempty_bar(slot));
                continue;
            }
            if (warp == 0) TRC(4, n_done, 0);
            if (ok && n_base > 0) ok = TWAIT(1, mbar_wait(bfull_bar(bs), bphase, err));
            if (warp == 0) TRC(4, n_done, 1);
            ok = ok && TWAIT(2, mbar_wait(tfull_bar(acc), aphase, err));
            if (warp == 0) TRC(4, n_done, 2);
            const long long t_e0 = prof ? clock64() : 0;
            ok = __all_sync(0xFFFFFFFFu, ok);
            if (!ok) break;
            tc_fence_after();
            const Item& it = *item_slot(slot);
            bool stored = false;
            if (dbg & 32) {
            } else if (it.base_map[0] >= 0)
                stored = epilogue_tile<EF>(it, tmem_base + acc * 128u, base_tile(bs), it.base_map[1] >= 0 ? 2 : 1, warp, lane, s_red, maps, cast_scale, cast_si,
                                       it.row0, it.col0, it.write_scale != 0, it.scale_inv_out, nullptr);
            else {
                epilogue(it, tmem_base + acc * 128u, warp, lane, s_red, 0, dbg);
                if (wide && it.rows > 128) epilogue(it, tmem_base + acc * 128u, warp, lane, s_red, 1, dbg);
            }
            tc_fence_before();
            __syncwarp();
            if (warp == 0) TRC(4, n_done, 3);
            if (prof) pw[3] += clock64() - t_e0;
            const long long t_p0 = prof ? clock64() : 0;
            if (lane == 0) { mbar_arrive(tempty_bar(acc)); mbar_arrive(iempty_bar(slot)); }
            if (n_base > 0) {
                // the base slot goes back to the producer once every epilogue thread is done with it and the TMA
                // store issued from it (if any) has read it.  That store wait is deferred by one item, so it
                // overlaps the next tile instead of stalling this warp.
                if (lane == 0) {
                    if (pending_slot >= 0) {
                        // (the group just committed by this tile's own store may stay in flight)
                        if (stored) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
                        else asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
                        mbar_arrive(bempty_bar(pending_slot));
                    }
                    if (!stored) mbar_arrive(bempty_bar(bs));
                }
                pending_slot = stored ? (int)bs : -1;
            }
            if (prof) pw[4] += clock64() - t_p0;
        }
        if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // (pending slot: kernel ends)
    }
#undef TWAIT
    if (prof && lane == 0 && (warp == 0 || warp >= PRODUCER_WARP)) {
        const int role = warp == 0 ? 0 : warp - PRODUCER_WARP + 1;       // epilogue, base producer, A, B, MMA, MMA 2 / sync
        pw[5] = clock64() - t_start;
        for (int q = 0; q < 6; ++q) prof[((size_t)blockIdx.x * 6 + role) * 6 + q] = pw[q];
    }
    tc_fence_before();
    __syncthreads();
    if (warp == MMA_WARP) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
    }
}

}  // namespace tc
}  // namespace gf8
