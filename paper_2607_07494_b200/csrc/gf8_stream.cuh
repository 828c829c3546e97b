// gf8_stream.cuh -- the streaming codec engine (sm_100a): ONE persistent, warp-specialised kernel per batched
// call that runs the whole whitening transform of every (tensor, rank) problem -- projections, S, Q', rank-2k
// update, tensor-wide amax, FP8 cast (a3-a6; PAPER.md:158 Eq. 14, :250 Eq. 22, Alg. 1 l.10-13) -- tensor by tensor,
// so a gradient is fetched from HBM once and every later reader finds it in L2.
//
// Low-rank form:   P'  = (Wg U_A) E_A            row panels of 256 rows        (K_PANEL_P)
//                                Q^T = Wg^T U_G                column panels of 256 columns  (K_PANEL_Q)
//                                (S E_A)^T = sum_i P.(i)^T U_G(i)   partial per row panel, summed in panel order (K_SP)
//                                Q.^T = (Q^T + U_A (S E_A)^T) E_G   last K-step of the column panel item
//                                W~  = Wg + [P' | U_G] [U_A | Q'^T]^T   128 x 128 tiles      (K_UPD)
// Work hand-out: both pipelines claim their work from a list by atomic counter (list order is start order).  Pass-1 items run in
// tensor order.  The update list holds, per tensor with a per-tensor scale, its tiles TWICE: pass A (amax only) and, a few hundred
// tiles later in the list, pass B (recompute, scale, cast, store) -- a tile depends only on counters of earlier list entries, so
// no CTA ever waits on another CTA's progress through its own tiles (an earlier version parked the FP32 tile in TMEM across
// the tensor amax: with 3 parking slots per SM every tensor became a grid-wide barrier and tail latencies set the pace).
// Per-block scaling and the FP32 tap are single-pass.  A lead limit keeps pass-1 at most `lead` bytes of gradient ahead of the
// update, so the update's re-reads of the gradient hit L2.
//
// Two pipelines share every SM, so a long panel item never delays the CTA's update tiles (whose tensors complete in
// lock step across CTAs) and the HBM-bound streaming of new gradients overlaps the issue-bound update epilogues:
//   update pipeline: warp 0 scheduler (+ base-tile TMA), 1 operand TMA, 2 MMA issue, 3 grid-level sync, 10-25 epilogue (cast the slot's previous tile, then park)
//   pass-1 pipeline: warp 4 item claim + operand TMA, 5 MMA issue, 6-9 epilogue
#pragma once
#include "gf8_tc.cuh"

namespace gf8 {
namespace st {

using namespace gf8::tc;     // PTX wrappers (mbarrier, TMA, tcgen05)

constexpr int NS = 2;                       // pass-1 operand ring stages
constexpr int STG_BYTES = 40960;            // [A 32 KB | B 8 KB]
constexpr int US = 2;                       // update operand ring stages
constexpr int USTG_BYTES = 32768;           // [A 16 KB | B 16 KB]: one K-atom of an update tile
constexpr int NB = 2;                       // streamed base tiles in flight
constexpr int BASE_BYTES = 32768;           // 128 x 128 BF16 (two 64-column halves)
constexpr int RS = 8;                       // update item ring entries
constexpr int PRS = 4;                      // pass-1 item ring entries
constexpr int UCHUNK = 4;                   // update tiles per claim
constexpr int NPARK = 3;                    // TMEM slots 0..2: update tiles (parked); slot 3: pass-1 items
constexpr int S_DATA = NS * STG_BYTES + US * USTG_BYTES + NB * BASE_BYTES;     // 208 KB
constexpr int S_MISC = 4096;
constexpr int S_BYTES = S_DATA + S_MISC;
constexpr int S_THREADS = 832;
// warp roles: the spinning / issuing roles take the low warp ids, the arithmetic-heavy epilogues the high ones
constexpr int W_USCHED = 0, W_ULOAD = 1, W_UMMA = 2, W_SYNC = 3, W_PPROD = 4, W_PMMA = 5, W_PEPI = 6, W_UEPI = 10;
static_assert(S_BYTES <= 227 * 1024, "shared memory budget");

enum Kind : int32_t { K_END = 0, K_PANEL_P = 1, K_PANEL_Q = 2, K_SP = 3, K_UPD = 5 };
// STensor.mode: M_AMAX (per-tensor scale: two passes over the update tiles), M_BLOCK, M_TAP; RItem.mode also M_CAST (pass B)
enum Mode : int32_t { M_AMAX = 0, M_BLOCK = 1, M_TAP = 2, M_CAST = 3 };
enum Pass : int32_t { P_AMAX = 0, P_CAST = 1, P_SINGLE = 2 };
// words of a tensor's sync block (zeroed before every launch)
enum Sync : int32_t { SY_AMAX = 0, SY_P = 1, SY_Q = 2, SY_S = 3, SY_QP = 4, SY_TILES = 5, SY_DONE = 6, SY_WORDS = 8 };

// One (tensor, rank) problem of a batched call.  Static part written at plan build; `src`-maps, codes, scale_inv,
// tap are patched per call by patch_kernel.
struct __align__(16) STensor {
    int32_t m, n, useA, useG;
    int32_t fmt, mode, n_tiles, tiles_n;
    int32_t nP, nQ, nQP, dep_idx;          // item counts; update tiles wait for sync[dep_idx] >= dep_target
    int32_t dep_target, upd_start, map_src_p, map_src_q;
    int32_t map_src_b, map_UAt, map_UGt, map_UA128;
    int32_t map_UA256, map_UG128, map_Pp128, map_Pp64;
    int32_t map_Qpt128, map_SEA, pad0, pad1;
    bf16* Pp; float* Spart; bf16* Qpt; bf16* SEA;
    const float* eA; const float* eG;
    uint8_t* codes; float* scale_inv; float* tap;
    uint32_t* sync;
    int64_t byte_pos;                      // gradient bytes of the tensors before this one (lead control)
    int64_t pad2[7];
};
static_assert(sizeof(STensor) == 256, "tensor record size");

// Pass-1 item.  gate_tensor >= 0: a panel may start only when that (earlier) tensor's update is complete (gate_total tiles
// parked), which keeps the gradient bytes between the two pipelines' frontiers within L2 (lead control).
struct __align__(16) P1Item { int32_t kind, tensor, r0, rows, gate_tensor, gate_total, pad0, pad1; };
// Entry of the update list: tensor, tile coordinates (ti | tj << 16) and pass (P_AMAX / P_CAST / P_SINGLE).
struct __align__(16) TileEnt { int32_t tensor, tij, pass, pad; };

// What a role needs to know about an item (shared-memory ring entry, written by the scheduler warp).
struct __align__(16) RItem {
    int32_t kind, slot, r0, c0;
    int32_t rows, cols, ksteps, mode;
    int32_t mapA0, mapA1, mapB0, mapB1;
    int32_t fmt, ld, nrb, bslot;
    int32_t total, first; float scale; int32_t out_f32;   // scale: pass-B tiles (from the tensor's amax); first: fused Q' step (pass-1)
    void* out; const float* base32; const float* colscale; uint32_t* sync;
    float* scale_inv; uint32_t* done_ctr;
};
static_assert(sizeof(RItem) == 128, "ring entry size");


__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_prefetch_2d(const CUtensorMap* map, int c0, int c1) {
    asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global [%0, {%1, %2}];" ::"l"(map), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tma_prefetch_3d(const CUtensorMap* map, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global [%0, {%1, %2, %3}];" ::"l"(map), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    return done != 0;
}
__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity) {     // one try_wait: sleeps up to ~1 us unless the phase completes
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity), "r"(1000u) : "memory");
    return done != 0;
}
__device__ __forceinline__ void mbar_nap(uint32_t bar, uint32_t parity) {     // sleep until the phase completes, ~0.3 us at most
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t}"
        ::"r"(bar), "r"(parity), "r"(300u) : "memory");
}
__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t ld_relaxed(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add(uint32_t* p, uint32_t v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// d = float(bf16 half of w) + c   (one FHADD.BF16 each; exact widening, one FP32 rounding)
__device__ __forceinline__ void add_bf16x2(uint32_t w, float c0, float c1, float& d0, float& d1) {
    asm("{\n\t.reg .b16 lo, hi;\n\tmov.b32 {lo, hi}, %2;\n\tadd.rn.f32.bf16 %0, lo, %3;\n\tadd.rn.f32.bf16 %1, hi, %4;\n\t}"
        : "=f"(d0), "=f"(d1) : "r"(w), "f"(c0), "f"(c1));
}
// max(m, |a|, |b|), NaN-propagating (a NaN amax makes the scale 1, S13): one FMNMX3
__device__ __forceinline__ float max3abs(float m, float a, float b) {
    float r;
    asm("max.NaN.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(fabsf(a)), "f"(fabsf(b)), "f"(m));
    return r;
}
__device__ __forceinline__ void tmem_ld16_nowait(uint32_t taddr, uint32_t* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
        ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
          "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
        : "memory");
}
__device__ __forceinline__ void fence_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }
// four FP8 codes of (v0..v3) * s : packed multiplies + packed converts
template <int FMT>
__device__ __forceinline__ uint32_t cast4(float v0, float v1, float v2, float v3, float s) {
    uint64_t a, b, ss;
    asm("mov.b64 %0, {%1, %1};" : "=l"(ss) : "f"(s));
    asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(v0), "f"(v1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(v2), "f"(v3));
    asm("mul.rn.f32x2 %0, %0, %1;" : "+l"(a) : "l"(ss));
    asm("mul.rn.f32x2 %0, %0, %1;" : "+l"(b) : "l"(ss));
    float x0, x1, x2, x3;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x0), "=f"(x1) : "l"(a));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x2), "=f"(x3) : "l"(b));
    return f32x4_to_fp8x4<FMT>(x0, x1, x2, x3);
}


// ---- per-call pointer patch: codes / scale_inv / tap pointers and the three gradient maps of every problem --------
// ptrs[3 p + {0, 1, 2}] = gradient, codes (or tap), scale_inv of problem p.  tmpl[3 s + v]: map templates of shape s.
__global__ void patch_kernel(STensor* T, int nT, const void* const* ptrs, const int* shape_of, const CUtensorMap* tmpl,
                             CUtensorMap* maps, int tap) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= nT) return;
    STensor& t = T[p];
    if (tap) { t.tap = (float*)ptrs[3 * p + 1]; t.codes = nullptr; t.scale_inv = nullptr; }
    else { t.codes = (uint8_t*)ptrs[3 * p + 1]; t.scale_inv = (float*)ptrs[3 * p + 2]; t.tap = nullptr; }
    const int idx[3] = {t.map_src_p, t.map_src_q, t.map_src_b};
    for (int v = 0; v < 3; ++v) {
        const uint4* src = reinterpret_cast<const uint4*>(tmpl + 3 * shape_of[p] + v);
        uint4* dst = reinterpret_cast<uint4*>(maps + idx[v]);
#pragma unroll
        for (int q = 0; q < 8; ++q) dst[q] = src[q];
        asm volatile("tensormap.replace.tile.global_address.global.b1024.b64 [%0], %1;" ::"l"(maps + idx[v]), "l"(ptrs[3 * p]) : "memory");
    }
    asm volatile("fence.proxy.tensormap::generic.release.gpu;" ::: "memory");
}

// ---- the kernel ------------------------------------------------------------------------------------------------------
// GF8_STREAM_PROF (debug builds only): per-role cycle accounting, 8 counters per role per CTA, written to `prof`.
#ifdef GF8_STREAM_PROF
#define PROF_DECL long long pf[8] = {0, 0, 0, 0, 0, 0, 0, 0}; const long long pf_t0 = clock64();
#define PROF(slot, ...) { const long long _t = clock64(); __VA_ARGS__; pf[slot] += clock64() - _t; }
#define PROF_OUT(role) { pf[7] = clock64() - pf_t0; if (prof) for (int _q = 0; _q < 8; ++_q) prof[((size_t)blockIdx.x * 8 + (role)) * 8 + _q] = pf[_q]; }
#else
#define PROF_DECL
#define PROF(slot, ...) { __VA_ARGS__; }
#define PROF_OUT(role) {}
#endif
__global__ void __launch_bounds__(S_THREADS, 1)
stream_kernel(const STensor* __restrict__ T, int nT, const P1Item* __restrict__ p1, int n_p1, int n_upd,
              const TileEnt* __restrict__ tiles, const uint32_t* sync_base, const CUtensorMap* __restrict__ maps, int* ctr, int* err,
              int tap, long long* prof) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t smem0 = smem_u32(smem_raw);
    if (smem0 & 1023u) { if (threadIdx.x == 0) atomicExch(err, 3); return; }
    const uint32_t ustg0 = smem0 + NS * STG_BYTES;               // update operand stages
    const uint32_t base0 = ustg0 + US * USTG_BYTES;              // update base tiles
    const uint32_t bars = smem0 + S_DATA;
    uint8_t* misc = smem_raw + S_DATA;
    // update pipeline barriers
    auto full_bar = [&](uint32_t s) { return bars + 8u * s; };                  // [US]
    auto empty_bar = [&](uint32_t s) { return bars + 8u * (2 + s); };           // [US]
    auto bfull_bar = [&](uint32_t s) { return bars + 8u * (4 + s); };           // [NB]
    auto bempty_bar = [&](uint32_t s) { return bars + 8u * (6 + s); };          // [NB]
    auto tfull_bar = [&](uint32_t s) { return bars + 8u * (8 + s); };           // [4] (slot 3: pass-1)
    auto tempty_bar = [&](uint32_t s) { return bars + 8u * (12 + s); };         // [4]
    auto ifull_bar = [&](uint32_t s) { return bars + 8u * (16 + s); };          // [RS]
    auto iempty_bar = [&](uint32_t s) { return bars + 8u * (24 + s); };         // [RS]
    // pass-1 pipeline barriers
    auto pfull_bar = [&](uint32_t s) { return bars + 8u * (38 + s); };          // [NS]
    auto pempty_bar = [&](uint32_t s) { return bars + 8u * (40 + s); };         // [NS]
    auto pifull_bar = [&](uint32_t s) { return bars + 8u * (42 + s); };         // [PRS]
    auto piempty_bar = [&](uint32_t s) { return bars + 8u * (46 + s); };        // [PRS]
    const uint32_t plocal_bar = bars + 8u * 50, drain_bar0 = bars + 8u * 51, drain_bar1 = bars + 8u * 52;
    auto amax_bar = [&](uint32_t s) { return bars + 8u * (53 + s); };           // [RS]
    uint32_t* s_tmem = reinterpret_cast<uint32_t*>(misc + 496);
    uint32_t* s_wmax = reinterpret_cast<uint32_t*>(misc + 2832);         // [RS][16] warp maxima of pass-A tiles, per ring entry
    uint32_t* s_wblk = reinterpret_cast<uint32_t*>(misc + 3344);         // [2][16] warp maxima of per-block-scaled tiles
    RItem* s_items = reinterpret_cast<RItem*>(misc + 768);               // [RS] x 128 B   -> 1792
    RItem* s_pitems = reinterpret_cast<RItem*>(misc + 1792);             // [PRS] x 128 B  -> 2304
    STensor* s_cur = reinterpret_cast<STensor*>(misc + 2304);            // tensor of the next update tile   -> 2560
    STensor* s_p1t = reinterpret_cast<STensor*>(misc + 2560);            // tensor of the pass-1 item        -> 2816
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < US; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int s = 0; s < NB; ++s) { mbar_init(bfull_bar(s), 1); mbar_init(bempty_bar(s), 16); }
        for (int s = 0; s < 3; ++s) { mbar_init(tfull_bar(s), 1); mbar_init(tempty_bar(s), 16); }
        mbar_init(tfull_bar(3), 1); mbar_init(tempty_bar(3), 4);
        for (int s = 0; s < RS; ++s) { mbar_init(ifull_bar(s), 1); mbar_init(iempty_bar(s), 19); mbar_init(amax_bar(s), 16); }
        for (int s = 0; s < NS; ++s) { mbar_init(pfull_bar(s), 1); mbar_init(pempty_bar(s), 1); }
        for (int s = 0; s < PRS; ++s) { mbar_init(pifull_bar(s), 1); mbar_init(piempty_bar(s), 5); }
        mbar_init(plocal_bar, 1); mbar_init(drain_bar0, 1); mbar_init(drain_bar1, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == W_UMMA) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tmem)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(s_tmem);
    auto errset = [&]() { return *reinterpret_cast<volatile int*>(err) != 0; };
#ifdef GF8_STREAM_PROF
    // event trace of CTA 0 and CTA 77 (tiles < 48): prof[20480 + (cta ? 2048 : 0) + (code * 48 + tile)] = globaltimer
    auto EV = [&](int code, uint32_t tile) {
        if ((blockIdx.x == 0 || blockIdx.x == 77) && tile < 48u && prof) {
            unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
            prof[20480 + (blockIdx.x ? 2048 : 0) + code * 48 + tile] = (long long)t;
        }
    };
#else
    auto EV = [&](int, uint32_t) {};
#endif
    // bounded barrier wait; the first one that times out leaves its source line in err[1] (read by gf8_sync_check)
    auto mw = [&](int line, uint32_t bar, uint32_t par, int* e) -> bool {
#ifdef GF8_STREAM_PROF
        if (lane == 0 && prof) prof[16384 + blockIdx.x * 32 + warp] = line;       // heartbeat: the wait this warp is in
#endif
        if (mbar_wait(bar, par, e)) return true;
        atomicCAS(e + 1, 0, line);
        return false;
    };
    auto load_tensor = [&](STensor* dst, int t) {          // 256 B record, lanes 0..15 (the record is patched per call: read from L2)
        if (lane < 16) reinterpret_cast<uint4*>(dst)[lane] = __ldcg(reinterpret_cast<const uint4*>(T + t) + lane);
        __syncwarp();
    };
    // blocking poll of a counter (converged warp); the data it guards is only read through TMA / ld.global.cg, i.e. from L2,
    // where the producer's release made it visible before the counter moved
    auto poll_ge = [&](const uint32_t* p, uint32_t target) -> bool {
        uint32_t v = 0;
        for (uint32_t spin = 0;; ++spin) {
            if (lane == 0) v = ld_relaxed(p);
            v = __shfl_sync(0xFFFFFFFFu, v, 0);
            if (v >= target) return true;
            if (spin > (1u << 24) || ((spin & 255u) == 255u && errset())) { if (lane == 0) atomicExch(err, 4); return false; }
        }
    };

    if (warp == W_USCHED) {
        // ===== update scheduler (converged warp): claims the next tile of the update list (atomic counter: list order is start
        // order), waits until its tensor allows it, writes the ring entry and streams the tile's base =====
        PROF_DECL
        uint32_t nring = 0, q = 0;
        int cur_t = -1, cur_pass = -1;
        float cur_scale = 1.0f, cur_si = 1.0f;
        bool ok = true;
        auto push = [&](const RItem& it) -> bool {               // lane 0 writes the entry
            const uint32_t slot = nring % RS, ph = (nring / RS) & 1u;
            bool w_ok;
            PROF(0, w_ok = mw(__LINE__, iempty_bar(slot), ph ^ 1u, err));
            if (!w_ok) return false;
            if (lane == 0) {
                const uint4* src = reinterpret_cast<const uint4*>(&it);
                uint4* dst = reinterpret_cast<uint4*>(s_items + slot);
#pragma unroll
                for (int w = 0; w < 8; ++w) dst[w] = src[w];
                mbar_arrive(ifull_bar(slot));                     // (release: the entry is visible to whoever acquires the barrier)
            }
            __syncwarp();
            ++nring;
            return true;
        };
        // Tiles are claimed UCHUNK at a time (consecutive list entries: mostly one row block of one tensor and pass), and the
        // next chunk's claim and entries are fetched while this chunk is issued, so the scheduler's round trips to L2 (claim,
        // entries, tensor record, counter poll, amax) are paid once per chunk and off the critical path.
        int u_next = 0;
        TileEnt e_next = {0, 0, 0, 0};
        auto claim = [&]() {                       // lanes 0..UCHUNK-1 end up with their entry of the next chunk
            int u = 0;
            if (lane == 0) u = atomicAdd(ctr + 1, UCHUNK);
            u_next = __shfl_sync(0xFFFFFFFFu, u, 0);
            if (lane < UCHUNK && u_next + lane < n_upd) e_next = tiles[u_next + lane];
        };
        claim();
        while (ok && u_next < n_upd) {
            const int u0 = u_next;
            const TileEnt e_mine = e_next;
            claim();                               // (in flight while this chunk is issued)
          for (int ci = 0; ci < UCHUNK && ok && u0 + ci < n_upd; ++ci) {
            TileEnt ent;
            ent.tensor = __shfl_sync(0xFFFFFFFFu, e_mine.tensor, ci); ent.tij = __shfl_sync(0xFFFFFFFFu, e_mine.tij, ci);
            ent.pass = __shfl_sync(0xFFFFFFFFu, e_mine.pass, ci);
            const bool new_t = cur_t != ent.tensor;
            if (new_t) { cur_t = ent.tensor; cur_pass = -1; PROF(4, load_tensor(s_cur, cur_t)); }
            const STensor& t = *s_cur;
            // pass A / single-pass tiles wait for the tensor's Q' (or P') panels; pass B tiles for the tensor's amax (all A tiles counted)
            if (cur_pass != ent.pass) {            // (checked once per tensor and pass: the counters only grow)
                if (ent.pass == P_CAST) { PROF(2, ok = poll_ge(t.sync + SY_TILES, (uint32_t)t.n_tiles)); }
                else if (t.dep_target) { PROF(1, ok = poll_ge(t.sync + SY_QP, (uint32_t)t.dep_target)); }
                if (!ok) break;
                cur_pass = ent.pass;
                cur_scale = 1.0f;
                if (ent.pass == P_CAST) {
                    // (the count that poll_ge saw carries a data dependency on every tile's amax atomic: the maximum is final)
                    uint32_t bits = 0;
                    if (lane == 0) bits = *reinterpret_cast<volatile uint32_t*>(t.sync + SY_AMAX);
                    bits = __shfl_sync(0xFFFFFFFFu, bits, 0);
                    scales_from_amax(bits, t.fmt == 0 ? 448.0f : 57344.0f, cur_scale, cur_si);
                }
            }
            if (lane == 0) EV(0, q);
            const int ti = ent.tij & 0xFFFF, tj = ent.tij >> 16;
            RItem it;
            it.kind = K_UPD; it.slot = (int)(q % NPARK); it.r0 = ti * 128; it.c0 = tj * 128;
            it.rows = min(128, t.m - it.r0); it.cols = min(128, t.n - it.c0);
            it.ksteps = (t.useA ? 1 : 0) + (t.useG ? 1 : 0);
            it.mode = ent.pass == P_AMAX ? M_AMAX : (ent.pass == P_CAST ? M_CAST : t.mode);
            it.mapA0 = t.useA ? t.map_Pp128 : t.map_UG128; it.mapB0 = t.useA ? t.map_UA128 : t.map_Qpt128;
            it.mapA1 = t.map_UG128; it.mapB1 = t.map_Qpt128;
            it.fmt = t.fmt; it.ld = t.n; it.nrb = 1; it.bslot = (int)(q % NB);
            it.total = t.n_tiles; it.first = 0; it.out_f32 = 0;
            it.out = t.mode == M_TAP ? (void*)t.tap : (void*)t.codes; it.base32 = nullptr; it.colscale = nullptr; it.sync = t.sync;
            it.scale_inv = t.mode == M_BLOCK ? t.scale_inv + (size_t)ti * t.tiles_n + tj : t.scale_inv;
            it.done_ctr = nullptr;
            it.scale = cur_scale;
            if (ent.pass == P_CAST && (ti | tj) == 0 && lane == 0) *t.scale_inv = cur_si;
            if (!(ok = push(it))) break;
            // base tile: 128 rows x 128 columns of the gradient (two 64-column halves) in one 3-D box
            const uint32_t bs = q % NB, bph = (q / NB) & 1u;
            PROF(3, ok = mw(__LINE__, bempty_bar(bs), bph ^ 1u, err));
            if (!ok) break;
            if (lane == 0) {
                const CUtensorMap* mp = maps + t.map_src_b;
                tmap_acquire(mp);
                mbar_expect_tx(bfull_bar(bs), BASE_BYTES);
                tma_load_3d(base0 + bs * BASE_BYTES, mp, 0, it.r0, tj * 2, bfull_bar(bs));
            }
            ++q;
          }
        }
        if (lane == 0) PROF_OUT(0)
        __syncwarp();
        RItem e;
        e.kind = K_END;
        push(e);
    } else if (warp == W_ULOAD) {
        // ===== update operand loader (converged warp, one elected lane issues the TMA loads) =====
        uint32_t stage = 0, phase = 0;
        bool ok = true;
        PROF_DECL
        for (uint32_t nr = 0; ok; ++nr) {
            const uint32_t slot = nr % RS;
            PROF(0, ok = mw(__LINE__, ifull_bar(slot), (nr / RS) & 1u, err));
            if (!ok) break;
            const RItem& it = s_items[slot];
            if (it.kind == K_END) break;
            const int ksteps = it.ksteps, r0 = it.r0, c0 = it.c0;
            const CUtensorMap* mA0 = maps + it.mapA0; const CUtensorMap* mB0 = maps + it.mapB0;
            const CUtensorMap* mA1 = maps + it.mapA1; const CUtensorMap* mB1 = maps + it.mapB1;
            __syncwarp();
            if (elect_one()) {
                mbar_arrive(iempty_bar(slot));
                tmap_acquire(mA0); tmap_acquire(mB0);
                if (ksteps > 1) { tmap_acquire(mA1); tmap_acquire(mB1); }
                fence_async_global();      // P', Q'^T were written by other CTAs through the generic proxy
            }
            __syncwarp();
            for (int t = 0; t < ksteps && ok; ++t) {
                PROF(2, ok = mw(__LINE__, empty_bar(stage), phase ^ 1u, err));
                if (!ok) break;
                const uint32_t sa = ustg0 + stage * USTG_BYTES, fb = full_bar(stage);
                if (elect_one()) {
                    mbar_expect_tx(fb, 32768u);
                    tma_load_2d(sa, t ? mA1 : mA0, 0, r0, fb);
                    tma_load_2d(sa + 16384u, t ? mB1 : mB0, 0, c0, fb);
                }
                __syncwarp();
                if (++stage == US) { stage = 0; phase ^= 1u; }
            }
        }
        if (lane == 0) PROF_OUT(1)
    } else if (warp == W_UMMA) {
        // ===== update MMA issuer (converged warp, one elected lane issues) =====
        uint32_t stage = 0, phase = 0;
        bool ok = true;
        PROF_DECL
        const uint32_t idesc = instr_desc(128, 0, 0);
        for (uint32_t nr = 0; ok; ++nr) {
            const uint32_t rslot = nr % RS;
            PROF(0, ok = mw(__LINE__, ifull_bar(rslot), (nr / RS) & 1u, err));
            if (!ok) break;
            const RItem& it = s_items[rslot];
            if (it.kind == K_END) break;
            const int ksteps = it.ksteps;
            __syncwarp();
            if (elect_one()) mbar_arrive(iempty_bar(rslot));
            const uint32_t slot = nr % NPARK;                        // (every ring entry before K_END is an update tile)
            PROF(1, ok = mw(__LINE__, tempty_bar(slot), ((nr / NPARK) & 1u) ^ 1u, err));
            if (!ok) break;
            tc_fence_after();
            if (lane == 0) EV(2, nr);
            const uint32_t d = tmem_base + slot * 128u;
            for (int t = 0; t < ksteps && ok; ++t) {
                PROF(3, ok = mw(__LINE__, full_bar(stage), phase, err));
                if (!ok) break;
                tc_fence_after();
                const uint32_t sa = ustg0 + stage * USTG_BYTES, sb = sa + 16384u;
                if (elect_one()) {
#pragma unroll
                    for (int kk = 0; kk < 4; ++kk)
                        tc_mma_bf16(d, smem_desc(sa + 32u * kk, 16u, 1024u), smem_desc(sb + 32u * kk, 16u, 1024u), idesc, (t | kk) ? 1u : 0u);
                    tc_commit(empty_bar(stage));
                }
                __syncwarp();
                if (++stage == US) { stage = 0; phase ^= 1u; }
            }
            if (ok && elect_one()) tc_commit(tfull_bar(slot));
            __syncwarp();
            if (lane == 0) EV(3, nr);
        }
        if (lane == 0) PROF_OUT(2)
        if (ok) {      // drain: no commit of this issuer may still be in flight when the CTA exits
            if (elect_one()) tc_commit(drain_bar0);
            __syncwarp();
            mw(__LINE__, drain_bar0, 0u, err);
        }
    }
    else if (warp == W_SYNC) {
        // ===== amax publisher (lane 0, follows the item ring): for a pass-A tile, the maximum of the 16 epilogue warps' maxima goes
        // to the tensor's amax word and then the tile is counted; pass-B tiles start once the count is complete.  It has a warp of
        // its own because the atomic's round trip to L2 would otherwise hold up an epilogue warp.
        if (lane == 0) {
            uint32_t par_mask = 0;                           // phase parity of each ring slot's amax barrier (only pass-A tiles use it)
            for (uint32_t n = 0;; ++n) {
                const uint32_t rslot = n % RS;
                if (!mw(__LINE__, ifull_bar(rslot), (n / RS) & 1u, err)) break;
                const RItem& it = s_items[rslot];
                if (it.kind == K_END) break;
                if (it.mode == M_AMAX) {
                    uint32_t* sync = it.sync;
                    if (!mw(__LINE__, amax_bar(rslot), (par_mask >> rslot) & 1u, err)) break;
                    par_mask ^= 1u << rslot;
                    uint32_t mx = 0;
#pragma unroll
                    for (int w = 0; w < 16; ++w) mx = max(mx, s_wmax[rslot * 16 + w]);
                    mbar_arrive(iempty_bar(rslot));
                    // the tile's amax reaches L2 (an atomic WITH return has been performed when its value arrives) before the tile is
                    // counted: the count carries a data dependency on the returned value instead of a (slow) gpu-scope release fence
                    const uint32_t old = atomicMax(sync + SY_AMAX, mx);
                    asm volatile("red.relaxed.gpu.global.add.u32 [%0], %1;" ::"l"(sync + SY_TILES), "r"(1u + (old & 0u)) : "memory");
                } else {
                    mbar_arrive(iempty_bar(rslot));
                }
            }
        }
    } else if (warp >= W_UEPI) {
        // ===== update epilogue warps (16): warp w reaches TMEM lanes 32 (w & 3) .. +31 and takes the 32-column quarter (w - W_UEPI) >> 2
        // of the tile, so a tile is ONE TMEM round trip per warp.  W~ = base + accumulator, then by mode: running amax (pass A), scale +
        // FP8 cast + store (pass B), both with a CTA-level maximum in between (per-128x128-block scaling), or the FP32 tap =====
        const int q4 = warp & 3, cq = (warp - W_UEPI) >> 2, ew = warp - W_UEPI;
        const int r = q4 * 32 + lane;                           // accumulator row of this thread
        const uint32_t lane_off = ((uint32_t)(q4 * 32) << 16) + 32u * (uint32_t)cq;
        bool ok = true;
        uint32_t nblk = 0;
        PROF_DECL
        for (uint32_t nq = 0; ok; ++nq) {
            const uint32_t rslot = nq % RS, slot = nq % NPARK, bs = nq % NB;
            PROF(0, ok = mw(__LINE__, ifull_bar(rslot), (nq / RS) & 1u, err));
            if (!ok) break;
            const RItem& it = s_items[rslot];
            if (it.kind == K_END) break;
            const int mode = it.mode;
            PROF(1, ok = mw(__LINE__, tfull_bar(slot), (nq / NPARK) & 1u, err) && mw(__LINE__, bfull_bar(bs), (nq / NB) & 1u, err));
            if (!ok) break;
#ifdef GF8_STREAM_PROF
            const long long _tw = clock64();
#endif
            tc_fence_after();
            if (ew == 0 && lane == 0) EV(4, nq);
            const uint32_t brow = base0 + bs * BASE_BYTES + (uint32_t)(cq >> 1) * 16384u + (uint32_t)r * 128u;
            uint32_t a[32];
            tmem_ld32_nowait(tmem_base + slot * 128u + lane_off, a);
            uint4 b[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = lds128(brow + (((uint32_t)(4 * (cq & 1) + j) ^ (uint32_t)(r & 7)) << 4));
            tmem_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) { mbar_arrive(tempty_bar(slot)); mbar_arrive(bempty_bar(bs)); }     // accumulator and base are in registers
            float* v = reinterpret_cast<float*>(a);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t w[4] = {b[j].x, b[j].y, b[j].z, b[j].w};
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    add_bf16x2(w[e], v[8 * j + 2 * e], v[8 * j + 2 * e + 1], v[8 * j + 2 * e], v[8 * j + 2 * e + 1]);
            }
            const bool row_ok = r < it.rows;
            float scale = it.scale;
            if (mode == M_TAP) {
                if (row_ok) {
                    float* trow = reinterpret_cast<float*>(it.out) + (int64_t)(it.r0 + r) * it.ld + it.c0 + 32 * cq;
#pragma unroll
                    for (int h = 0; h < 8; ++h)
                        if (32 * cq + 4 * h < it.cols) *reinterpret_cast<float4*>(trow + 4 * h) = make_float4(v[4 * h], v[4 * h + 1], v[4 * h + 2], v[4 * h + 3]);
                }
            } else {
                if (mode != M_CAST) {
                    float mx = 0.0f;
#pragma unroll
                    for (int e = 0; e < 16; ++e) mx = max3abs(mx, v[2 * e], v[2 * e + 1]);
                    uint32_t wm;                                // (non-negative floats and NaN order as integers)
                    asm volatile("redux.sync.max.u32 %0, %1, 0xffffffff;" : "=r"(wm) : "r"(__float_as_uint(mx)));
                    if (mode == M_AMAX) {
                        // (one buffer and barrier per ring entry: the publisher warp frees the entry only after it has read them)
                        if (lane == 0) { s_wmax[rslot * 16 + ew] = wm; mbar_arrive(amax_bar(rslot)); }
                    } else {        // M_BLOCK: the 16 warps exchange their maxima (CTA-level barrier of the epilogue warps)
                        if (lane == 0) s_wblk[(nblk & 1u) * 16 + ew] = wm;
                        asm volatile("bar.sync 3, 512;" ::: "memory");
                        uint32_t bits = 0;
#pragma unroll
                        for (int w = 0; w < 16; ++w) bits = max(bits, s_wblk[(nblk & 1u) * 16 + w]);
                        ++nblk;
                        float si;
                        scales_from_amax(bits, it.fmt == 0 ? 448.0f : 57344.0f, scale, si);
                        if (ew == 0 && lane == 0) *it.scale_inv = si;
                    }
                }
                if (mode != M_AMAX) {
                    uint4 cd[2];
                    uint32_t* cw = reinterpret_cast<uint32_t*>(cd);
                    if (it.fmt == 0) {
#pragma unroll
                        for (int j = 0; j < 8; ++j) cw[j] = cast4<0>(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3], scale);
                    } else {
#pragma unroll
                        for (int j = 0; j < 8; ++j) cw[j] = cast4<1>(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3], scale);
                    }
                    if (row_ok) {
                        uint8_t* orow = reinterpret_cast<uint8_t*>(it.out) + (int64_t)(it.r0 + r) * it.ld + it.c0 + 32 * cq;
#pragma unroll
                        for (int h = 0; h < 2; ++h)
                            if (32 * cq + 16 * h < it.cols) *reinterpret_cast<uint4*>(orow + 16 * h) = cd[h];
                    }
                    // (lead control of the pass-1 pipeline counts finished tiles; an approximate count is all it needs)
                    if (ew == 0 && lane == 0) asm volatile("red.relaxed.gpu.global.add.u32 [%0], 1;" ::"l"(it.sync + SY_DONE) : "memory");
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(iempty_bar(rslot));
            if (ew == 0 && lane == 0) EV(5, nq);
#ifdef GF8_STREAM_PROF
            pf[2] += clock64() - _tw;
#endif
        }
        if (ew == 0 && lane == 0) PROF_OUT(3)
    }
    else if (warp == W_PPROD) {
        // ===== pass-1 producer (converged warp): claims the next item of the list, writes it into the pass-1 ring and streams its
        // operand K-steps; gradient K-steps are prefetched into L2 a few steps ahead of the two-stage shared-memory ring =====
        PROF_DECL
        uint32_t nring = 0, stage = 0, phase = 0, n_sp = 0;
        bool ok = true;
        auto push = [&](const RItem& it) -> bool {
            const uint32_t slot = nring % PRS, ph = (nring / PRS) & 1u;
            bool w_ok;
            PROF(0, w_ok = mw(__LINE__, piempty_bar(slot), ph ^ 1u, err));
            if (!w_ok) return false;
            if (lane == 0) {
                const uint4* src = reinterpret_cast<const uint4*>(&it);
                uint4* dst = reinterpret_cast<uint4*>(s_pitems + slot);
#pragma unroll
                for (int w = 0; w < 8; ++w) dst[w] = src[w];
                mbar_arrive(pifull_bar(slot));
            }
            __syncwarp();
            ++nring;
            return true;
        };
        // one K-step: wait for a free stage, then A (bytes_a) and B (8 KB) by TMA.  akind: 0 = 2-D box at (ca, ra), 1 = 3-D box at (0, ra, ca)
        auto kstep = [&](const CUtensorMap* mA, int akind, int ca, int ra, uint32_t bytes_a, const CUtensorMap* mB, int cb, int rb_) -> bool {
            bool w_ok;
            PROF(3, w_ok = mw(__LINE__, pempty_bar(stage), phase ^ 1u, err));
            if (!w_ok) return false;
            const uint32_t sa = smem0 + stage * STG_BYTES, fb = pfull_bar(stage);
            if (elect_one()) {
                mbar_expect_tx(fb, bytes_a + 8192u);
                if (akind) tma_load_3d(sa, mA, 0, ra, ca, fb); else tma_load_2d(sa, mA, ca, ra, fb);
                tma_load_2d(sa + 32768u, mB, cb, rb_, fb);
            }
            __syncwarp();
            if (++stage == NS) { stage = 0; phase ^= 1u; }
            return true;
        };
        constexpr int PF = 6;                         // L2 prefetch distance in K-steps (32 KB of gradient each)
        while (ok) {
            int c = 0;
            if (lane == 0) c = atomicAdd(ctr, 1);
            c = __shfl_sync(0xFFFFFFFFu, c, 0);
            if (c >= n_p1) break;
            P1Item pi;
            if (lane == 0) pi = p1[c];
            pi.kind = __shfl_sync(0xFFFFFFFFu, pi.kind, 0); pi.tensor = __shfl_sync(0xFFFFFFFFu, pi.tensor, 0);
            pi.r0 = __shfl_sync(0xFFFFFFFFu, pi.r0, 0); pi.rows = __shfl_sync(0xFFFFFFFFu, pi.rows, 0);
            pi.gate_tensor = __shfl_sync(0xFFFFFFFFu, pi.gate_tensor, 0); pi.gate_total = __shfl_sync(0xFFFFFFFFu, pi.gate_total, 0);
            PROF(4, load_tensor(s_p1t, pi.tensor));
            const STensor& t = *s_p1t;
            // lead control: this panel's tensor may not run further ahead of the update frontier than the plan's lead
            if (pi.gate_tensor >= 0) { PROF(1, ok = poll_ge(sync_base + (size_t)pi.gate_tensor * SY_WORDS + SY_DONE, (uint32_t)pi.gate_total)); if (!ok) break; }
            const bool both = t.useA && t.useG, isP = pi.kind == K_PANEL_P;
            RItem it;
            it.kind = pi.kind; it.slot = 3; it.r0 = pi.r0; it.c0 = 0; it.rows = pi.rows; it.cols = 64; it.mode = 0;
            it.mapA0 = isP ? t.map_src_p : t.map_src_q; it.mapB0 = isP ? t.map_UAt : t.map_UGt; it.mapA1 = it.mapB1 = -1;
            it.fmt = 0; it.ld = 64; it.nrb = pi.rows > 128 ? 2 : 1; it.bslot = 0;
            it.total = 0; it.first = (!isP && both) ? 1 : 0;              // first: a Q panel whose last K-step adds U_A (S E_A)^T
            it.scale = 1.0f; it.out_f32 = 0; it.base32 = nullptr; it.sync = t.sync; it.scale_inv = nullptr;
            const int base_steps = isP ? (t.n + 63) / 64 : (t.m + 63) / 64;
            it.ksteps = base_steps + it.first;
            it.out = isP ? (void*)t.Pp : (void*)t.Qpt; it.colscale = isP ? t.eA : t.eG;
            it.done_ctr = (isP && both) ? nullptr : t.sync + SY_QP;      // (a P panel of a two-sided layer is followed by its S partial)
            if (!(ok = push(it))) break;
            const CUtensorMap* mA = maps + it.mapA0; const CUtensorMap* mB = maps + it.mapB0;
            const int r0 = pi.r0;
            if (elect_one()) {
                tmap_acquire(mA); tmap_acquire(mB);
                for (int ks = 0; ks < min(PF, base_steps); ++ks) {
                    if (isP) tma_prefetch_2d(mA, 64 * ks, r0); else tma_prefetch_3d(mA, 0, 64 * ks, r0 >> 6);
                }
            }
            __syncwarp();
            for (int ks = 0; ks < base_steps && ok; ++ks) {
                if (ks + PF < base_steps && elect_one()) {
                    if (isP) tma_prefetch_2d(mA, 64 * (ks + PF), r0); else tma_prefetch_3d(mA, 0, 64 * (ks + PF), r0 >> 6);
                }
                __syncwarp();
                ok = isP ? kstep(mA, 0, 64 * ks, r0, 32768u, mB, 64 * ks, 0) : kstep(mA, 1, r0 >> 6, 64 * ks, 32768u, mB, 64 * ks, 0);
            }
            if (!ok) break;
            if (it.first) {
                // Q'^T = (Q^T + U_A (S E_A)^T) E_G: once the tensor's (S E_A)^T is complete, one more K-step adds U_A (S E_A)^T to
                // the Q^T accumulators (A = U_A rows of this column panel, K-major; B = (S E_A)^T as [g][a])
                PROF(2, ok = poll_ge(t.sync + SY_S, 1u));
                if (!ok) break;
                const CUtensorMap* mU = maps + t.map_UA256; const CUtensorMap* mS = maps + t.map_SEA;
                if (elect_one()) { tmap_acquire(mU); tmap_acquire(mS); fence_async_global(); }
                __syncwarp();
                if (!(ok = kstep(mU, 0, 0, r0, 32768u, mS, 0, 0))) break;
            } else if (isP && both) {
                // S partial of this row panel: (S E_A)^T_i = P'(i)^T U_G(i), K = the panel's rows; P'(i) was just written by this
                // CTA's pass-1 epilogue (local barrier), read back MN-major through TMA
                RItem sp = it;
                sp.kind = K_SP; sp.nrb = 1; sp.ksteps = (pi.rows + 63) / 64; sp.first = 0;
                sp.mapA0 = t.map_Pp64; sp.mapB0 = t.map_UGt;
                sp.out = t.Spart + (size_t)(r0 >> 8) * 4096; sp.base32 = t.Spart; sp.colscale = nullptr; sp.total = t.nP;
                sp.scale_inv = reinterpret_cast<float*>(t.SEA); sp.done_ctr = t.sync + SY_P;
                if (!(ok = push(sp))) break;
                PROF(2, ok = mw(__LINE__, plocal_bar, n_sp & 1u, err));
                ++n_sp;
                if (!ok) break;
                const CUtensorMap* mP = maps + t.map_Pp64; const CUtensorMap* mG = maps + t.map_UGt;
                if (elect_one()) { tmap_acquire(mP); tmap_acquire(mG); fence_async_global(); }
                __syncwarp();
                for (int ks = 0; ks < sp.ksteps && ok; ++ks) ok = kstep(mP, 0, 0, r0 + 64 * ks, 8192u, mG, r0 + 64 * ks, 0);
                if (!ok) break;
            }
        }
        if (lane == 0) PROF_OUT(4)
        RItem e;
        e.kind = K_END;
        push(e);
    } else if (warp == W_PMMA) {
        // ===== pass-1 MMA issuer: accumulators in TMEM slot 3 (two 64-column halves, one per 128-row block of the panel) =====
        uint32_t stage = 0, phase = 0;
        bool ok = true;
        PROF_DECL
        const uint32_t d = tmem_base + 3u * 128u;
        for (uint32_t nr = 0; ok; ++nr) {
            const uint32_t rslot = nr % PRS;
            PROF(0, ok = mw(__LINE__, pifull_bar(rslot), (nr / PRS) & 1u, err));
            if (!ok) break;
            const RItem& it = s_pitems[rslot];
            const int kind = it.kind;
            if (kind == K_END) break;
            const int ksteps = it.ksteps, nrb = it.nrb, fused = it.first;
            __syncwarp();
            if (elect_one()) mbar_arrive(piempty_bar(rslot));
            const bool mn = kind == K_PANEL_Q || kind == K_SP;
            PROF(1, ok = mw(__LINE__, tempty_bar(3), (nr & 1u) ^ 1u, err));
            if (!ok) break;
            tc_fence_after();
            for (int t = 0; t < ksteps && ok; ++t) {
                PROF(3, ok = mw(__LINE__, pfull_bar(stage), phase, err));
                if (!ok) break;
                tc_fence_after();
                const uint32_t sa = smem0 + stage * STG_BYTES, sb = sa + 32768u;
                const bool a_mn = mn && !(fused && t == ksteps - 1);          // (the fused Q' step reads U_A K-major)
                const uint32_t idesc = instr_desc(64, a_mn ? 1 : 0, 0);
                if (elect_one()) {
#pragma unroll
                    for (int kk = 0; kk < 4; ++kk) {
                        const uint64_t db = smem_desc(sb + 32u * kk, 16u, 1024u);
                        for (int rb = 0; rb < nrb; ++rb) {
                            const uint64_t da = a_mn ? smem_desc(sa + 16384u * rb + 2048u * kk, 8192u, 1024u)
                                                     : smem_desc(sa + 16384u * rb + 32u * kk, 16u, 1024u);
                            tc_mma_bf16(d + 64u * rb, da, db, idesc, (t | kk) ? 1u : 0u);
                        }
                    }
                    tc_commit(pempty_bar(stage));
                }
                __syncwarp();
                if (++stage == NS) { stage = 0; phase ^= 1u; }
            }
            if (ok && elect_one()) tc_commit(tfull_bar(3));
            __syncwarp();
        }
        if (lane == 0) PROF_OUT(5)
        if (ok) {
            if (elect_one()) tc_commit(drain_bar1);
            __syncwarp();
            mw(__LINE__, drain_bar1, 0u, err);
        }
    } else {
        // ===== pass-1 epilogue warps W_PEPI..+3 (a warp reaches the TMEM lane quarter warp & 3): panel rows straight to global memory =====
        const int q4 = warp & 3;
        const int r = q4 * 32 + lane, tid = threadIdx.x - W_PEPI * 32;
        const uint32_t lane_off = (uint32_t)(q4 * 32) << 16;
        volatile int* s_last = reinterpret_cast<volatile int*>(misc + 504);
        volatile int* s_pok = reinterpret_cast<volatile int*>(misc + 2816);      // [4]
        bool ok = true;
        PROF_DECL
        auto group_sync = [&]() { asm volatile("bar.sync 2, 128;" ::: "memory"); };
        for (uint32_t nr = 0; ok; ++nr) {
            const uint32_t rslot = nr % PRS;
            PROF(0, ok = mw(__LINE__, pifull_bar(rslot), (nr / PRS) & 1u, err));
            const RItem& it = s_pitems[rslot];
            const int kind = it.kind;
            if (ok && kind == K_END) break;
            if (ok) { PROF(1, ok = mw(__LINE__, tfull_bar(3), nr & 1u, err)); }
            // the four warps leave together (they meet at CTA-level barriers below): agree on `ok` first
            if (lane == 0) s_pok[warp - W_PEPI] = ok ? 1 : 0;
            group_sync();
            ok = (s_pok[0] & s_pok[1] & s_pok[2] & s_pok[3]) != 0;
            group_sync();
            if (!ok) break;
            tc_fence_after();
            const int nrb = it.nrb;
            for (int rb = 0; rb < nrb; ++rb) {
                const int rr = 128 * rb + r;
                const bool row_ok = kind == K_SP ? r < 64 : rr < it.rows;
                const int64_t grow = it.r0 + rr;
                const uint32_t taddr = tmem_base + 3u * 128u + lane_off + 64u * (uint32_t)rb;
#pragma unroll 1
                for (int ch = 0; ch < 4; ++ch) {         // (rolled: see the update park warps)
                    uint32_t a[16];
                    tmem_ld16_nowait(taddr + 16u * ch, a);
                    tmem_wait();
                    if (rb == nrb - 1 && ch == 3) {      // accumulators are in registers: the MMAs of the next item may overwrite them
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(tempty_bar(3));
                    }
                    if (!row_ok) continue;
                    if (kind == K_SP) {              // FP32 partial [a][g] of this row panel
                        float4* o = reinterpret_cast<float4*>(reinterpret_cast<float*>(it.out) + r * 64 + 16 * ch);
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            __stcg(o + e, make_float4(__uint_as_float(a[4 * e]), __uint_as_float(a[4 * e + 1]), __uint_as_float(a[4 * e + 2]), __uint_as_float(a[4 * e + 3])));
                        continue;
                    }
                    uint32_t w[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const float2 cs = __ldg(reinterpret_cast<const float2*>(it.colscale + 16 * ch) + e);
                        const __nv_bfloat162 h2 = __floats2bfloat162_rn(__uint_as_float(a[2 * e]) * cs.x, __uint_as_float(a[2 * e + 1]) * cs.y);
                        w[e] = *reinterpret_cast<const uint32_t*>(&h2);
                    }
                    uint4* o = reinterpret_cast<uint4*>(reinterpret_cast<bf16*>(it.out) + grow * 64 + 16 * ch);
                    o[0] = make_uint4(w[0], w[1], w[2], w[3]);
                    o[1] = make_uint4(w[4], w[5], w[6], w[7]);
                }
            }
            // completion: the four warps' stores happen-before the release below (CTA barrier, then a gpu-scope release by one thread)
            fence_async_global();            // these panels are read back through TMA (async proxy)
            uint32_t* done_ctr = it.done_ctr;
            const int total = it.total;
            const float* parts = it.base32;
            bf16* sea = reinterpret_cast<bf16*>(it.scale_inv);
            uint32_t* sync = it.sync;
            __syncwarp();
            if (lane == 0) mbar_arrive(piempty_bar(rslot));
            group_sync();
            if (kind == K_SP) {
                // the panel that completes the tensor's set of partials sums them in panel order (deterministic) into (S E_A)^T
                if (tid == 0) {
                    uint32_t old;
                    asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(old) : "l"(done_ctr) : "memory");
                    *s_last = old == (uint32_t)(total - 1) ? 1 : 0;
                }
                group_sync();
                if (*s_last) {
                    float acc[32];
#pragma unroll
                    for (int e = 0; e < 32; ++e) acc[e] = 0.0f;
                    for (int p = 0; p < total; ++p) {
                        const float4* src = reinterpret_cast<const float4*>(parts + (size_t)p * 4096 + tid * 32);
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            const float4 x = __ldcg(src + e);
                            acc[4 * e] += x.x; acc[4 * e + 1] += x.y; acc[4 * e + 2] += x.z; acc[4 * e + 3] += x.w;
                        }
                    }
                    const int a_ = (tid * 32) >> 6, g0 = (tid * 32) & 63;       // element (a, g0 + e) -> SEA[g0 + e][a]
#pragma unroll
                    for (int e = 0; e < 32; ++e) sea[(g0 + e) * 64 + a_] = __float2bfloat16_rn(acc[e]);
                    fence_async_global();
                    group_sync();
                    if (tid == 0) red_release_add(sync + SY_S, 1u);
                }
            } else if (done_ctr) {
                if (tid == 0) red_release_add(done_ctr, 1u);
            } else {
                if (tid == 0) mbar_arrive(plocal_bar);          // P' of this panel is in global memory: its S partial may start
            }
        }
        if (tid == 0) PROF_OUT(6)
    }
#ifdef GF8_STREAM_PROF
    if (lane == 0 && prof) prof[16384 + blockIdx.x * 32 + warp] = 9999;
#endif
    tc_fence_before();
    __syncthreads();
    if (warp == W_UMMA) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
    }
}

}  // namespace st
}  // namespace gf8
