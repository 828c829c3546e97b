// gf8_stream.cuh -- the streaming codec engine (sm_100a): ONE persistent, warp-specialised kernel per batched
// call that runs the whole whitening transform of every (tensor, rank) problem -- projections, S, Q', rank-2k
// update, tensor-wide amax, FP8 cast (a3-a6; PAPER.md:158 Eq. 14, :250 Eq. 22, Alg. 1 l.10-13) -- tensor by tensor,
// so a gradient is fetched from HBM once and every later reader finds it in L2.
//
// Low-rank form:   P'  = (Wg U_A) E_A            row panels of 256 rows        (K_PANEL_P)
//                                Q^T = Wg^T U_G                column panels of 256 columns  (K_PANEL_Q)
//                                (S E_A)^T = P'^T U_G          one item per tensor           (K_S)
//                                Q'^T = (Q^T + U_A (S E_A)^T) E_G                            (K_QP)
//                                W~  = Wg + [P' | U_G] [U_A | Q'^T]^T   128 x 128 tiles      (K_UPD)
// Work hand-out: the "pass-1" items (P, Q, S, Q') sit in one list in tensor-group order and are claimed
// dynamically (atomic counter); the update tiles are assigned statically (tile u -> CTA u mod grid) so that the
// FP32 W~ tile can stay PARKED in TMEM (3 of the 4 accumulator slots) until its tensor's amax is complete
// (release / acquire counters in global memory), and is then scaled, cast and stored without a second pass.
// A CTA's scheduler warp prefers its next update tile when that tile's tensor is ready, else claims pass-1 work,
// bounded by a lead of `lead_bytes` of gradient so the update's re-read of the gradient hits L2.
// Deadlock freedom: every wait is on work that is earlier in list / tile order and already owned by a resident
// CTA (grid <= #SMs, 1 CTA / SM); a CTA never holds more than three parked tiles of incomplete tensors, and
// host code only sends tensors with <= 3 * grid tiles here.
//
// Roles (12 warps): 0-7 epilogue, 8 scheduler (+ base-tile TMA), 9 operand TMA, 10 MMA issue, 11 grid-level sync.
#pragma once
#include "gf8_tc.cuh"

namespace gf8 {
namespace st {

using namespace gf8::tc;     // PTX wrappers (mbarrier, TMA, tcgen05)

constexpr int NS = 3;                       // operand ring stages
constexpr int STG_BYTES = 40960;            // [A 32 KB | B 8 KB]  or  [A 16 KB | B 16 KB] (update)
constexpr int NB = 3;                       // streamed base tiles in flight
constexpr int BASE_BYTES = 32768;           // 128 x 128 BF16 (two 64-column halves)
constexpr int RS = 8;                       // item ring entries
constexpr int NPARK = 3;                    // TMEM slots 0..2: update tiles (parked); slot 3: pass-1 items
constexpr int S_DATA = NS * STG_BYTES + NB * BASE_BYTES;     // 218 KB... see static_assert below
constexpr int S_MISC = 2048;
constexpr int S_BYTES = S_DATA + S_MISC;
constexpr int S_THREADS = 384;
static_assert(S_BYTES <= 227 * 1024, "shared memory budget");

enum Kind : int32_t { K_END = 0, K_PANEL_P = 1, K_PANEL_Q = 2, K_S = 3, K_QP = 4, K_UPD = 5 };
enum Mode : int32_t { M_PARK = 0, M_BLOCK = 1, M_TAP = 2 };
// words of a tensor's sync block (zeroed before every launch)
enum Sync : int32_t { SY_AMAX = 0, SY_P = 1, SY_Q = 2, SY_S = 3, SY_QP = 4, SY_TILES = 5, SY_WORDS = 8 };

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
    bf16* Pp; float* Qt; bf16* Qpt; bf16* SEA;
    const float* eA; const float* eG;
    uint8_t* codes; float* scale_inv; float* tap;
    uint32_t* sync;
    int64_t byte_pos;                      // gradient bytes of the tensors before this one (lead control)
    int64_t pad2;
};

struct P1Item { int32_t kind, tensor, r0, rows; };

// What a role needs to know about an item (shared-memory ring entry, written by the scheduler warp).
struct __align__(16) RItem {
    int32_t kind, slot, r0, c0;
    int32_t rows, cols, ksteps, mode;
    int32_t mapA0, mapA1, mapB0, mapB1;
    int32_t fmt, ld, nrb, bslot;
    int32_t total, first, n_cols_tile, out_f32;      // total: tiles of the tensor; first: this tile writes scale_inv
    void* out; const float* base32; const float* colscale; uint32_t* sync;
    float* scale_inv; uint32_t* done_ctr;
};
static_assert(sizeof(RItem) == 128, "ring entry size");

struct Parked { uint32_t* sync; float* scale_inv; uint8_t* out; int32_t ld, row0, col0, rows, cols, fmt, total, first, local, pad; };

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    return done != 0;
}
__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
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
__global__ void __launch_bounds__(S_THREADS, 1)
stream_kernel(const STensor* __restrict__ T, int nT, const P1Item* __restrict__ p1, int n_p1, int n_upd,
              const CUtensorMap* __restrict__ maps, int* ctr, int* err, long long lead_bytes, int tap) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t smem0 = smem_u32(smem_raw);
    if (smem0 & 1023u) { if (threadIdx.x == 0) atomicExch(err, 3); return; }
    const uint32_t base0 = smem0 + NS * STG_BYTES;
    const uint32_t bars = smem0 + S_DATA;
    uint8_t* misc = smem_raw + S_DATA;
    auto full_bar = [&](uint32_t s) { return bars + 8u * s; };
    auto empty_bar = [&](uint32_t s) { return bars + 8u * (3 + s); };
    auto bfull_bar = [&](uint32_t s) { return bars + 8u * (6 + s); };
    auto bempty_bar = [&](uint32_t s) { return bars + 8u * (9 + s); };
    auto tfull_bar = [&](uint32_t s) { return bars + 8u * (12 + s); };
    auto tempty_bar = [&](uint32_t s) { return bars + 8u * (16 + s); };
    auto ifull_bar = [&](uint32_t s) { return bars + 8u * (20 + s); };
    auto iempty_bar = [&](uint32_t s) { return bars + 8u * (28 + s); };
    auto parked_bar = [&](uint32_t s) { return bars + 8u * (36 + s); };
    auto sready_bar = [&](uint32_t s) { return bars + 8u * (39 + s); };
    const uint32_t pdone_bar = bars + 8u * 42, drain_bar = bars + 8u * 43;
    uint32_t* s_tmem = reinterpret_cast<uint32_t*>(misc + 352);
    float* s_scale = reinterpret_cast<float*>(misc + 368);
    uint32_t* s_wmax = reinterpret_cast<uint32_t*>(misc + 384);          // [3][8]
    volatile int* s_nupd = reinterpret_cast<volatile int*>(misc + 480);  // parked tiles of this CTA (-1: not known yet)
    Parked* s_park = reinterpret_cast<Parked*>(misc + 512);              // [3]
    RItem* s_items = reinterpret_cast<RItem*>(misc + 768);               // [RS]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int s = 0; s < NB; ++s) { mbar_init(bfull_bar(s), 1); mbar_init(bempty_bar(s), 8); }
        for (int s = 0; s < 4; ++s) { mbar_init(tfull_bar(s), 1); mbar_init(tempty_bar(s), 8); }
        for (int s = 0; s < RS; ++s) { mbar_init(ifull_bar(s), 1); mbar_init(iempty_bar(s), 10); }
        for (int s = 0; s < NPARK; ++s) { mbar_init(parked_bar(s), 8); mbar_init(sready_bar(s), 1); }
        mbar_init(pdone_bar, 8); mbar_init(drain_bar, 1);
        *s_nupd = -1;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 10) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tmem)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(s_tmem);
    auto errset = [&]() { return *reinterpret_cast<volatile int*>(err) != 0; };

    if (warp == 8) {
        // ===== scheduler (lane 0): chooses this CTA's next item, writes it into the ring, streams update base tiles =====
        if (lane == 0) {
            uint32_t nring = 0, q = 0;
            int u = blockIdx.x, tu = 0;
            int old0 = -1, old1 = -1, old2 = -1;          // tensors of the update tiles q-3, q-2, q-1 (-1: nothing to wait for)
            int n_parked = 0;
            bool ok = true;
            auto push = [&](const RItem& it) -> bool {
                const uint32_t slot = nring % RS, ph = (nring / RS) & 1u;
                if (!mbar_wait(iempty_bar(slot), ph ^ 1u, err)) return false;
                const uint4* src = reinterpret_cast<const uint4*>(&it);
                uint4* dst = reinterpret_cast<uint4*>(s_items + slot);
#pragma unroll
                for (int w = 0; w < 8; ++w) dst[w] = src[w];
                mbar_arrive(ifull_bar(slot));             // (release: the entry is visible to whoever acquires the barrier)
                ++nring;
                return true;
            };
            auto wait_ge = [&](const uint32_t* p, uint32_t target) -> bool {
                for (uint32_t spin = 0; ld_acquire(p) < target; ++spin) {
                    if (spin > (1u << 22) || ((spin & 255u) == 255u && errset())) { atomicExch(err, 4); return false; }
                    __nanosleep(64);
                }
                return true;
            };
            while (ok) {
                while (tu < nT && u >= T[tu].upd_start + T[tu].n_tiles) ++tu;
                const bool have_upd = u < n_upd && tu < nT;
                bool can = false;
                if (have_upd) {
                    const STensor& t = T[tu];
                    can = t.dep_target == 0 || ld_acquire(t.sync + t.dep_idx) >= (uint32_t)t.dep_target;
                    if (can && old0 >= 0) { const STensor& o = T[old0]; can = ld_acquire(o.sync + SY_TILES) >= (uint32_t)o.n_tiles; }
                }
                if (can) {
                    const STensor& t = T[tu];
                    const int tile = u - t.upd_start, ti = tile / t.tiles_n, tj = tile % t.tiles_n;
                    RItem it;
                    it.kind = K_UPD; it.slot = (int)(q % NPARK); it.r0 = ti * 128; it.c0 = tj * 128;
                    it.rows = min(128, t.m - it.r0); it.cols = min(128, t.n - it.c0);
                    it.ksteps = (t.useA ? 1 : 0) + (t.useG ? 1 : 0); it.mode = t.mode;
                    it.mapA0 = t.useA ? t.map_Pp128 : t.map_UG128; it.mapB0 = t.useA ? t.map_UA128 : t.map_Qpt128;
                    it.mapA1 = t.map_UG128; it.mapB1 = t.map_Qpt128;
                    it.fmt = t.fmt; it.ld = t.n; it.nrb = 1; it.bslot = (int)(q % NB);
                    it.total = t.n_tiles; it.first = tile == 0 ? 1 : 0; it.n_cols_tile = 128; it.out_f32 = 0;
                    it.out = t.mode == M_TAP ? (void*)t.tap : (void*)t.codes; it.base32 = nullptr; it.colscale = nullptr; it.sync = t.sync;
                    it.scale_inv = t.mode == M_BLOCK ? t.scale_inv + (size_t)ti * t.tiles_n + tj : t.scale_inv;
                    it.done_ctr = nullptr;
                    if (!(ok = push(it))) break;
                    // base tile: 128 rows x 128 columns of the gradient (two 64-column halves) in one 3-D box
                    const uint32_t bs = q % NB, bph = (q / NB) & 1u;
                    if (!(ok = mbar_wait(bempty_bar(bs), bph ^ 1u, err))) break;
                    const CUtensorMap* mp = maps + t.map_src_b;
                    tmap_acquire(mp);
                    mbar_expect_tx(bfull_bar(bs), BASE_BYTES);
                    tma_load_3d(base0 + bs * BASE_BYTES, mp, 0, it.r0, tj * 2, bfull_bar(bs));
                    old0 = old1; old1 = old2; old2 = t.mode == M_PARK ? tu : -1;
                    if (t.mode != M_TAP) ++n_parked;
                    u += (int)gridDim.x; ++q;
                    continue;
                }
                int c = *reinterpret_cast<volatile int*>(ctr);
                if (c < n_p1) {
                    const P1Item pk = p1[c];
                    const bool panel = pk.kind == K_PANEL_P || pk.kind == K_PANEL_Q;
                    if (!panel || !have_upd || T[pk.tensor].byte_pos - T[tu].byte_pos <= lead_bytes) {
                        c = atomicAdd(ctr, 1);
                        if (c < n_p1) {
                            const P1Item pi = p1[c];
                            const STensor& t = T[pi.tensor];
                            RItem it;
                            it.kind = pi.kind; it.slot = 3; it.r0 = pi.r0; it.c0 = 0; it.rows = pi.rows; it.cols = 64; it.mode = 0;
                            it.mapA1 = it.mapB1 = -1; it.fmt = 0; it.ld = 64; it.nrb = pi.rows > 128 ? 2 : 1; it.bslot = 0;
                            it.total = it.first = 0; it.n_cols_tile = 64; it.out_f32 = 0; it.base32 = nullptr; it.colscale = nullptr;
                            it.sync = t.sync; it.scale_inv = nullptr;
                            if (pi.kind == K_PANEL_P) {
                                it.ksteps = (t.n + 63) / 64; it.mapA0 = t.map_src_p; it.mapB0 = t.map_UAt;
                                it.out = t.Pp; it.colscale = t.eA; it.done_ctr = t.sync + SY_P;
                            } else if (pi.kind == K_PANEL_Q) {
                                it.ksteps = (t.m + 63) / 64; it.mapA0 = t.map_src_q; it.mapB0 = t.map_UGt;
                                if (t.useA) { it.out = t.Qt; it.out_f32 = 1; } else { it.out = t.Qpt; it.colscale = t.eG; }
                                it.done_ctr = t.sync + SY_Q;
                            } else if (pi.kind == K_S) {
                                it.ksteps = (t.m + 63) / 64; it.mapA0 = t.map_Pp64; it.mapB0 = t.map_UGt;
                                it.out = t.SEA; it.done_ctr = t.sync + SY_S; it.nrb = 1;
                                if (!(ok = wait_ge(t.sync + SY_P, (uint32_t)t.nP))) break;
                            } else {   // K_QP
                                it.ksteps = 1; it.mapA0 = t.map_UA256; it.mapB0 = t.map_SEA;
                                it.out = t.Qpt; it.base32 = t.Qt; it.colscale = t.eG; it.done_ctr = t.sync + SY_QP;
                                if (!(ok = wait_ge(t.sync + SY_S, 1u) && wait_ge(t.sync + SY_Q, (uint32_t)t.nQ))) break;
                            }
                            if (!(ok = push(it))) break;
                            continue;
                        }
                    }
                }
                if (!have_upd && c >= n_p1) break;
                if (errset()) { ok = false; break; }
                __nanosleep(200);
            }
            *s_nupd = n_parked;
            RItem e;
            e.kind = K_END;
            push(e);
        }
    } else if (warp == 9) {
        // ===== operand loader (converged warp, one elected lane issues the TMA loads) =====
        uint32_t stage = 0, phase = 0;
        bool ok = true;
        for (uint32_t nr = 0; ok; ++nr) {
            const uint32_t slot = nr % RS;
            if (!(ok = mbar_wait(ifull_bar(slot), (nr / RS) & 1u, err))) break;
            const RItem& it = s_items[slot];
            const int kind = it.kind;
            if (kind == K_END) break;
            const int ksteps = it.ksteps, r0 = it.r0, c0 = it.c0;
            const CUtensorMap* mA0 = maps + it.mapA0; const CUtensorMap* mB0 = maps + it.mapB0;
            const CUtensorMap* mA1 = maps + (it.mapA1 >= 0 ? it.mapA1 : it.mapA0);
            const CUtensorMap* mB1 = maps + (it.mapB1 >= 0 ? it.mapB1 : it.mapB0);
            __syncwarp();
            if (elect_one()) {
                mbar_arrive(iempty_bar(slot));
                tmap_acquire(mA0); tmap_acquire(mB0);
                if (kind == K_UPD && ksteps > 1) { tmap_acquire(mA1); tmap_acquire(mB1); }
                fence_async_global();      // P', Q'^T, (S E_A)^T were written by other CTAs through the generic proxy
            }
            __syncwarp();
            for (int t = 0; t < ksteps && ok; ++t) {
                if (!(ok = mbar_wait(empty_bar(stage), phase ^ 1u, err))) break;
                const uint32_t sa = smem0 + stage * STG_BYTES, fb = full_bar(stage);
                if (elect_one()) {
                    if (kind == K_PANEL_P) {
                        mbar_expect_tx(fb, 40960u);
                        tma_load_2d(sa, mA0, 64 * t, r0, fb);
                        tma_load_2d(sa + 32768u, mB0, 64 * t, 0, fb);
                    } else if (kind == K_PANEL_Q) {
                        mbar_expect_tx(fb, 40960u);
                        tma_load_3d(sa, mA0, 0, 64 * t, r0 >> 6, fb);
                        tma_load_2d(sa + 32768u, mB0, 64 * t, 0, fb);
                    } else if (kind == K_S) {
                        mbar_expect_tx(fb, 16384u);
                        tma_load_2d(sa, mA0, 0, 64 * t, fb);
                        tma_load_2d(sa + 32768u, mB0, 64 * t, 0, fb);
                    } else if (kind == K_QP) {
                        mbar_expect_tx(fb, 40960u);
                        tma_load_2d(sa, mA0, 0, r0, fb);
                        tma_load_2d(sa + 32768u, mB0, 0, 0, fb);
                    } else {   // K_UPD
                        mbar_expect_tx(fb, 32768u);
                        tma_load_2d(sa, t ? mA1 : mA0, 0, r0, fb);
                        tma_load_2d(sa + 16384u, t ? mB1 : mB0, 0, c0, fb);
                    }
                }
                __syncwarp();
                if (++stage == NS) { stage = 0; phase ^= 1u; }
            }
        }
    } else if (warp == 10) {
        // ===== MMA issuer (converged warp, one elected lane issues) =====
        uint32_t stage = 0, phase = 0, use0 = 0, use1 = 0, use2 = 0, use3 = 0;
        bool ok = true;
        for (uint32_t nr = 0; ok; ++nr) {
            const uint32_t rslot = nr % RS;
            if (!(ok = mbar_wait(ifull_bar(rslot), (nr / RS) & 1u, err))) break;
            const RItem& it = s_items[rslot];
            const int kind = it.kind;
            if (kind == K_END) break;
            const int ksteps = it.ksteps, nrb = it.nrb;
            const uint32_t slot = (uint32_t)it.slot;
            __syncwarp();
            if (elect_one()) mbar_arrive(iempty_bar(rslot));
            const bool upd = kind == K_UPD, a_mn = kind == K_PANEL_Q || kind == K_S;
            const uint32_t idesc = instr_desc(upd ? 128 : 64, a_mn ? 1 : 0, 0);
            const uint32_t b_off = upd ? 16384u : 32768u;
            const uint32_t uses = slot == 0 ? use0 : (slot == 1 ? use1 : (slot == 2 ? use2 : use3));
            if (slot == 0) ++use0; else if (slot == 1) ++use1; else if (slot == 2) ++use2; else ++use3;
            if (!(ok = mbar_wait(tempty_bar(slot), (uses & 1u) ^ 1u, err))) break;
            tc_fence_after();
            const uint32_t d = tmem_base + slot * 128u;
            for (int t = 0; t < ksteps && ok; ++t) {
                if (!(ok = mbar_wait(full_bar(stage), phase, err))) break;
                tc_fence_after();
                const uint32_t sa = smem0 + stage * STG_BYTES, sb = sa + b_off;
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
                    tc_commit(empty_bar(stage));
                }
                __syncwarp();
                if (++stage == NS) { stage = 0; phase ^= 1u; }
            }
            if (ok && elect_one()) tc_commit(tfull_bar(slot));
            __syncwarp();
        }
        if (ok) {      // drain: no commit of this issuer may still be in flight when the CTA exits
            if (elect_one()) tc_commit(drain_bar);
            __syncwarp();
            mbar_wait(drain_bar, 0u, err);
        }
    }
    else if (warp == 11) {
        // ===== grid-level sync (lanes 0..2, one per parking slot): tile parked -> tensor counter; tensor complete -> scale =====
        if (lane < NPARK) {
            for (uint32_t k = 0;; ++k) {
                bool stop = false;
                for (uint32_t spin = 0; !mbar_test(parked_bar(lane), k & 1u); ++spin) {
                    const int tot = *s_nupd;
                    if ((tot >= 0 && (int)(k * NPARK + lane) >= tot) || ((spin & 1023u) == 1023u && errset())) { stop = true; break; }
                    __nanosleep(64);
                }
                if (stop) break;
                const Parked pk = s_park[lane];
                uint32_t mx = 0;
#pragma unroll
                for (int w = 0; w < 8; ++w) mx = max(mx, s_wmax[lane * 8 + w]);
                float scale, si;
                const float fmax = pk.fmt == 0 ? 448.0f : 57344.0f;
                if (pk.local) {
                    scales_from_amax(mx, fmax, scale, si);
                    *pk.scale_inv = si;
                } else {
                    if (mx) atomicMax(pk.sync + SY_AMAX, mx);
                    red_release_add(pk.sync + SY_TILES, 1u);
                    bool bad = false;
                    for (uint32_t spin = 0; ld_acquire(pk.sync + SY_TILES) < (uint32_t)pk.total; ++spin) {
                        if (spin > (1u << 22) || ((spin & 255u) == 255u && errset())) { bad = true; break; }
                        __nanosleep(64);
                    }
                    if (bad) { atomicExch(err, 2); break; }
                    scales_from_amax(*reinterpret_cast<volatile uint32_t*>(pk.sync + SY_AMAX), fmax, scale, si);
                    if (pk.first) *pk.scale_inv = si;
                }
                s_scale[lane] = scale;
                mbar_arrive(sready_bar(lane));
            }
        }
    } else {
        // ===== epilogue warps 0..7: each warp follows the item ring on its own (no block-level barrier) =====
        const int q4 = warp & 3, half = warp >> 2;
        const int r = q4 * 32 + lane;                           // accumulator row (TMEM lane) of this thread
        const uint32_t lane_off = (uint32_t)(q4 * 32) << 16;
        uint32_t nr = 0, nq = 0, ncast = 0, use3 = 0, idle = 0;
        bool have = false, done = false, ok = true;
        auto test = [&](uint32_t bar, uint32_t par) -> bool {
            uint32_t v = 0;
            if (lane == 0) v = mbar_test(bar, par) ? 1u : 0u;
            return __shfl_sync(0xFFFFFFFFu, v, 0) != 0;
        };
        while (ok) {
            // (1) the oldest parked tile whose scale has arrived: scale, cast, store, free its TMEM slot
            if (ncast < nq && test(sready_bar(ncast % NPARK), (ncast / NPARK) & 1u)) {
                const uint32_t slot = ncast % NPARK;
                const Parked pk = s_park[slot];
                const float scale = s_scale[slot];
                const uint32_t taddr = tmem_base + slot * 128u + lane_off + (uint32_t)half * 64u;
                const bool row_ok = r < pk.rows;
                uint8_t* orow = pk.out + (int64_t)(pk.row0 + r) * pk.ld + pk.col0 + 64 * half;
#pragma unroll
                for (int g = 0; g < 2; ++g) {
                    uint32_t a[32];
                    tmem_ld32_nowait(taddr + 32u * g, a);
                    tmem_wait();
                    uint4 cd[2];
                    uint32_t* cw = reinterpret_cast<uint32_t*>(cd);
                    if (pk.fmt == 0) {
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            cw[j] = cast4<0>(__uint_as_float(a[4 * j]), __uint_as_float(a[4 * j + 1]), __uint_as_float(a[4 * j + 2]), __uint_as_float(a[4 * j + 3]), scale);
                    } else {
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            cw[j] = cast4<1>(__uint_as_float(a[4 * j]), __uint_as_float(a[4 * j + 1]), __uint_as_float(a[4 * j + 2]), __uint_as_float(a[4 * j + 3]), scale);
                    }
                    if (row_ok) {
#pragma unroll
                        for (int h = 0; h < 2; ++h)
                            if (64 * half + 32 * g + 16 * h < pk.cols) *reinterpret_cast<uint4*>(orow + 32 * g + 16 * h) = cd[h];
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty_bar(slot));
                ++ncast; idle = 0;
                continue;
            }
            if (!done) {
                const uint32_t rslot = nr % RS;
                if (!have && test(ifull_bar(rslot), (nr / RS) & 1u)) {
                    have = true;
                    if (s_items[rslot].kind == K_END) { done = true; have = false; }
                }
                if (have) {
                    const RItem& it = s_items[rslot];
                    const int kind = it.kind;
                    const uint32_t slot = (uint32_t)it.slot;
                    const bool upd = kind == K_UPD;
                    const uint32_t tpar = upd ? (nq / NPARK) & 1u : use3 & 1u;
                    if (test(tfull_bar(slot), tpar) && (!upd || test(bfull_bar(nq % NB), (nq / NB) & 1u))) {
                        tc_fence_after();
                        if (upd) {
                            const uint32_t bs = nq % NB;
                            const uint32_t taddr = tmem_base + slot * 128u + lane_off + (uint32_t)half * 64u;
                            const uint32_t brow = base0 + bs * BASE_BYTES + (uint32_t)half * 16384u + (uint32_t)r * 128u;
                            const int mode = it.mode;
                            float mx = 0.0f;
                            float* trow = mode == M_TAP ? reinterpret_cast<float*>(it.out) + (int64_t)(it.r0 + r) * it.ld + it.c0 + 64 * half : nullptr;
#pragma unroll
                            for (int g = 0; g < 2; ++g) {
                                uint32_t a[32];
                                tmem_ld32_nowait(taddr + 32u * g, a);
                                uint4 b[4];
#pragma unroll
                                for (int j = 0; j < 4; ++j) b[j] = lds128(brow + (((uint32_t)(4 * g + j) ^ (uint32_t)(r & 7)) << 4));
                                tmem_wait();
                                float v[32];
#pragma unroll
                                for (int j = 0; j < 4; ++j) {
                                    const uint32_t w[4] = {b[j].x, b[j].y, b[j].z, b[j].w};
#pragma unroll
                                    for (int e = 0; e < 4; ++e)
                                        add_bf16x2(w[e], __uint_as_float(a[8 * j + 2 * e]), __uint_as_float(a[8 * j + 2 * e + 1]), v[8 * j + 2 * e], v[8 * j + 2 * e + 1]);
                                }
                                if (mode == M_TAP) {
                                    if (r < it.rows) {
#pragma unroll
                                        for (int h = 0; h < 8; ++h)
                                            if (64 * half + 32 * g + 4 * h < it.cols)
                                                *reinterpret_cast<float4*>(trow + 32 * g + 4 * h) = make_float4(v[4 * h], v[4 * h + 1], v[4 * h + 2], v[4 * h + 3]);
                                    }
                                } else {
#pragma unroll
                                    for (int e = 0; e < 16; ++e) mx = max3abs(mx, v[2 * e], v[2 * e + 1]);
                                    uint32_t wv[32];
#pragma unroll
                                    for (int e = 0; e < 32; ++e) wv[e] = __float_as_uint(v[e]);
                                    tmem_st32(taddr + 32u * g, wv);
                                }
                            }
                            if (mode == M_TAP) {
                                tc_fence_before();
                                __syncwarp();
                                if (lane == 0) { mbar_arrive(tempty_bar(slot)); mbar_arrive(bempty_bar(bs)); }
                                ++ncast;                     // nothing parked: the tile is finished
                            } else {
                                tmem_wait_st();
                                const uint32_t wm = warp_max_u32(__float_as_uint(mx));     // (non-negative floats and NaN order as integers)
                                if (lane == 0) s_wmax[slot * 8 + warp] = wm;
                                if (threadIdx.x == 0) {
                                    Parked pk;
                                    pk.sync = it.sync; pk.scale_inv = it.scale_inv; pk.out = reinterpret_cast<uint8_t*>(it.out);
                                    pk.ld = it.ld; pk.row0 = it.r0; pk.col0 = it.c0; pk.rows = it.rows; pk.cols = it.cols; pk.fmt = it.fmt;
                                    pk.total = it.total; pk.first = it.first; pk.local = mode == M_BLOCK ? 1 : 0; pk.pad = 0;
                                    s_park[slot] = pk;
                                }
                                tc_fence_before();
                                __syncwarp();
                                if (lane == 0) { mbar_arrive(parked_bar(slot)); mbar_arrive(bempty_bar(bs)); }
                            }
                            ++nq;
                        } else {
                            // pass-1 item: a panel of up to 256 rows x 64 columns (row block = warp >> 2), straight to global memory
                            const int rb = half, rr = 128 * rb + r;
                            const bool row_ok = rb < it.nrb && rr < it.rows && (kind != K_S || r < 64);
                            const int64_t grow = it.r0 + rr;
                            const uint32_t taddr = tmem_base + 3u * 128u + lane_off + 64u * (uint32_t)rb;
                            if (rb < it.nrb) {
#pragma unroll 1
                                for (int c0 = 0; c0 < 64; c0 += 16) {
                                    uint32_t a[16];
                                    tmem_ld16(taddr + c0, a);
                                    if (!row_ok) continue;
                                    float v[16];
#pragma unroll
                                    for (int e = 0; e < 16; ++e) v[e] = __uint_as_float(a[e]);
                                    if (kind == K_S) {
                                        bf16* o = reinterpret_cast<bf16*>(it.out);
#pragma unroll
                                        for (int e = 0; e < 16; ++e) o[(int64_t)(c0 + e) * 64 + r] = __float2bfloat16_rn(v[e]);
                                        continue;
                                    }
                                    if (it.base32) {
                                        const float4* bp = reinterpret_cast<const float4*>(it.base32 + grow * 64 + c0);
#pragma unroll
                                        for (int e = 0; e < 4; ++e) {
                                            const float4 x = __ldcg(bp + e);
                                            v[4 * e] += x.x; v[4 * e + 1] += x.y; v[4 * e + 2] += x.z; v[4 * e + 3] += x.w;
                                        }
                                    }
                                    if (it.colscale) {
#pragma unroll
                                        for (int e = 0; e < 16; ++e) v[e] *= __ldg(it.colscale + c0 + e);
                                    }
                                    if (it.out_f32) {
                                        float4* o = reinterpret_cast<float4*>(reinterpret_cast<float*>(it.out) + grow * 64 + c0);
#pragma unroll
                                        for (int e = 0; e < 4; ++e) o[e] = make_float4(v[4 * e], v[4 * e + 1], v[4 * e + 2], v[4 * e + 3]);
                                    } else {
                                        uint32_t w[8];
#pragma unroll
                                        for (int e = 0; e < 8; ++e) {
                                            const __nv_bfloat162 h2 = __floats2bfloat162_rn(v[2 * e], v[2 * e + 1]);
                                            w[e] = *reinterpret_cast<const uint32_t*>(&h2);
                                        }
                                        uint4* o = reinterpret_cast<uint4*>(reinterpret_cast<bf16*>(it.out) + grow * 64 + c0);
                                        o[0] = make_uint4(w[0], w[1], w[2], w[3]);
                                        o[1] = make_uint4(w[4], w[5], w[6], w[7]);
                                    }
                                }
                            }
                            fence_async_global();            // these panels are read back through TMA (async proxy) by other CTAs
                            tc_fence_before();
                            __syncwarp();
                            if (lane == 0) { mbar_arrive(tempty_bar(3)); mbar_arrive(pdone_bar); }
                            if (warp == 0) {                 // all eight warps' stores happen-before this release
                                ok = mbar_wait(pdone_bar, use3 & 1u, err);
                                if (lane == 0) red_release_add(it.done_ctr, 1u);
                            }
                            ++use3;
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(iempty_bar(rslot));
                        ++nr; have = false; idle = 0;
                        continue;
                    }
                }
            } else if (ncast == nq) break;
            if (++idle > (1u << 24)) { if (lane == 0) atomicExch(err, 5); break; }
            if ((idle & 4095u) == 4095u && errset()) break;
            __nanosleep(20);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 10) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
    }
}

}  // namespace st
}  // namespace gf8
