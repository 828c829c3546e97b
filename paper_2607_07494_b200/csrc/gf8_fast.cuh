// gf8_fast.cuh -- host side of the FAST (tensor-core) path: TMA maps, per-slot scratch, cached launch
// plans, and the stage sequence that turns encode / reduce_decoded / whiten into lists of tc::Item.
// Included by gf8_api.cu after gf8_ctx.cuh.  Arithmetic lives in gf8_tc.cuh; nothing here computes.
#pragma once
#include <algorithm>

#include "gf8_ctx.cuh"
#include "gf8_tc.cuh"

// A cached launch plan: everything a batched call needs on the device, built on first use of a given
// argument list (steady-state training calls repeat the same pointers every step).
struct Plan {
    CUtensorMap* d_maps = nullptr;
    gf8::tc::Item* d_items = nullptr;
    // stages: 0 P' and Q^T, 1 S, 2 Q'^T, 3 update tiles (amax / block cast / store), 4 update tiles (cast),
    //         5 update strips (amax / block cast), 6 update strips (cast), 7 fused update (opt-in)
    int stage_off[8] = {0, 0, 0, 0, 0, 0, 0, 0}, stage_cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int stage_wide[8] = {0, 0, 0, 0, 0, 0, 0, 0};  // the stage holds 256-row panel items: wide operand stages (kmode 3)
    int stage_base[8] = {0, 0, 0, 0, 0, 0, 0, 0};  // streamed base tiles per item in that stage's launch (0, 1 or 2)
    bool ef = false;                     // f1: the update stages run the error-feedback instance of the kernel
    bool pair5 = false;                  // stage 5 holds (amax item, cast item) pairs: one launch for both update passes (kmode 6)
    int runs = 0;                        // launches so far: the first one acquires its tensor maps with proxy fences
    int* d_ctr = nullptr;                // one item counter per stage (dynamic item hand-out), zeroed before every run
    uint32_t* d_amax = nullptr;          // one word per TC problem (per-tensor scaling)
    size_t n_amax = 0;
    size_t n_plain_amax = 0;             // amax words of the grouped Euclidean encode, after the n_amax words
    std::vector<int> grouped;            // plain problems taken by the grouped Euclidean encode (BF16, per-tensor scale)
    struct Convert { const float* src; gf8::bf16 *dst, *dst_lo; int64_t numel; };
    std::vector<Convert> converts;       // FP32 gradient -> BF16 MMA operand copies
    std::vector<int> plain;              // batch indices served by the per-problem (non-TC) path
    struct Reduce { int batch_index; float* uhat; gf8::bf16 *u16, *u16_lo; };
    std::vector<Reduce> reduces;         // decode: payload reduction into the slot before the stages
};

namespace {

using gf8::bf16;
using gf8::tc::Item;

constexpr int FAST_MAX_KP = 512;   // GF8_MAX_RANK: panels are cut into 128-column accumulator chunks
constexpr size_t FAST_MAX_PLANS = 64;

inline int pad64(int k) { return (k + 63) / 64 * 64; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

gf8_status fast_init(gf8_ctx* c) {
    if (c->encode_tiled) return GF8_OK;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    CU_TRY(c, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
    if (!fn || q != cudaDriverEntryPointSuccess) return fail(c, GF8_ERR_CUDA, "cuTensorMapEncodeTiled not available");
    c->encode_tiled = fn;
    GF_TRY(dmalloc(c, &c->d_err, 4));
    GF_TRY(dmalloc(c, &c->d_prof, (size_t)32768));
    CU_TRY(c, cudaMemset(c->d_err, 0, 4 * sizeof(int)));
    CU_TRY(c, cudaFuncSetAttribute(gf8::tc::tc_items_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   gf8::tc::SMEM_BYTES));
    CU_TRY(c, cudaFuncSetAttribute(gf8::tc::tc_items_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   gf8::tc::SMEM_BYTES));
    return GF8_OK;
}

// BF16 row-major matrix [rows][cols] (leading dimension ld elements) -> TMA map, 64 x 64 boxes, 128 B swizzle,
// out-of-bounds elements read as zero.
gf8_status make_map1(gf8_ctx* c, CUtensorMap* out, const void* ptr, uint64_t rows, uint64_t cols, uint64_t ld, uint32_t box_rows) {
    const cuuint64_t gdim[2] = {cols, rows};
    const cuuint64_t gstride[1] = {ld * 2};
    const cuuint32_t box[2] = {64, box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = ((EncodeTiledFn)c->encode_tiled)(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), gdim,
                                                        gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                        CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(c, GF8_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d) for %llu x %llu", (int)r,
                                       (unsigned long long)rows, (unsigned long long)cols);
    return GF8_OK;
}

// Both box heights of a BF16 matrix: out[0] = 64-row boxes, out[1] = 128-row boxes.
gf8_status make_map(gf8_ctx* c, CUtensorMap* out, const void* ptr, uint64_t rows, uint64_t cols, uint64_t ld) {
    GF_TRY(make_map1(c, &out[0], ptr, rows, cols, ld, 64));
    return make_map1(c, &out[1], ptr, rows, cols, ld, 128);
}

// FP8 code matrix [rows][cols] bytes -> TMA store map, 128 x 128 boxes (one update tile), 128 B swizzle.
gf8_status make_map_u8(gf8_ctx* c, CUtensorMap* out, const void* ptr, uint64_t rows, uint64_t cols, bool per_warp = false) {
    const cuuint64_t gdim[2] = {cols, rows};
    const cuuint64_t gstride[1] = {cols};
    // per_warp: 64 x 32 boxes, no swizzle (one epilogue warp's sub-tile); else 128 x 128 boxes, 128 B swizzle
    const cuuint32_t box[2] = {per_warp ? 64u : 128u, per_warp ? 32u : 128u};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = ((EncodeTiledFn)c->encode_tiled)(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(ptr), gdim,
                                                        gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                        per_warp ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(c, GF8_ERR_CUDA, "cuTensorMapEncodeTiled (u8) failed (%d) for %llu x %llu", (int)r,
                                       (unsigned long long)rows, (unsigned long long)cols);
    return GF8_OK;
}

// U (d x k FP32) -> U16 (d x kp BF16, zero-padded) and its transpose Ut16 (kp x d).
__global__ void pack_basis_kernel(const float* __restrict__ U, int d, int k, int kp, bf16* __restrict__ U16,
                                  bf16* __restrict__ Ut16, bf16* __restrict__ U16_lo, bf16* __restrict__ Ut16_lo) {
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < (int64_t)d * kp;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(idx / kp), col = (int)(idx % kp);
        const float x = col < k ? U[(int64_t)i * k + col] : 0.0f;
        const bf16 v = __float2bfloat16_rn(x);
        const bf16 lo = __float2bfloat16_rn(x - __bfloat162float(v));
        U16[idx] = v;
        Ut16[(int64_t)col * d + i] = v;
        U16_lo[idx] = lo;
        Ut16_lo[(int64_t)col * d + i] = lo;
    }
}

gf8_status fast_pack_basis(gf8_ctx* c, cudaStream_t st, SideState& s) {
    if (!s.U16) return GF8_OK;
    pack_basis_kernel<<<grid_for(c, (int64_t)s.d * s.kp, 256, 4), 256, 0, st>>>(s.U, s.d, s.k, s.kp, s.U16, s.Ut16,
                                                                                s.U16_lo, s.Ut16_lo);
    LAUNCH_CHECK(c);
    return GF8_OK;
}

// Called from gf8_create for every layer: decides eligibility and allocates the BF16 basis copies.
gf8_status fast_init_layer(gf8_ctx* c, LayerState& L) {
    L.tc_ok = false;
    if ((c->precision != GF8_PREC_FAST && !c->tc_exact) || L.desc.side == GF8_SIDE_NONE) return GF8_OK;
    if (L.desc.d_out < 64 || L.desc.d_in < 64) return GF8_OK;
    if ((L.in.used && pad64(L.in.k) > FAST_MAX_KP) || (L.out.used && pad64(L.out.k) > FAST_MAX_KP)) return GF8_OK;
    GF_TRY(fast_init(c));
    for (SideState* s : {&L.in, &L.out}) {
        if (!s->used) continue;
        GF_TRY(dmalloc(c, &s->U16, (size_t)s->d * s->kp));
        GF_TRY(dmalloc(c, &s->Ut16, (size_t)s->kp * s->d));
        GF_TRY(make_map(c, s->map_U16, s->U16, s->d, s->kp, s->kp));
        GF_TRY(make_map(c, s->map_Ut16, s->Ut16, s->kp, s->d, s->d));
        GF_TRY(dmalloc(c, &s->U16_lo, (size_t)s->d * s->kp));
        GF_TRY(dmalloc(c, &s->Ut16_lo, (size_t)s->kp * s->d));
        GF_TRY(make_map(c, s->map_U16_lo, s->U16_lo, s->d, s->kp, s->kp));
        GF_TRY(make_map(c, s->map_Ut16_lo, s->Ut16_lo, s->kp, s->d, s->d));
    }
    L.tc_ok = true;
    return GF8_OK;
}

gf8_status fast_slot(gf8_ctx* c, LayerState& L, size_t idx, bool need_src16, bool need_uhat, bool need_split,
                     Slot** out) {
    while (L.slots.size() <= idx) L.slots.push_back(nullptr);
    const size_t m = L.desc.d_out, n = L.desc.d_in;
    const size_t kpA = L.in.used ? L.in.kp : 0, kpG = L.out.used ? L.out.kp : 0;
    if (!L.slots[idx]) {
        Slot* s = new (std::nothrow) Slot();
        if (!s) return fail(c, GF8_ERR_NOMEM, "host allocation failed");
        // the slot is published only once every buffer and map exists: a failed attempt leaves no half-built slot behind
        // (its device buffers stay on the context's allocation list and are released by gf8_destroy)
        auto init = [&]() -> gf8_status {
            if (kpA) {
                GF_TRY(dmalloc(c, &s->Pp, m * kpA));
                GF_TRY(make_map(c, s->map_Pp, s->Pp, m, kpA, kpA));
            }
            if (kpG) {
                GF_TRY(dmalloc(c, &s->Qt, n * kpG));
                GF_TRY(dmalloc(c, &s->Qpt, n * kpG));
                GF_TRY(make_map(c, s->map_Qpt, s->Qpt, n, kpG, kpG));
            }
            if (kpA && kpG) {
                GF_TRY(dmalloc(c, &s->SEA, kpG * kpA));
                GF_TRY(make_map(c, s->map_SEA, s->SEA, kpG, kpA, kpA));
            }
            return GF8_OK;
        };
        const gf8_status st = init();
        if (st != GF8_OK) { delete s; return st; }
        L.slots[idx] = s;
    }
    Slot* s = L.slots[idx];
    if (need_src16 && !s->src16) {
        GF_TRY(dmalloc(c, &s->src16, m * n));
        GF_TRY(make_map(c, s->map_src16, s->src16, m, n, n));
    }
    if (need_uhat && !s->Uhat) GF_TRY(dmalloc(c, &s->Uhat, m * n));
    if (need_split && !s->src16_lo) {
        GF_TRY(dmalloc(c, &s->src16_lo, m * n));
        GF_TRY(make_map(c, s->map_src16_lo, s->src16_lo, m, n, n));
        if (kpA) {
            GF_TRY(dmalloc(c, &s->Pp_lo, m * kpA));
            GF_TRY(make_map(c, s->map_Pp_lo, s->Pp_lo, m, kpA, kpA));
        }
        if (kpG) {
            GF_TRY(dmalloc(c, &s->Qpt_lo, n * kpG));
            GF_TRY(make_map(c, s->map_Qpt_lo, s->Qpt_lo, n, kpG, kpG));
        }
        if (kpA && kpG) {
            GF_TRY(dmalloc(c, &s->SEA_lo, kpG * kpA));
            GF_TRY(make_map(c, s->map_SEA_lo, s->SEA_lo, kpG, kpA, kpA));
        }
    }
    *out = s;
    return GF8_OK;
}


// ---- plan builder ------------------------------------------------------------------------------------
struct PlanBuilder {
    std::vector<CUtensorMap> maps;
    std::map<const void*, int> map_index;      // buffer -> index (static maps are shared by all problems)
    std::vector<Item> stage[8];
    std::vector<int> prob0;                    // stage 0: the problem (add_transform call) each item belongs to
    int cur_problem = 0;
    bool pair_ok = true;                       // every strip item of stages 5 / 6 so far can run in a pair launch
    // registers both box heights of a buffer; returns the index of the 64-row-box map, +1 is the 128-row-box map
    int add_map(const void* key, const CUtensorMap* m2) {
        auto it = map_index.find(key);
        if (it != map_index.end()) return it->second;
        maps.push_back(m2[0]);
        maps.push_back(m2[1]);
        map_index[key] = (int)maps.size() - 2;
        return (int)maps.size() - 2;
    }
    int add_single(const void* key, const CUtensorMap& m) {
        auto it = map_index.find(key);
        if (it != map_index.end()) return it->second;
        maps.push_back(m);
        map_index[key] = (int)maps.size() - 1;
        return (int)maps.size() - 1;
    }
};

struct Final {                  // what the last stage of a transform does with W~ (or Wg^)
    int mode;                   // EPI_AMAX (+ EPI_CAST), EPI_BLOCKCAST or EPI_STORE
    int fmt;
    const void* base; int base_type;
    void* out; int out_type;
    uint32_t* amax; float* scale_inv;
    uint32_t* done;             // fused update: the tensor's parked-tile counter (next to its amax word)
    int base_map[2];            // TMA-streamed base tile(s) (hi [+ lo]); -1: base read straight from global memory
    int out_map;                // TMA store map of the output (codes or BF16); -1: direct stores
    float* resid;               // f1: the tensor's FP32 error-feedback residual (null: plain codec)
};

inline Item blank_item() {
    Item it;
    memset(&it, 0, sizeof(it));
    it.base_map[0] = it.base_map[1] = it.out_map = -1;
    return it;
}

// Stages of out = T_G src T_A (inverse: T^-1) in the low-rank form; src_map indexes the BF16 source.
// split: every BF16 operand x is carried as hi + lo (x_hi = bf16(x), x_lo = bf16(x - x_hi)) and each product
// expands to hi*hi + lo*hi + hi*lo, which brings the tensor-core result to ~FP32 accuracy at 3x the MMAs.
// src_lo_map < 0 means the source is exactly BF16 (a BF16 gradient) and needs no residual.
void add_transform(PlanBuilder& pb, LayerState& L, Slot* s, int src_map, int src_lo_map, bool inverse, bool split,
                   const Final& f, const EngineOptions& opt, int c_num_sms = 148) {
    using namespace gf8::tc;
    const int m = L.desc.d_out, n = L.desc.d_in;
    const bool useA = L.in.used, useG = L.out.used;
    const int kpA = useA ? L.in.kp : 0, kpG = useG ? L.out.kp : 0;
    const float* eA = inverse ? L.in.ebar : L.in.e;
    const float* eG = inverse ? L.out.ebar : L.out.e;
    struct MapPair { int hi, lo; };
    auto pair = [&](bool use, const void* bh, const CUtensorMap* mh, const void* bl, const CUtensorMap* ml) {
        MapPair r{-1, -1};
        if (use) { r.hi = pb.add_map(bh, mh); if (split) r.lo = pb.add_map(bl, ml); }
        return r;
    };
    const MapPair mUA = pair(useA, L.in.U16, L.in.map_U16, L.in.U16_lo, L.in.map_U16_lo);
    const MapPair mUAt = pair(useA, L.in.Ut16, L.in.map_Ut16, L.in.Ut16_lo, L.in.map_Ut16_lo);
    const MapPair mUG = pair(useG, L.out.U16, L.out.map_U16, L.out.U16_lo, L.out.map_U16_lo);
    const MapPair mUGt = pair(useG, L.out.Ut16, L.out.map_Ut16, L.out.Ut16_lo, L.out.map_Ut16_lo);
    const MapPair mPp = pair(useA, s->Pp, s->map_Pp, s->Pp_lo, s->map_Pp_lo);
    const MapPair mQpt = pair(useG, s->Qpt, s->map_Qpt, s->Qpt_lo, s->map_Qpt_lo);
    const MapPair mSEA = pair(useA && useG, s->SEA, s->map_SEA, s->SEA_lo, s->map_SEA_lo);
    const MapPair mSrc{src_map, src_lo_map};
    // append the product A * B^T (hi*hi [+ lo*hi + hi*lo]) to an item
    // (map indices point at the 64-row-box map of a buffer; +1 is its 128-row-box map: a K-major A atom and a
    //  128-row B atom are one box each, an MN-major A atom is two 64 x 64 boxes)
    auto add_product = [&](Item& it, int& seg, MapPair a, MapPair b, int atoms, int a_c0, int a_r0, int b_c0, int b_r0) {
        const int ao = it.a_mn ? 0 : 1, bo = it.N == 128 ? 1 : 0;
        auto one = [&](int ma, int mb) {
            it.map_a[seg] = ma + ao; it.map_b[seg] = mb + bo; it.atoms[seg] = atoms;
            it.a_c0[seg] = a_c0; it.a_r0[seg] = a_r0; it.b_c0[seg] = b_c0; it.b_r0[seg] = b_r0;
            ++seg;
        };
        one(a.hi, b.hi);
        if (a.lo >= 0) one(a.lo, b.hi);
        if (b.lo >= 0) one(a.hi, b.lo);
    };
    // panels wider than 128 basis columns are cut into 128-column accumulator chunks (nc).
    // The row panels (P') and the column panels (Q^T) of a problem both stream the whole source: they share stage 0
    // and stay next to each other in its item list, so the CTAs working on one problem at a time fetch every source
    // byte from HBM once and find it in L2 the second time.
    const int problem = pb.cur_problem++;
    auto push0 = [&](const Item& it) { pb.stage[0].push_back(it); pb.prob0.push_back(problem); };
    // (kp <= 64: one item covers 256 rows, its two 128-row accumulators share every basis atom the loader brings in)
    const int stepA = kpA <= 64 ? 256 : 128, stepG = kpG <= 64 ? 256 : 128;
    if (useA)      // P' = (src U_A) E_A : row panels
        for (int i0 = 0; i0 < m; i0 += stepA)
            for (int nc = 0; nc < kpA; nc += 128) {
                Item it = blank_item();
                int seg = 0;
                it.N = std::min(128, kpA - nc);
                add_product(it, seg, mSrc, mUAt, (n + 63) / 64, 0, i0, 0, nc);
                it.tri = (seg == 3 && it.N <= 64) ? 1 : 0;      // split products of one operand pair: interleaved per K-atom
                it.mode = EPI_STORE; it.out = s->Pp; it.out_lo = split ? s->Pp_lo : nullptr; it.out_ld = kpA;
                it.out_type = TY_BF16; it.colscale = eA + nc;
                it.row0 = i0; it.col0 = nc; it.rows = std::min(stepA, m - i0); it.cols = it.N;
                push0(it);
            }
    if (useG) {    // Q^T = src^T U_G : column panels (A is MN-major)
        for (int j0 = 0; j0 < n; j0 += stepG)
            for (int nc = 0; nc < kpG; nc += 128) {
                Item it = blank_item();
                int seg = 0;
                it.a_mn = 1; it.N = std::min(128, kpG - nc);
                add_product(it, seg, mSrc, mUGt, (m + 63) / 64, j0, 0, 0, nc);
                it.tri = (seg == 3 && it.N <= 64) ? 1 : 0;
                it.mode = EPI_STORE; it.row0 = j0; it.col0 = nc; it.rows = std::min(stepG, n - j0); it.cols = it.N;
                if (useA) { it.out = s->Qt; it.out_ld = kpG; it.out_type = TY_F32; }
                else {
                    it.out = s->Qpt; it.out_lo = split ? s->Qpt_lo : nullptr; it.out_ld = kpG; it.out_type = TY_BF16;
                    it.colscale = eG + nc;
                }
                push0(it);
            }
        if (useA) {
            // (S E_A)^T = P'^T U_G, stored transposed as SEA[g][a]
            for (int a0 = 0; a0 < kpA; a0 += 128)
                for (int nc = 0; nc < kpG; nc += 128) {
                    Item it = blank_item();
                    int seg = 0;
                    it.a_mn = 1; it.N = std::min(128, kpG - nc);
                    add_product(it, seg, mPp, mUGt, (m + 63) / 64, a0, 0, 0, nc);
                    it.mode = EPI_STORE_T; it.out = s->SEA; it.out_lo = split ? s->SEA_lo : nullptr; it.out_ld = kpA;
                    it.out_type = TY_BF16;
                    it.row0 = a0; it.col0 = nc; it.rows = std::min(128, kpA - a0); it.cols = it.N;
                    pb.stage[1].push_back(it);
                }
            // Q'^T = (Q^T + U_A (S E_A)^T) E_G
            for (int j0 = 0; j0 < n; j0 += stepG)
                for (int nc = 0; nc < kpG; nc += 128) {
                    Item it = blank_item();
                    int seg = 0;
                    it.N = std::min(128, kpG - nc);
                    add_product(it, seg, mUA, mSEA, kpA / 64, 0, j0, 0, nc);
                    it.mode = EPI_STORE; it.base = s->Qt; it.base_ld = kpG; it.base_type = TY_F32;
                    it.out = s->Qpt; it.out_lo = split ? s->Qpt_lo : nullptr; it.out_ld = kpG; it.out_type = TY_BF16;
                    it.colscale = eG + nc;
                    it.row0 = j0; it.col0 = nc; it.rows = std::min(stepG, n - j0); it.cols = it.N;
                    pb.stage[2].push_back(it);
                }
        }
    }
    // rank-(kA + kG) update of the streamed base tile
    const int tiles_n = (n + 127) / 128;
    // Strip items (encode, K = kpA + kpG <= 128): one item = up to 256 rows x all columns; its A tiles [P' | U_G] stay
    // resident in shared memory and every B K-atom [U_A | Q'^T] serves both row blocks, which halves the bytes TMA has
    // to bring in per output tile (96 KB -> 48 KB) and amortises the per-item hand-shakes over 2 x n / 128 tiles.
    if (!split && kpA + kpG <= 128 && f.base_map[0] >= 0 && f.base_map[1] < 0 && f.out_map >= 0 &&
        (f.mode == EPI_AMAX || f.mode == EPI_BLOCKCAST) && !opt.nostrip && !opt.fuse) {
        // Pair launches (opt-in, GF8_TC_PAIR=1; per-tensor scaling): the strips are cut into sub-strips of about PAIR_TILES column
        // tiles (393 KB of gradient), each an (amax item, cast item) pair that one CTA runs back to back; the cast items start
        // once the tensor's `done` word has counted every amax item (8 epilogue warps each).  148 sub-strips in flight are 58 MB:
        // the cast pass finds its gradient tiles in L2 (measured: 12.9 GB of DRAM reads for both passes instead of 23.4).  A
        // tensor must not have more pairs than the launch has CTAs (its join would never complete), and a sub-strip must be
        // longer than the base ring (see the producer's deferred claim).  Not the default: DESIGN.md 5 says why it is not faster.
        constexpr int PAIR_TILES = 6;                        // column tiles per sub-strip (768 columns)
        const bool pairs = f.mode == EPI_AMAX && opt.pair && !opt.static_items && f.done;
        const int col_tiles = (n + 127) / 128;
        const int n_chunk = pairs ? (col_tiles + PAIR_TILES - 1) / PAIR_TILES : 1;      // column tiles spread evenly over the chunks
        const int n_pairs = ((m + 255) / 256) * n_chunk;
        if (!pairs || n_pairs > c_num_sms / 2) pb.pair_ok = false;
        for (int i0 = 0; i0 < m; i0 += 256)
          for (int q = 0, c0 = 0; q < n_chunk; ++q) {
            const int cw = pairs ? 128 * (col_tiles / n_chunk + (q < col_tiles % n_chunk ? 1 : 0)) : n;
            const int c_this = c0;
            c0 += cw;
            Item it = blank_item();
            int seg = 0;
            it.N = 128; it.fmt = f.fmt; it.strip = 1;
            if (useA) add_product(it, seg, mPp, mUA, kpA / 64, 0, i0, 0, c_this);
            if (useG) add_product(it, seg, mUG, mQpt, kpG / 64, 0, i0, 0, c_this);
            it.base_type = f.base_type; it.base_map[0] = f.base_map[0] + 1;
            it.row0 = i0; it.col0 = c_this; it.rows = std::min(256, m - i0); it.cols = std::min(cw, n - c_this);
            if (((it.rows + 127) / 128) * ((it.cols + 127) / 128) < 4) pb.pair_ok = false;      // (longer than the base ring)
            it.mode = f.mode; it.out = f.out; it.out_ld = n; it.out_map = f.out_map; it.scale_inv_out = f.scale_inv;
            it.out_lo = f.resid;                                   // (amax / cast modes: out_lo carries the feedback residual)
            if (f.mode == EPI_AMAX) {
                it.amax = f.amax;
                if (pairs) { it.sync = 1; it.base = f.done; it.base_ld = (int64_t)n_pairs * gf8::tc::EPI_WARPS; }
                pb.stage[5].push_back(it);
                it.mode = EPI_CAST; it.write_scale = (i0 == 0 && c_this == 0) ? 1 : 0;
                if (pairs) it.sync = 2;
                pb.stage[6].push_back(it);
            } else {
                pb.stage[5].push_back(it);
            }
          }
        return;
    }
    for (int i0 = 0; i0 < m; i0 += 128)
        for (int j0 = 0; j0 < n; j0 += 128) {
            Item it = blank_item();
            int seg = 0;
            it.N = 128; it.fmt = f.fmt;
            if (useA) add_product(it, seg, mPp, mUA, kpA / 64, 0, i0, 0, j0);
            if (useG) add_product(it, seg, mUG, mQpt, kpG / 64, 0, i0, 0, j0);
            it.base = f.base; it.base_ld = n; it.base_type = f.base_type;
            it.row0 = i0; it.col0 = j0; it.rows = std::min(128, m - i0); it.cols = std::min(128, n - j0);
            it.mode = f.mode;
            it.base_map[0] = f.base_map[0] >= 0 ? f.base_map[0] + 1 : -1;      // 128-row boxes
            it.base_map[1] = f.base_map[1] >= 0 ? f.base_map[1] + 1 : -1;
            const int n_tiles = ((m + 127) / 128) * tiles_n;
            if (f.mode == EPI_AMAX && f.done && f.out_map >= 0 && it.base_map[0] >= 0 && n_tiles <= gf8::tc::FUSE_LAG * c_num_sms &&
                opt.fuse) {
                // fused update (opt-in, GF8_TC_FUSE=1): one pass parks the FP32 tile in TMEM, the cast
                // follows when the tensor amax is complete.  It needs every CTA of the launch co-resident.
                it.amax = f.amax; it.out = f.out; it.out_ld = n; it.scale_inv_out = f.scale_inv; it.out_map = f.out_map;
                it.write_scale = (i0 == 0 && j0 == 0) ? 1 : 0;
                it.base = f.done; it.base_ld = n_tiles;
                pb.stage[7].push_back(it);
            } else if (f.mode == EPI_AMAX) {
                it.amax = f.amax; it.out_lo = f.resid; it.out_ld = n;
                pb.stage[3].push_back(it);
                it.mode = EPI_CAST; it.out = f.out; it.out_ld = n; it.scale_inv_out = f.scale_inv; it.out_map = f.out_map;
                it.write_scale = (i0 == 0 && j0 == 0) ? 1 : 0;
                pb.stage[4].push_back(it);
            } else if (f.mode == EPI_BLOCKCAST) {
                it.out = f.out; it.out_ld = n; it.out_map = f.out_map; it.out_lo = f.resid;
                it.scale_inv_out = f.scale_inv + (size_t)(i0 / 128) * tiles_n + j0 / 128;
                pb.stage[3].push_back(it);
            } else {
                it.out = f.out; it.out_ld = n; it.out_type = f.out_type; it.out_map = f.out_map;
                pb.stage[3].push_back(it);
            }
        }
}

void plan_free(Plan* p) {
    if (!p) return;
    cudaFree(p->d_maps);
    cudaFree(p->d_items);
    cudaFree(p->d_amax);
    cudaFree(p->d_ctr);
    delete p;
}

// Upload the builder's maps and items (longest contractions first within a stage: CTAs take items round-robin).
gf8_status plan_finish(gf8_ctx* c, PlanBuilder& pb, Plan* p) {
    std::vector<Item> all;
    if (pb.prob0.size() == pb.stage[0].size() && !pb.stage[0].empty()) {
        // stage 0: heaviest problems first, each problem's panels contiguous (L2 reuse of the source, see add_transform)
        std::vector<int64_t> work(pb.cur_problem, 0);
        for (size_t i = 0; i < pb.stage[0].size(); ++i)
            for (int g = 0; g < gf8::tc::NSEG; ++g) work[pb.prob0[i]] += pb.stage[0][i].atoms[g];
        std::vector<int> order(pb.stage[0].size());
        for (size_t i = 0; i < order.size(); ++i) order[i] = (int)i;
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
            const int pa = pb.prob0[a], pq = pb.prob0[b];
            if (work[pa] != work[pq]) return work[pa] > work[pq];
            return pa < pq;
        });
        // Waves (items are handed out in list order, so list order is start order).  Within a problem the row panels
        // sweep the source along its columns and the column panels along its rows; when one kind is rho times longer
        // (m != n), the short panels are cut into rho bands along the long panels' sweep and band b is listed one
        // wave later than band b - 1, for a group of as many problems as the SMs hold at once.  Each band then runs
        // while the long panels cross it, and the second reader of a source byte finds it in L2.
        struct Prob { std::vector<int> lng, sht; int rho = 1; };
        std::vector<Prob> probs;
        for (size_t q = 0; q < order.size();) {
            const int pid = pb.prob0[order[q]];
            std::vector<int> rowp, colp;
            int64_t ar = 0, ac = 0;
            for (; q < order.size() && pb.prob0[order[q]] == pid; ++q) {
                const Item& it = pb.stage[0][order[q]];
                int64_t a = 0;
                for (int g = 0; g < gf8::tc::NSEG; ++g) a += it.atoms[g];
                if (it.a_mn) { colp.push_back(order[q]); ac = a; } else { rowp.push_back(order[q]); ar = a; }
            }
            Prob pr;
            const bool col_long = ac > ar;
            pr.lng = col_long ? colp : rowp;
            pr.sht = col_long ? rowp : colp;
            if (pr.lng.empty()) { pr.lng.swap(pr.sht); }
            const int64_t al = std::max(ar, ac), as = std::min(ar, ac);
            pr.rho = (!pr.sht.empty() && as > 0) ? (int)std::max<int64_t>(1, (al + as / 2) / as) : 1;
            pr.rho = std::min<int>(pr.rho, (int)std::max<size_t>(1, pr.sht.size()));
            probs.push_back(std::move(pr));
        }
        std::vector<Item> sorted;
        sorted.reserve(order.size());
        for (size_t g0 = 0; g0 < probs.size();) {
            const Prob& first = probs[g0];
            const int per = (int)first.lng.size() + (int)((first.sht.size() + first.rho - 1) / first.rho);
            const size_t G = (size_t)std::max(1, c->num_sms / std::max(1, per));
            const size_t g1 = std::min(probs.size(), g0 + G);
            int waves = 1;
            for (size_t q = g0; q < g1; ++q) waves = std::max(waves, probs[q].rho);
            for (int w = 0; w < waves; ++w)
                for (size_t q = g0; q < g1; ++q) {
                    const Prob& pr = probs[q];
                    if (w == 0) for (int i : pr.lng) sorted.push_back(pb.stage[0][i]);
                    if (w < pr.rho) {
                        const size_t nb = (pr.sht.size() + pr.rho - 1) / pr.rho;
                        for (size_t k = (size_t)w * nb; k < std::min(pr.sht.size(), (size_t)(w + 1) * nb); ++k)
                            sorted.push_back(pb.stage[0][pr.sht[k]]);
                    }
                }
            g0 = g1;
        }
        pb.stage[0].swap(sorted);
    }
    // pair launch: stage 5 becomes (amax item, cast item) pairs in call order; otherwise the sync marks are dropped and the two
    // passes run as two launches
    bool pair5 = pb.pair_ok && !pb.stage[5].empty() && pb.stage[5].size() == pb.stage[6].size();
    for (size_t i = 0; pair5 && i < pb.stage[5].size(); ++i) pair5 = pb.stage[5][i].sync == 1 && pb.stage[6][i].sync == 2;
    if (pair5) {
        std::vector<Item> merged;
        merged.reserve(2 * pb.stage[5].size());
        for (size_t i = 0; i < pb.stage[5].size(); ++i) { merged.push_back(pb.stage[5][i]); merged.push_back(pb.stage[6][i]); }
        pb.stage[5].swap(merged);
        pb.stage[6].clear();
    } else {
        for (int s = 5; s <= 6; ++s)
            for (Item& it : pb.stage[s]) if (it.sync) { it.sync = 0; it.base = nullptr; it.base_ld = 0; }
    }
    p->pair5 = pair5;
    for (int s = 0; s < 8; ++s) {
        const bool grouped = (s == 0 && pb.prob0.size() == pb.stage[0].size()) || (s == 5 && pair5);
        if (!grouped) std::stable_sort(pb.stage[s].begin(), pb.stage[s].end(), [](const Item& a, const Item& b) {
            int64_t ta = 0, tb = 0;
            for (int g = 0; g < gf8::tc::NSEG; ++g) { ta += a.atoms[g]; tb += b.atoms[g]; }
            if (a.strip) ta *= (int64_t)((a.rows + 127) / 128) * ((a.cols + 127) / 128);
            if (b.strip) tb *= (int64_t)((b.rows + 127) / 128) * ((b.cols + 127) / 128);
            return ta > tb;
        });
        p->stage_off[s] = (int)all.size();
        p->stage_cnt[s] = (int)pb.stage[s].size();
        for (const Item& it : pb.stage[s]) {
            p->stage_base[s] = std::max(p->stage_base[s], (it.base_map[0] >= 0 ? 1 : 0) + (it.base_map[1] >= 0 ? 1 : 0));
            if (!it.strip && it.rows > 128) p->stage_wide[s] |= 1;
            if (it.N > 64) p->stage_wide[s] |= 2;
        }
        if (!(p->stage_wide[s] & 1)) p->stage_wide[s] = 0;            // 0 none, 1 wide (B <= 8 KB), 3 wide with N = 128 items
        bool all_tri = !pb.stage[s].empty() && !c->opt.notri;
        for (const Item& it : pb.stage[s]) all_tri = all_tri && it.tri != 0;
        if (all_tri) p->stage_wide[s] = 5;                            // 5: every item interleaves its split products (kmode 5)
        else for (Item& it : pb.stage[s]) it.tri = 0;
        all.insert(all.end(), pb.stage[s].begin(), pb.stage[s].end());
    }
    if (all.empty()) return GF8_OK;
    void* q = nullptr;
    if (cudaMalloc(&q, pb.maps.size() * sizeof(CUtensorMap)) != cudaSuccess) { cudaGetLastError(); return fail(c, GF8_ERR_NOMEM, "plan maps"); }
    p->d_maps = (CUtensorMap*)q;
    if (cudaMalloc(&q, all.size() * sizeof(Item)) != cudaSuccess) { cudaGetLastError(); return fail(c, GF8_ERR_NOMEM, "plan items"); }
    p->d_items = (Item*)q;
    if (cudaMalloc(&q, 8 * sizeof(int)) != cudaSuccess) { cudaGetLastError(); return fail(c, GF8_ERR_NOMEM, "plan counters"); }
    p->d_ctr = (int*)q;
    CU_TRY(c, cudaMemcpy(p->d_maps, pb.maps.data(), pb.maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice));
    CU_TRY(c, cudaMemcpy(p->d_items, all.data(), all.size() * sizeof(Item), cudaMemcpyHostToDevice));
    return GF8_OK;
}

gf8_status plan_store(gf8_ctx* c, const std::vector<uint64_t>& key, Plan* p) {
    if (c->plan_order.size() >= FAST_MAX_PLANS) {
        CU_TRY(c, cudaDeviceSynchronize());
        Plan* old = c->plan_order.front();
        c->plan_order.erase(c->plan_order.begin());
        for (auto it = c->plans.begin(); it != c->plans.end(); ++it)
            if (it->second == old) { c->plans.erase(it); break; }
        plan_free(old);
    }
    c->plans[key] = p;
    c->plan_order.push_back(p);
    return GF8_OK;
}

gf8_status plan_run_stages(gf8_ctx* c, cudaStream_t st, Plan* p) {
    p->runs++;
    if (p->d_ctr) CU_TRY(c, cudaMemsetAsync(p->d_ctr, 0, 8 * sizeof(int), st));
    for (int s = 0; s < 8; ++s) {
        if (!p->stage_cnt[s]) continue;
        const bool pair = s == 5 && p->pair5;
        const int grid = std::min(pair ? p->stage_cnt[s] / 2 : p->stage_cnt[s], c->num_sms);
        const int n_base = p->stage_base[s];
        // shared-memory split: update stages keep a short operand ring (their operands are L2-resident) and give
        // the rest to base tiles in flight (the HBM stream); panel stages give everything to the operand ring
        const int fuse = s == 7 ? 1 : 0, strip = (s == 5 || s == 6) ? 1 : 0, wide = p->stage_wide[s] && !n_base ? 1 : 0;
        const int kmode0 = fuse ? 1 : (pair ? 6 : strip ? 2 : (wide ? (p->stage_wide[s] == 5 ? 5 : (p->stage_wide[s] == 3 ? 4 : 3)) : 0));
        // tile items with streamed bases (the update stages of decode and of ranks above 64) are handed out in runs of 8
        const int claim_chunk = ((s == 3 || s == 4) && n_base > 0 && !fuse) ? 8 : 1;
        const int kmode = kmode0 | (claim_chunk > 1 ? claim_chunk << 8 : 0);
        // shared-memory split of the tile-mode update stages: 3 operand stages + the rest as base tiles in flight
        int n_stages = n_base ? (strip ? 4 : 3) : (wide ? (p->stage_wide[s] == 5 ? 2 : (p->stage_wide[s] == 3 ? 4 : 5)) : gf8::tc::MAX_STAGES), dbg = 0;
#ifdef GF8_DEBUG
        int only = -1;
#endif
        // (strip stages: 64 KB of resident A tiles + 4 x 16 KB of B atoms = the first four 32 KB units, then 3 base slots)
        // (the fused stage gives one base slot's worth of shared memory to its two code-tile staging buffers)
        const int n_bslots = fuse ? 3 : (n_base ? std::max(1, (gf8::tc::MAX_STAGES - n_stages) / n_base) : 1);
        if (n_base && !fuse && n_stages + n_bslots * n_base > gf8::tc::MAX_STAGES) n_stages = gf8::tc::MAX_STAGES - n_bslots * n_base;
        if (fuse && grid < c->num_sms && p->stage_cnt[s] > grid) return fail(c, GF8_ERR_BAD_STATE, "fused stage needs a full grid");
#ifdef GF8_DEBUG
        // GF8_TC_DBG (debug only, results are wrong with the ablation bits): 1 skip the MMAs, 2 skip the tensor-map
        // fences, 4 print a per-role wait profile, 32 skip the update epilogue's work, 64 skip the streamed base loads,
        // 128 skip the strip B loads, 256 print each stage's device time (serialises the stream), 2048 (with 4) print the
        // timeline of CTA 1's items 6..15 per role (tile items: publish / loads / MMA / epilogue, cycles), 4096 / 8192 / 16384
        // skip the base loads / column multipliers / stores of the panel epilogue
        if (const char* e = getenv("GF8_TC_DBG")) dbg = atoi(e);
        if (const char* e = getenv("GF8_TC_ONLY")) only = atoi(e);
        if (only >= 0 && only != s) continue;
        cudaEvent_t ev0 = nullptr, ev1 = nullptr;
        if (dbg & 256) { cudaEventCreate(&ev0); cudaEventCreate(&ev1); cudaEventRecord(ev0, st); }
        static std::vector<std::pair<int, std::pair<cudaEvent_t, cudaEvent_t>>> pend;     // bit 9: the same without serialising
        if (dbg & 512) {
            if (s == 0 || pend.size() > 64) {
                for (auto& e : pend) {
                    float ms = 0;
                    cudaEventSynchronize(e.second.second); cudaEventElapsedTime(&ms, e.second.first, e.second.second);
                    fprintf(stderr, "stage %d (async): %.1f us\n", e.first, ms * 1e3);
                    cudaEventDestroy(e.second.first); cudaEventDestroy(e.second.second);
                }
                pend.clear();
            }
            cudaEvent_t a, b;
            cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, st);
            pend.push_back({s, {a, b}});
        }
#endif
        gf8_ctx::StageEvent sev{s, nullptr, nullptr};
        if (c->stage_timing) {
            if (!c->stage_event_pool.empty()) { sev = c->stage_event_pool.back(); c->stage_event_pool.pop_back(); sev.stage = s; }
            else { CU_TRY(c, cudaEventCreate(&sev.a)); CU_TRY(c, cudaEventCreate(&sev.b)); }
            CU_TRY(c, cudaEventRecord(sev.a, st));
        }
        auto* kern = (p->ef && s >= 3) ? gf8::tc::tc_items_kernel<true> : gf8::tc::tc_items_kernel<false>;     // (f1: update stages only)
        kern<<<grid, gf8::tc::THREADS, gf8::tc::SMEM_BYTES, st>>>(
            p->d_items + p->stage_off[s], p->stage_cnt[s], p->d_maps, c->d_err, n_stages, n_base, n_bslots, kmode, dbg, (dbg & 4) ? c->d_prof : nullptr,
            (fuse || c->opt.static_items) ? nullptr : p->d_ctr + s);
        if (c->stage_timing) { CU_TRY(c, cudaEventRecord(sev.b, st)); c->stage_events.push_back(sev); }
#ifdef GF8_DEBUG
        if (dbg & 512) cudaEventRecord(pend.back().second.second, st);
        if (dbg & 256) {                 // GF8_TC_DBG bit 8: per-stage device time (serialises the stream)
            float ms = 0;
            cudaEventRecord(ev1, st); cudaEventSynchronize(ev1); cudaEventElapsedTime(&ms, ev0, ev1);
            fprintf(stderr, "stage %d: %d items, %.1f us\n", s, p->stage_cnt[s], ms * 1e3);
            cudaEventDestroy(ev0); cudaEventDestroy(ev1);
        }
        if ((dbg & 2048) && (dbg & 4)) {      // bit 11: item timeline of CTA 1 (tile items): cycles since the CTA's first event
            std::vector<long long> t(5 * 48 * 4);
            cudaDeviceSynchronize();
            cudaMemcpy(t.data(), c->d_prof + 8192, t.size() * sizeof(long long), cudaMemcpyDeviceToHost);
            long long t0 = 0;
            for (long long x : t) if (x > 0 && (t0 == 0 || x < t0)) t0 = x;
            const char* rn[5] = {"prod", "ldA", "ldB", "mma", "epi"};
            for (int it = 6; it < 16; ++it) {
                fprintf(stderr, "stage %d item %2d:", s, it);
                for (int r = 0; r < 5; ++r) {
                    fprintf(stderr, "  %s", rn[r]);
                    for (int e = 0; e < 4; ++e) { const long long x = t[(r * 48 + it) * 4 + e]; fprintf(stderr, " %6lld", x > 0 ? x - t0 : -1); }
                }
                fprintf(stderr, "\n");
            }
            cudaMemset(c->d_prof + 8192, 0, t.size() * sizeof(long long));
        }
        if (dbg & 4) {
            std::vector<long long> h((size_t)c->num_sms * 36);
            cudaMemcpy(h.data(), c->d_prof, h.size() * sizeof(long long), cudaMemcpyDeviceToHost);
            const char* roles[6] = {"epilogue", "base", "load A", "load B", "mma", "mma 2"};
            for (int r = 0; r < 6; ++r) {
                double a[6] = {0, 0, 0, 0, 0, 0};
                for (int b = 0; b < grid; ++b) for (int q = 0; q < 6; ++q) a[q] += (double)h[((size_t)b * 6 + r) * 6 + q] / grid;
                fprintf(stderr, "stage %d %-8s waits[0..2] %.0f %.0f %.0f  work %.0f  post %.0f  total %.0f cycles (avg/CTA)\n", s, roles[r], a[0], a[1], a[2], a[3], a[4], a[5]);
            }
        }
#endif
        LAUNCH_CHECK(c);
    }
    return GF8_OK;
}

}  // namespace
