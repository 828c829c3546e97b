// gf8_ctx.cuh -- internal: the context behind the opaque gf8_ctx of include/gf8.h, and small host helpers.
#pragma once
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <vector>

#include <cuda.h>

#include "../../include/gf8.h"
#include "gf8_common.cuh"

namespace {

struct SideState {
    int d = 0, k = 0;
    bool used = false;
    float* factor = nullptr;   // d x d FP32 (lazy)
    bool has_factor = false;   // at least one update / set
    float* U = nullptr;        // d x k FP32 row-major
    float* mu = nullptr;       // k
    float* e = nullptr;        // k  encode multipliers
    float* ebar = nullptr;     // k  decode multipliers
    float* rho = nullptr;      // 1
    bool has_start = false, has_basis = false;
    // FAST path (tensor cores): rank padded to a multiple of 64, BF16 copies of the basis, TMA maps
    int kp = 0;
    gf8::bf16* U16 = nullptr;  // d x kp   (zero-padded columns)
    gf8::bf16* Ut16 = nullptr; // kp x d
    gf8::bf16 *U16_lo = nullptr, *Ut16_lo = nullptr;   // BF16 residuals U - bf16(U) (split-operand products)
    // every TMA map exists for 64-row boxes [0] and 128-row boxes [1] (64 columns = one 128 B swizzle span)
    CUtensorMap map_U16[2], map_Ut16[2], map_U16_lo[2], map_Ut16_lo[2];
};

// Per (layer, occurrence-in-batch) scratch of the FAST path; buffers and their TMA maps are static.
struct Slot {
    gf8::bf16* Pp = nullptr;   // m x kpA   P' = (src U_A) E_A
    float* Qt = nullptr;       // n x kpG   Q^T
    gf8::bf16* Qpt = nullptr;  // n x kpG   Q'^T
    gf8::bf16* SEA = nullptr;  // kpG x kpA S E_A
    gf8::bf16 *Pp_lo = nullptr, *Qpt_lo = nullptr, *SEA_lo = nullptr;   // residuals, lazy (split products)
    CUtensorMap map_Pp[2], map_Qpt[2], map_SEA[2], map_Pp_lo[2], map_Qpt_lo[2], map_SEA_lo[2];
    float* Uhat = nullptr;     // m x n FP32 reduced payload (decode), lazy
    gf8::bf16* src16 = nullptr;// m x n BF16 copy of an FP32 source (decode, FP32 gradients), lazy
    gf8::bf16* src16_lo = nullptr;
    CUtensorMap map_src16[2], map_src16_lo[2];
};

struct LayerState {
    gf8_layer_desc desc;
    SideState in, out;         // in: A / U_A (d_in), out: Gf / U_G (d_out)
    size_t n_scales = 1;
    uint32_t* amax_bits = nullptr;   // n_scales
    float* scale = nullptr;          // n_scales
    float* P = nullptr;              // m x kA
    float* Q = nullptr;              // kG x n
    float* S = nullptr;              // kG x kA
    bool tc_ok = false;              // FAST path eligible (tensor-core engine)
    std::vector<Slot*> slots;
};

}  // namespace

constexpr int GF8_HOST_CHUNKS = 12;   // gf8_step_host pipelines a step in at most this many chunks of tensors

struct RefreshScratch {
    double *V = nullptr, *Y = nullptr, *Gm = nullptr, *Bm = nullptr, *Zm = nullptr, *Zs = nullptr, *mu64 = nullptr;
};

// Engine switches, read ONCE from the environment in gf8_create (experiments / fall-backs; defaults are what bench.py times).
struct EngineOptions {
    bool nostrip = false;        // GF8_TC_NOSTRIP: update as 128 x 128 tile items instead of 256-row strips
    bool fuse = false;           // GF8_TC_FUSE: single-pass update with W~ parked in TMEM (static round-robin; slower: DESIGN.md 5)
    bool notri = false;          // GF8_TC_NOTRI: split products as three K-loops instead of interleaved per K-atom
    bool static_items = false;   // GF8_TC_STATIC: static item assignment instead of the atomic hand-out
    bool pair = false;           // GF8_TC_PAIR: both update passes of the encode in ONE launch of (amax, cast) item pairs
};

struct gf8_ctx {
    EngineOptions opt;
    int device = 0;
    gf8_precision precision = GF8_PREC_EXACT;
    bool tc_exact = false;           // EXACT on the tensor-core engine with hi + lo operands (opt-in, GF8_EXACT_TC=1)
    std::vector<LayerState> layers;
    std::vector<void*> allocs;
    float* wt_scratch = nullptr;     // max m*n FP32
    // refresh scratch (FP64): one set per concurrent refresh stream (gf8_refresh_basis_many); set 0 serves single calls
    RefreshScratch rs[1];
    size_t rs_dk = 0, rs_k = 0;
    // batched refresh (gf8_refresh.cuh): scratch arena (doubles), job records, and the event that guards their reuse
    double* rb_arena = nullptr; size_t rb_arena_cap = 0;
    void* rb_jobs = nullptr; size_t rb_jobs_cap = 0;
    cudaEvent_t rb_ev = nullptr; bool rb_busy = false;
    // auxiliary stream: the streaming kernels of Euclidean tensors overlap the tensor-core stages of a batched call
    cudaStream_t aux_stream = nullptr;
    cudaEvent_t aux_fork_ev = nullptr, aux_join_ev = nullptr;
    void* gemm_ws = nullptr; size_t gemm_ws_bytes = 0;   // split-K workspace of the SIMT GEMM (partial products, summed in order)
    float* ef_scratch = nullptr; size_t ef_cap = 0;   // FP32 W~ of a chunk of problems (gf8_encode_ef_many)
    // tap scratch (gf8_quantize_f32 with arbitrary shapes)
    uint32_t* tap_amax = nullptr; float* tap_scale = nullptr; size_t tap_cap = 0;
    // host-step staging; copy-in / copy-out streams and the per-chunk events of the pipelined gf8_step_host
    cudaStream_t hs_in = nullptr, hs_out = nullptr;
    cudaEvent_t hs_start = nullptr, hs_done = nullptr, hs_in_ev[GF8_HOST_CHUNKS] = {}, hs_comp_ev[GF8_HOST_CHUNKS] = {};
    std::vector<void*> stage_allocs;
    std::vector<void*> st_grads; std::vector<uint8_t*> st_codes; std::vector<float*> st_sinv; std::vector<void*> st_out;
    std::vector<int> st_layers; int st_R = 0; int st_dt = -1;
    // FAST path: cached launch plans (device item lists + tensor maps), error flag, driver entry point
    std::map<std::vector<uint64_t>, struct Plan*> plans;
    std::vector<struct Plan*> plan_order;
    std::vector<struct SPlan*> splans;                          // streaming-engine plans (keyed by the layer list of a call)
    bool stream_attr_set = false;
    bool use_stream = false;         // streaming engine (gf8_stream.cuh) instead of the staged item engine for the shapes it takes
    int* d_err = nullptr;
    // factor GEMM (gf8_factor.cuh): job records of a call, staged through two pinned / device buffer pairs
    void* fac_h[2] = {nullptr, nullptr};
    void* fac_d[2] = {nullptr, nullptr};
    cudaEvent_t fac_ev[2] = {nullptr, nullptr};
    bool fac_busy[2] = {false, false};
    size_t fac_cap = 0;              // job records per buffer
    int fac_cur = 0;
    bool fac_attr_set = false;
    size_t chol_smem_set = 0, jacobi_smem_set = 0;   // dynamic shared memory sizes the refresh kernels are opted in to
    long long* d_prof = nullptr;     // debug profile of the TC kernel (GF8_TC_DBG & 4)
    void* encode_tiled = nullptr;    // cuTensorMapEncodeTiled, resolved at run time (no link-time libcuda)
    bool tc_attr_set = false;
    int64_t launches = 0;
    // stage timing (gf8_set_stage_timing): event pairs recorded around stage launches, drained by gf8_stage_times
    bool stage_timing = false;
    struct StageEvent { int stage; cudaEvent_t a, b; };
    std::vector<StageEvent> stage_events, stage_event_pool;
    int num_sms = 148;
    int aux_per_sm = 0;              // > 0: cap streaming grids at this many CTAs per SM (kernels that share SMs with the TC engine)
    char err[512] = {0};
};

namespace {

gf8_status fail(gf8_ctx* c, gf8_status s, const char* fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return s;
}

#define CU_TRY(ctx, expr)                                                                            \
    do {                                                                                             \
        cudaError_t _e = (expr);                                                                     \
        if (_e != cudaSuccess)                                                                       \
            return fail((ctx), GF8_ERR_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), \
                        __FILE__, __LINE__);                                                         \
    } while (0)

#define GF_TRY(expr)                       \
    do {                                   \
        gf8_status _s = (expr);            \
        if (_s != GF8_OK) return _s;       \
    } while (0)

#define LAUNCH_CHECK(ctx)                  \
    do {                                   \
        (ctx)->launches++;                 \
        CU_TRY((ctx), cudaGetLastError()); \
    } while (0)

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

template <typename T>
gf8_status dmalloc(gf8_ctx* c, T** p, size_t count, std::vector<void*>* track = nullptr) {
    void* q = nullptr;
    cudaError_t e = cudaMalloc(&q, count * sizeof(T) + 16);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(c, GF8_ERR_NOMEM, "cudaMalloc of %zu bytes failed: %s", count * sizeof(T), cudaGetErrorString(e));
    }
    (track ? *track : c->allocs).push_back(q);
    *p = static_cast<T*>(q);
    return GF8_OK;
}

inline size_t n_scales_of(int scaling, int64_t m, int64_t n) {
    return scaling == GF8_SCALE_TENSOR ? 1 : (size_t)((m + 127) / 128) * (size_t)((n + 127) / 128);
}
inline float fmax_of(int fmt) { return fmt == GF8_E4M3 ? 448.0f : 57344.0f; }

inline int grid_for(gf8_ctx* c, int64_t work_items, int threads, int per_sm) {
    int64_t blocks = (work_items + threads - 1) / threads;
    const int64_t cap = (int64_t)c->num_sms * (c->aux_per_sm > 0 ? std::min(per_sm, c->aux_per_sm) : per_sm);
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    return (int)blocks;
}

}  // namespace
