/* gf8.h -- C ABI of the B200-native GeoFP8 gradient codec (arXiv 2607.07494, "GeoFP8").
 *
 * The library implements the data-parallel hot path of the paper: per weight-gradient matrix
 *   Wg (d_out x d_in, row-major, Eq. 5)
 * it keeps K-FAC factors A = E[a a^T], Gf = E[delta delta^T] (Eq. 4), reduces each to a
 * damped rank-k eigen model (Eq. 24), whitens Wg into near-isotropic coordinates
 *   W~ = T_G Wg T_A,  T = I + U_k diag(e) U_k^T            (PAPER.md:158 Eq. 14, :180 Eq. 18, :250 Eq. 22)
 * scales and casts W~ to FP8 (Eq. 16; Alg. 1 l.12-13), and on the receive side
 * dequantises R payloads, sums them in FP32 (Eq. 1; Alg. 1 l.20-21) and maps back
 *   Wg^ = T_G^-1 U^ T_A^-1                                   (PAPER.md:172 Eq. 17, :184 Eq. 19).
 * DESIGN.md lists every reading taken where the paper is silent (S1..S15).
 *
 * Conventions (all entry points):
 *  - Every data pointer is a DEVICE pointer to caller-owned memory unless the parameter name ends
 *    in `_host`.  The library never frees caller memory and never keeps a caller pointer past
 *    the stream-ordered completion of the call.  Pointers must be 16-byte aligned.
 *  - Matrices are dense row-major.  Wg is [d_out][d_in] (the nn.Linear.weight.grad layout).
 *    codes: one byte per element, same layout.  Block scales: row-major over the
 *    ceil(d_out/128) x ceil(d_in/128) grid.
 *  - d_out and d_in must be multiples of 16 (else GF8_ERR_UNSUPPORTED).
 *  - `stream` is a cudaStream_t passed as void*.  Calls are asynchronous on that stream, run no host
 *    eigensolver and have no CPU fallback.  A ctx serves ONE stream at a time: its scratch is shared by
 *    consecutive calls, so calls on different streams must be ordered by the caller.
 *  - The ctx owns factors, bases, multipliers, scratch and cached launch plans.  What a call may do besides
 *    launching kernels:
 *      * FIRST call with a new argument list (layers, and for encode / decode the data pointers): builds and caches
 *        the call's plan -- device item lists and TMA tensor maps -- with cudaMalloc and small synchronous copies.
 *        A loop that reuses its buffers pays this once (64 plans are kept; the oldest is dropped after a
 *        device synchronisation).
 *      * buffers that grow allocate when they grow: factor accumulators (d^2 FP32 per side) at the first
 *        gf8_factor_update / gf8_set_factor of a layer, the refresh arena, the error-feedback scratch, the
 *        staging of gf8_step_host.
 *      * steady state: no allocation, no host synchronisation -- except that the pinned records of the batched
 *        factor / refresh calls are double-buffered and a call waits (cudaEventSynchronize) for the call two
 *        before it if that one is still running.
 *  - Reproducibility: every path sums in a fixed order (tensor-core pipelines, the batched geometry calls, and the FP32 /
 *    FP64 SIMT GEMM, whose split-K partial products go through a workspace and are added up in split order): the same call
 *    on the same inputs returns the same bits from run to run.
 *  - Errors: a gf8_status is returned; nothing throws or aborts across the ABI.  Argument errors
 *    are detected before any launch.  gf8_last_error(ctx) gives a message for the last failure.
 *  - One ctx (hence one basis per layer) is shared by all R simulated ranks (S12).
 */
#ifndef GF8_H
#define GF8_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gf8_ctx gf8_ctx;

typedef enum {
    GF8_OK = 0,
    GF8_ERR_INVALID_ARG = 1,
    GF8_ERR_BAD_STATE = 2,   /* e.g. encode on a whitened layer before a basis exists */
    GF8_ERR_UNSUPPORTED = 3, /* misaligned pointer, dims not multiple of 16, rank too large */
    GF8_ERR_NOMEM = 4,
    GF8_ERR_CUDA = 5
} gf8_status;

typedef enum { GF8_E4M3 = 0, GF8_E5M2 = 1 } gf8_format;           /* ref [24] */
typedef enum { GF8_SCALE_TENSOR = 0, GF8_SCALE_BLOCK128 = 1 } gf8_scaling;
/* Which factors whiten the layer.  NONE = Euclidean branch (Alg. 1 l.3-8);
 * IN = the paper's deployed form (Eq. 18-19); OUT, BOTH = Eq. 14 / Table I variants. */
typedef enum { GF8_SIDE_NONE = 0, GF8_SIDE_IN = 1, GF8_SIDE_OUT = 2, GF8_SIDE_BOTH = 3 } gf8_side;
typedef enum { GF8_DT_BF16 = 0, GF8_DT_F32 = 1 } gf8_dtype;
/* EXACT: transform within 1e-4 relative Frobenius of the FP64 oracle (FP32 arithmetic, or
 *        BF16x3 split operands on the tensor cores).
 * FAST : single-pass BF16 tensor-core operands, 2e-3 tier. */
typedef enum { GF8_PREC_EXACT = 0, GF8_PREC_FAST = 1 } gf8_precision;

#define GF8_MAX_RANK 512   /* k <= min(d, 512) */
#define GF8_MAX_R 64       /* simulated ranks per reduce call */

typedef struct {
    int32_t d_out, d_in;       /* m, n */
    int32_t rank_in, rank_out; /* k of U_A (input side), k of U_G (output side); ignored if unused */
    int32_t side;              /* gf8_side */
    int32_t fmt;               /* gf8_format */
    int32_t scaling;           /* gf8_scaling */
    float damping;             /* lambda, added to eigenvalues at refresh (S3) */
    float ema_beta;            /* beta of the factor EMA after the first update (S4); 0 = replace */
} gf8_layer_desc;

/* ---- lifetime ---------------------------------------------------------------------------------- */
/* Creates a context on CUDA device `device` for `n_layers` gradient matrices. */
gf8_status gf8_create(gf8_ctx** out, int device, const gf8_layer_desc* layers_host, int n_layers,
                      gf8_precision precision);
gf8_status gf8_destroy(gf8_ctx* ctx);
/* code_bytes = d_out*d_in; n_scales = 1 or ceil(d_out/128)*ceil(d_in/128). */
gf8_status gf8_payload_size(const gf8_ctx* ctx, int layer, size_t* code_bytes, size_t* n_scales);
const char* gf8_status_string(gf8_status s);
const char* gf8_last_error(const gf8_ctx* ctx);
/* Synchronises `stream` and reports asynchronous failures: GF8_ERR_CUDA if a kernel faulted or if the
 * tensor-core engine flagged a pipeline time-out (its bounded waits drain instead of hanging the GPU). */
gf8_status gf8_sync_check(gf8_ctx* ctx, void* stream);
/* Number of kernels this context has launched so far (bench.py's gpu_launches). */
int64_t gf8_launch_count(const gf8_ctx* ctx);
/* Per-launch timing of the tensor-core engine's stages, for roofline reporting (bench.py).  While enabled, every stage launch
 * of a batched FAST call is bracketed by CUDA events on the call's stream (no host synchronisation is added).
 * gf8_stage_times synchronises `stream`, then writes, for stage s in 0..7 (0 panels P' and Q^T, 1 S, 2 Q'^T, 3 / 4 update tiles
 * (amax or store / cast), 5 / 6 update strips (amax / cast), 7 fused update), the summed device milliseconds and the number of
 * launches since the last call, and resets the sums.  ms_out / n_out: HOST arrays of 8. */
gf8_status gf8_set_stage_timing(gf8_ctx* ctx, int enable);
gf8_status gf8_stage_times(gf8_ctx* ctx, float* ms_out_host, int* n_out_host, void* stream);

/* ---- geometry state (every K steps) ------------------------------------------------ */
/* a1.  A <- beta A + (1-beta) X^T X / T,  Gf likewise from Delta (Eq. 4).  The first
 * update of a layer replaces (beta ignored).  act is [T][d_in], gout is [T][d_out], both `dt`;
 * a side the layer does not use may be NULL.  Damping is NOT stored in the accumulator. */
gf8_status gf8_factor_update(gf8_ctx* ctx, int layer, const void* act, const void* gout, int64_t T,
                             gf8_dtype dt, void* stream);
/* a2.  Rank-k eigenbasis of each factor of the layer by subspace iteration (Eq. 24):
 * V <- orth(V0); n_iter x { V <- orth(A V) }; Rayleigh-Ritz with a single-CTA Jacobi eigensolve;
 * U = V Z; multipliers e, ebar from (mu, rho, lambda).  V0 is the basis currently in the ctx
 * (seed it with gf8_set_basis; the library holds no RNG).  GF8_ERR_BAD_STATE without a factor or
 * a start basis. */
gf8_status gf8_refresh_basis(gf8_ctx* ctx, int layer, int n_iter, void* stream);

/* ---- codec (every step) -------------------------------------------------------------------------- */
/* a3-a6.  codes[m*n], scale_inv[n_scales] <- FP8 payload of the whitened gradient. */
gf8_status gf8_encode(gf8_ctx* ctx, int layer, const void* grad, gf8_dtype dt, uint8_t* codes,
                      float* scale_inv, void* stream);
/* f1.  gf8_encode with ERROR FEEDBACK in the transformed coordinates (PAPER.md:318 Algorithm 1 l.11-15; :354):
 *   U~ = U + R;  s = Scale(U~);  codes = Q(U~; s);  R <- U~ - Dequantize(codes; s)
 * U is the whitened gradient (the gradient itself for a GF8_SIDE_NONE layer).  resid: DEVICE, FP32, gf8_resid_size()
 * floats, 16-byte aligned, caller-owned, one buffer per (tensor, rank); zero it before the first step; it is read and
 * overwritten and is OPAQUE state: FAST contexts keep the residual of a whitened tensor-core layer (BF16 gradients) in the
 * tile order of the update epilogue, into which the feedback is fused; every other case is row-major.  gf8_resid_export
 * writes it out row-major [d_out][d_in] (out: DEVICE, d_out*d_in floats; dt = the gradients' type the buffer was used with).
 * Every element is one IEEE FP32 add, multiply, cast, multiply and subtract: on the same U the codes, scales and residual are
 * bit-identical to oracle O8.  With resid == 0 the payload equals gf8_encode's. */
gf8_status gf8_resid_size(gf8_ctx* ctx, int layer, size_t* n_floats);
gf8_status gf8_resid_export(gf8_ctx* ctx, int layer, gf8_dtype dt, const float* resid, float* out, void* stream);
gf8_status gf8_encode_ef(gf8_ctx* ctx, int layer, const void* grad, gf8_dtype dt, float* resid, uint8_t* codes,
                         float* scale_inv, void* stream);
/* f2.  Synchronised scales (Algorithm 1 l.4-5 "s <- Scale(Wg); s <- AllReduce_MAX(s)", l.17-19 scale-
 * synchronisation steps): the amax on its own, and the cast with an agreed amax.
 *   gf8_amax: amax_out[n_scales] (DEVICE, FP32) <- amax of the tensor the quantizer would see (the whitened gradient; the
 *             gradient itself for a GF8_SIDE_NONE layer), per tensor or per 128 x 128 block.  The caller takes the maximum
 *             over ranks (its all-reduce) and passes it back as amax_sync.
 *   gf8_encode_scaled: scale = fmax / amax_sync, scale_inv = amax_sync / fmax (the quantizer's rule and degenerate cases),
 *             codes = Q(x * scale); scale_inv[n_scales] is written.  With amax_sync == gf8_amax's output the payload equals
 *             gf8_encode's.
 * f3.  Vulnerability profile: hits (DEVICE, two 64-bit counters, caller-zeroed, may be NULL) accumulates
 *             hits[0] += number of codes equal to +-(largest finite value), hits[1] += number of nonzero inputs whose code
 *             is +-0 or +-(smallest subnormal) -- fused into the cast, no extra pass.  A layer's score is
 *             (hits[0] + hits[1]) / elements averaged over the profiling window (S16). */
gf8_status gf8_amax(gf8_ctx* ctx, int layer, const void* grad, gf8_dtype dt, float* amax_out, void* stream);
gf8_status gf8_encode_scaled(gf8_ctx* ctx, int layer, const void* grad, gf8_dtype dt, const float* amax_sync,
                             uint8_t* codes, float* scale_inv, unsigned long long* hits, void* stream);
/* R = 1 case of gf8_reduce_decoded without averaging. */
gf8_status gf8_decode(gf8_ctx* ctx, int layer, const uint8_t* codes, const float* scale_inv,
                      void* grad_out, gf8_dtype dt, void* stream);
/* a7-a8.  U^ = (1/R) sum_r val(codes_r) * scale_inv_r in FP32, rank order, fused multiply-add
 * (standing in for the all-reduce, S8), then unwhiten.  codes_host / scale_inv_host
 * are HOST arrays of R device pointers. */
gf8_status gf8_reduce_decoded(gf8_ctx* ctx, int layer, const uint8_t* const* codes_host,
                              const float* const* scale_inv_host, int R, int average, void* grad_out,
                              gf8_dtype dt, void* stream);

/* ---- batched forms: n layers per call, grouped launches (launch granularity) ---------- */
/* layers_host[n]; grads_host / codes_host / scale_inv_host are HOST arrays of n device pointers. */
gf8_status gf8_encode_many(gf8_ctx* ctx, int n, const int* layers_host, const void* const* grads_host,
                           gf8_dtype dt, uint8_t* const* codes_host, float* const* scale_inv_host,
                           void* stream);
/* resid_host: HOST array of n device pointers (see gf8_encode_ef). */
gf8_status gf8_encode_ef_many(gf8_ctx* ctx, int n, const int* layers_host, const void* const* grads_host,
                              gf8_dtype dt, float* const* resid_host, uint8_t* const* codes_host,
                              float* const* scale_inv_host, void* stream);
/* codes_host / scale_inv_host: HOST arrays of n*R device pointers, index [i*R + r]. */
gf8_status gf8_reduce_decoded_many(gf8_ctx* ctx, int n, const int* layers_host,
                                   const uint8_t* const* codes_host, const float* const* scale_inv_host,
                                   int R, int average, void* const* grads_out_host, gf8_dtype dt,
                                   void* stream);
gf8_status gf8_factor_update_many(gf8_ctx* ctx, int n, const int* layers_host, const void* const* acts_host,
                                  const void* const* gouts_host, const int64_t* T_host, gf8_dtype dt,
                                  void* stream);
gf8_status gf8_refresh_basis_many(gf8_ctx* ctx, int n, const int* layers_host, int n_iter, void* stream);

/* ---- end-to-end with HOST buffers (bench.py's e2e leg) ------------------------------------------- */
/* One whole codec step for n layers and R simulated ranks with pinned HOST gradients:
 * H2D of every rank's gradient, encode, reduce_decoded, D2H of the decoded gradients.
 * grads_host_ptrs[i*R + r] -> host buffer of layer i, rank r (dt); out_host_ptrs[i] -> host buffer
 * receiving the decoded gradient (dt).  Staging memory is owned by the ctx (allocated on first use).
 * The call returns after the stream work is enqueued; synchronise the stream before reading. */
gf8_status gf8_step_host(gf8_ctx* ctx, int n, const int* layers_host, const void* const* grads_host_ptrs,
                         int R, int average, void* const* out_host_ptrs, gf8_dtype dt, void* stream);

/* ---- state access: checkpoint, oracle hand-off, parity taps ---------------------------------------- */
/* side: GF8_SIDE_IN (A, d_in) or GF8_SIDE_OUT (Gf, d_out).  f is d x d FP32 row-major (device). */
gf8_status gf8_get_factor(gf8_ctx* ctx, int layer, int side, float* f, void* stream);
gf8_status gf8_set_factor(gf8_ctx* ctx, int layer, int side, const float* f, void* stream);
/* U: d x k FP32 row-major; mu: k Ritz values (descending); rho_host: isotropic tail + lambda.
 * set: mu == NULL installs U as a start basis only (not usable by the codec until refreshed). */
gf8_status gf8_get_basis(gf8_ctx* ctx, int layer, int side, float* U, float* mu, float* rho_host,
                         void* stream);
gf8_status gf8_set_basis(gf8_ctx* ctx, int layer, int side, const float* U, const float* mu, float rho,
                         void* stream);
/* Transform-stage tap (gate G2): out = (float) W~ of one gradient, m x n FP32. */
gf8_status gf8_whiten_f32(gf8_ctx* ctx, int layer, const void* grad, gf8_dtype dt, float* out,
                          void* stream);
/* Quantizer alone (gate G1): codes, scale_inv <- FP32 tensor `in` (m x n). */
gf8_status gf8_quantize_f32(gf8_ctx* ctx, int fmt, int scaling, const float* in, int64_t m, int64_t n,
                            uint8_t* codes, float* scale_inv, void* stream);
/* Reduce alone (gate G4): out (m x n FP32) <- R payloads. */
gf8_status gf8_reduce_f32(gf8_ctx* ctx, int fmt, int scaling, const uint8_t* const* codes_host,
                          const float* const* scale_inv_host, int R, int average, int64_t m, int64_t n,
                          float* out, void* stream);

/* ---- no-allocation entry point ------------------------------------------------------------------------------------- */
/* The quantizer (a5 + a6; gf8_quantize_f32's arithmetic, bit for bit) for callers that cannot call cudaMalloc: code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it.  It takes NO context and calls no cudaMalloc, cudaFree
 * or allocating library routine: the amax words and scales it needs between its kernels live in a static device array of
 * GF8_NOALLOC_MAX_SCALES entries (512 KB, held by every GPU that loads the library until the process exits).
 *   in: DEVICE, m x n FP32 row-major; codes: DEVICE, m*n bytes; scale_inv: DEVICE, 1 float (GF8_SCALE_TENSOR) or
 *   ceil(m/128)*ceil(n/128) floats (GF8_SCALE_BLOCK128); n a multiple of 16; pointers 16-byte aligned.  It runs on the
 *   CURRENT device (cudaSetDevice is the caller's), asynchronously on `stream`.
 *   Limit: at most GF8_NOALLOC_MAX_SCALES scales, i.e. any size with per-tensor scaling and up to 65536 blocks of 128 x 128
 *   (e.g. 32768 x 32768) with per-block scaling; beyond that GF8_ERR_UNSUPPORTED with a message (gf8_noalloc_last_error,
 *   thread-local) and nothing is launched.
 *   Every call on a device shares the one array: calls that OVERLAP on the GPU (different streams, or graph branches
 *   without an edge between them) race on it -- order them on one stream.  The array keeps the previous call's contents;
 *   the call clears what must start at zero itself. */
#define GF8_NOALLOC_MAX_SCALES 65536
gf8_status gf8_quantize_f32_noalloc(int fmt, int scaling, const float* in, int64_t m, int64_t n, uint8_t* codes,
                                    float* scale_inv, void* stream);
const char* gf8_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GF8_H */
