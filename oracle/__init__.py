"""ctypes binding of the CPU oracle (oracle/gf8_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  Nothing under paper_2607_07494_b200/ imports this module and this module
imports nothing from it.  All arithmetic lives in the C++ file; this file marshals numpy arrays.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gf8_oracle.cpp")
_LIB = os.path.join(_HERE, "libgf8_oracle.so")

E4M3, E5M2 = 0, 1
SCALE_TENSOR, SCALE_BLOCK128 = 0, 1


def build(force=False):
    """Compile the oracle with g++ (no -ffast-math, no FMA contraction).

    GF8_ORACLE_SANITIZE=1 builds and loads an AddressSanitizer + UndefinedBehaviorSanitizer copy instead
    (libgf8_oracle_san.so; run python with LD_PRELOAD=$(g++ -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0):
    the hygiene run of profiles/r02_sanitizers.txt."""
    san = os.environ.get("GF8_ORACLE_SANITIZE") == "1"
    out = os.path.join(_HERE, "libgf8_oracle_san.so") if san else _LIB
    if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
        return out
    cmd = ["g++", "-O1" if san else "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math"]
    if san:
        cmd += ["-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]
    subprocess.check_call(cmd + ["-o", out, _SRC])
    return out


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _declare(_lib)
    return _lib


_pd = C.POINTER(C.c_double)
_pf = C.POINTER(C.c_float)
_pb = C.POINTER(C.c_uint8)
_ph = C.POINTER(C.c_uint16)
_i64 = C.c_int64


def _declare(L):
    L.gf8o_fp8_max.restype = C.c_double
    L.gf8o_fp8_max.argtypes = [C.c_int]
    L.gf8o_fp8_to_double.restype = C.c_double
    L.gf8o_fp8_to_double.argtypes = [C.c_int, C.c_uint8]
    L.gf8o_fp8_from_float.restype = C.c_uint8
    L.gf8o_fp8_from_float.argtypes = [C.c_int, C.c_float]
    L.gf8o_quantize.argtypes = [C.c_int, C.c_int, _pf, _i64, _i64, _pb, _pf]
    L.gf8o_amax.argtypes = [C.c_int, _pf, _i64, _i64, _pf]
    L.gf8o_quantize_scaled.argtypes = [C.c_int, C.c_int, _pf, _i64, _i64, _pf, _pb, _pf, C.POINTER(C.c_uint64)]
    L.gf8o_ef_quantize.argtypes = [C.c_int, C.c_int, _pf, _pf, _i64, _i64, _pb, _pf]
    L.gf8o_reduce.argtypes = [C.c_int, C.c_int, C.POINTER(_pb), C.POINTER(_pf), C.c_int, C.c_int,
                              _i64, _i64, _pf]
    L.gf8o_factor_accumulate.argtypes = [_pd, C.c_int, C.c_double, _pd, _i64, _i64]
    L.gf8o_jacobi_eig.argtypes = [_pd, C.c_int, _pd, _pd]
    L.gf8o_multipliers.argtypes = [_pd, C.c_int, _i64, C.c_double, C.c_double, _pd, _pd, _pd]
    L.gf8o_refresh_basis.argtypes = [_pd, _i64, C.c_int, _pd, C.c_int, C.c_double, _pd, _pd, _pd, _pd, _pd]
    L.gf8o_brute_basis.argtypes = [_pd, _i64, C.c_int, C.c_double, _pd, _pd, _pd, _pd, _pd]
    L.gf8o_build_T.argtypes = [_pd, _pd, _i64, C.c_int, _pd]
    L.gf8o_whiten_dense.argtypes = [_pd, _i64, _i64, _pd, _pd, _pd]
    L.gf8o_whiten_lowrank.argtypes = [_pd, _i64, _i64, _pd, _pd, C.c_int, _pd, _pd, C.c_int, _pd]
    L.gf8o_to_bf16.argtypes = [_pd, _i64, _ph]
    L.gf8o_from_bf16.argtypes = [_ph, _i64, _pd]
    L.gf8o_to_f32.argtypes = [_pd, _i64, _pf]
    L.gf8o_metrics.argtypes = [_pd, _pd, _i64, _pd]
    _pi = C.POINTER(C.c_int64)
    L.gf8o_factor_entries.argtypes = [_pd, _i64, _i64, _pi, _pi, _i64, _pd]
    L.gf8o_whiten_samples.argtypes = [_pd, _i64, _i64, _pd, _pd, C.c_int, _pd, _pd, C.c_int, _pi, _pi, _i64, _pd]
    L.gf8o_set_num_threads.argtypes = [C.c_int]
    L.gf8o_num_threads.restype = C.c_int


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t):
    return a.ctypes.data_as(t) if a is not None else None


# ---- FP8 ----------------------------------------------------------------------------------------
def fp8_max(fmt):
    return lib().gf8o_fp8_max(fmt)


def fp8_to_double(fmt, code):
    return lib().gf8o_fp8_to_double(fmt, int(code))


def fp8_from_float(fmt, y):
    return lib().gf8o_fp8_from_float(fmt, float(np.float32(y)))


def fp8_table(fmt):
    return np.array([fp8_to_double(fmt, c) for c in range(256)])


# ---- codec ----------------------------------------------------------------------------------------
def n_scales(scaling, m, n):
    return 1 if scaling == SCALE_TENSOR else ((m + 127) // 128) * ((n + 127) // 128)


def quantize(x_f32, fmt=E4M3, scaling=SCALE_TENSOR):
    """x_f32: (m, n) float32 -> (codes uint8 (m, n), scale_inv float32 (n_scales,))."""
    x = np.ascontiguousarray(x_f32, dtype=np.float32)
    m, n = x.shape
    codes = np.empty((m, n), dtype=np.uint8)
    sinv = np.empty(n_scales(scaling, m, n), dtype=np.float32)
    lib().gf8o_quantize(fmt, scaling, _p(x, _pf), m, n, _p(codes, _pb), _p(sinv, _pf))
    return codes, sinv


def amax(x_f32, scaling=SCALE_TENSOR):
    """O9: amax per tensor / per 128 x 128 block (bit-pattern maximum of |x|)."""
    x = np.ascontiguousarray(x_f32, dtype=np.float32)
    m, n = x.shape
    out = np.empty(n_scales(scaling, m, n), np.float32)
    lib().gf8o_amax(scaling, _p(x, _pf), m, n, _p(out, _pf))
    return out


def quantize_scaled(x_f32, amax_sync, fmt=E4M3, scaling=SCALE_TENSOR):
    """O9: cast with an externally agreed amax.  Returns (codes, scale_inv, (upper hits, lower hits))."""
    x = np.ascontiguousarray(x_f32, dtype=np.float32)
    m, n = x.shape
    a = np.ascontiguousarray(amax_sync, dtype=np.float32)
    assert a.shape == (n_scales(scaling, m, n),)
    codes = np.empty((m, n), np.uint8)
    sinv = np.empty_like(a)
    hits = (C.c_uint64 * 2)()
    lib().gf8o_quantize_scaled(fmt, scaling, _p(x, _pf), m, n, _p(a, _pf), _p(codes, _pb), _p(sinv, _pf), hits)
    return codes, sinv, (int(hits[0]), int(hits[1]))


def ef_quantize(u_f32, resid_f32, fmt=E4M3, scaling=SCALE_TENSOR):
    """O8: error-feedback quantizer.  Returns (codes, scale_inv, new residual); the inputs are not modified."""
    u = np.ascontiguousarray(u_f32, dtype=np.float32)
    r = np.array(resid_f32, dtype=np.float32, order="C", copy=True)
    assert u.ndim == 2 and r.shape == u.shape
    m, n = u.shape
    codes = np.empty((m, n), np.uint8)
    sinv = np.empty(n_scales(scaling, m, n), np.float32)
    lib().gf8o_ef_quantize(fmt, scaling, _p(u, _pf), _p(r, _pf), m, n, _p(codes, _pb), _p(sinv, _pf))
    return codes, sinv, r


def reduce(codes_list, sinv_list, fmt=E4M3, scaling=SCALE_TENSOR, average=True):
    """R payloads -> FP32 (m, n): fmaf in rank order, then * (1/R)."""
    R = len(codes_list)
    cs = [np.ascontiguousarray(c, dtype=np.uint8) for c in codes_list]
    ss = [np.ascontiguousarray(s, dtype=np.float32) for s in sinv_list]
    m, n = cs[0].shape
    cp = (_pb * R)(*[_p(c, _pb) for c in cs])
    sp = (_pf * R)(*[_p(s, _pf) for s in ss])
    out = np.empty((m, n), dtype=np.float32)
    lib().gf8o_reduce(fmt, scaling, cp, sp, R, 1 if average else 0, m, n, _p(out, _pf))
    return out


# ---- geometry state -------------------------------------------------------------------------------
def factor_accumulate(X, A=None, beta=0.0):
    """O1: returns the updated d x d factor (float64).  A=None means first call."""
    X = _d(X)
    T, d = X.shape
    first = A is None
    A = np.zeros((d, d)) if first else _d(A).copy()
    lib().gf8o_factor_accumulate(_p(A, _pd), 1 if first else 0, float(beta), _p(X, _pd), T, d)
    return A


def jacobi_eig(B):
    B = _d(B)
    n = B.shape[0]
    Z = np.empty((n, n))
    M = np.empty(n)
    lib().gf8o_jacobi_eig(_p(B, _pd), n, _p(Z, _pd), _p(M, _pd))
    return M, Z


def multipliers(mu, d, trace, lam):
    mu = _d(mu)
    k = mu.shape[0]
    rho = C.c_double()
    e = np.empty(k)
    eb = np.empty(k)
    lib().gf8o_multipliers(_p(mu, _pd), k, d, float(trace), float(lam), C.byref(rho), _p(e, _pd), _p(eb, _pd))
    return rho.value, e, eb


class Basis:
    """U (d, k), mu (k,), rho, e (k,), ebar (k,) -- all float64."""

    def __init__(self, U, mu, rho, e, ebar):
        self.U, self.mu, self.rho, self.e, self.ebar = U, mu, rho, e, ebar

    @property
    def k(self):
        return self.U.shape[1]


def refresh_basis(A, V0, q, lam):
    A = _d(A)
    V0 = _d(V0)
    d, k = V0.shape
    U = np.empty((d, k))
    mu = np.empty(k)
    e = np.empty(k)
    eb = np.empty(k)
    rho = C.c_double()
    lib().gf8o_refresh_basis(_p(A, _pd), d, k, _p(V0, _pd), int(q), float(lam), _p(U, _pd), _p(mu, _pd),
                             C.byref(rho), _p(e, _pd), _p(eb, _pd))
    return Basis(U, mu, rho.value, e, eb)


def brute_basis(A, k, lam):
    A = _d(A)
    d = A.shape[0]
    U = np.empty((d, k))
    mu = np.empty(k)
    e = np.empty(k)
    eb = np.empty(k)
    rho = C.c_double()
    lib().gf8o_brute_basis(_p(A, _pd), d, k, float(lam), _p(U, _pd), _p(mu, _pd), C.byref(rho),
                           _p(e, _pd), _p(eb, _pd))
    return Basis(U, mu, rho.value, e, eb)


def build_T(U, e):
    U = _d(U)
    e = _d(e)
    d, k = U.shape
    T = np.empty((d, d))
    lib().gf8o_build_T(_p(U, _pd), _p(e, _pd), d, k, _p(T, _pd))
    return T


# ---- transform ------------------------------------------------------------------------------------
def whiten_dense(W, TG=None, TA=None):
    W = _d(W)
    m, n = W.shape
    TG = _d(TG) if TG is not None else None
    TA = _d(TA) if TA is not None else None
    out = np.empty((m, n))
    lib().gf8o_whiten_dense(_p(W, _pd), m, n, _p(TG, _pd), _p(TA, _pd), _p(out, _pd))
    return out


def whiten_lowrank(W, UG=None, eG=None, UA=None, eA=None):
    """O3 (with e) / O6 (with ebar).  Sides are switched off by passing None."""
    W = _d(W)
    m, n = W.shape
    kG = kA = 0
    if UG is not None:
        UG, eG = _d(UG), _d(eG)
        kG = UG.shape[1]
    if UA is not None:
        UA, eA = _d(UA), _d(eA)
        kA = UA.shape[1]
    out = np.empty((m, n))
    lib().gf8o_whiten_lowrank(_p(W, _pd), m, n, _p(UG, _pd), _p(eG, _pd), kG, _p(UA, _pd), _p(eA, _pd), kA,
                              _p(out, _pd))
    return out


# ---- sampled outputs (full-size parity: one output element at a time, by its plain definition) ----
def _idx(a):
    return np.ascontiguousarray(a, dtype=np.int64)


def factor_entries(X, ii, jj):
    """O1 at sampled (i, j): A[i][j] = mean_t x_t[i] x_t[j] (no EMA)."""
    X = _d(X)
    T, d = X.shape
    ii, jj = _idx(ii), _idx(jj)
    out = np.empty(ii.shape[0])
    pi = C.POINTER(C.c_int64)
    lib().gf8o_factor_entries(_p(X, _pd), T, d, ii.ctypes.data_as(pi), jj.ctypes.data_as(pi), ii.shape[0], _p(out, _pd))
    return out


def whiten_samples(W, ii, jj, UG=None, eG=None, UA=None, eA=None):
    """O3 (with e) / O6 (with ebar) at sampled (i, j), dense form of Eq. 14 / 17."""
    W = _d(W)
    m, n = W.shape
    kG = kA = 0
    if UG is not None:
        UG, eG = _d(UG), _d(eG)
        kG = UG.shape[1]
    if UA is not None:
        UA, eA = _d(UA), _d(eA)
        kA = UA.shape[1]
    ii, jj = _idx(ii), _idx(jj)
    out = np.empty(ii.shape[0])
    pi = C.POINTER(C.c_int64)
    lib().gf8o_whiten_samples(_p(W, _pd), m, n, _p(UG, _pd), _p(eG, _pd), kG, _p(UA, _pd), _p(eA, _pd), kA,
                              ii.ctypes.data_as(pi), jj.ctypes.data_as(pi), ii.shape[0], _p(out, _pd))
    return out


# ---- conversions / metrics -----------------------------------------------------------------------
def to_bf16_bits(x):
    x = _d(x)
    out = np.empty(x.shape, dtype=np.uint16)
    lib().gf8o_to_bf16(_p(x, _pd), x.size, _p(out, _ph))
    return out


def from_bf16_bits(b):
    b = np.ascontiguousarray(b, dtype=np.uint16)
    out = np.empty(b.shape)
    lib().gf8o_from_bf16(_p(b, _ph), b.size, _p(out, _pd))
    return out


def to_f32(x):
    x = _d(x)
    out = np.empty(x.shape, dtype=np.float32)
    lib().gf8o_to_f32(_p(x, _pd), x.size, _p(out, _pf))
    return out


def metrics(ghat, g):
    """Eq. 21: dict(RelL2, Cos, MaxErr, MSE)."""
    a, b = _d(ghat).ravel(), _d(g).ravel()
    out = np.empty(4)
    lib().gf8o_metrics(_p(a, _pd), _p(b, _pd), a.size, _p(out, _pd))
    return dict(RelL2=out[0], Cos=out[1], MaxErr=out[2], MSE=out[3])


def num_threads():
    return lib().gf8o_num_threads()


def set_num_threads(n):
    lib().gf8o_set_num_threads(int(n))


# ---- whole-codec helpers (composition only; every step above is a C++ call) -----------------------
def encode(W, basisG=None, basisA=None, fmt=E4M3, scaling=SCALE_TENSOR):
    """O3 + O4 on one gradient: returns (codes, scale_inv, wt_f32)."""
    wt = whiten_lowrank(W, basisG.U if basisG else None, basisG.e if basisG else None,
                        basisA.U if basisA else None, basisA.e if basisA else None)
    x = to_f32(wt)
    codes, sinv = quantize(x, fmt, scaling)
    return codes, sinv, x


def encode_ef(W, resid_f32, basisG=None, basisA=None, fmt=E4M3, scaling=SCALE_TENSOR):
    """O3 + O8 on one gradient: returns (codes, scale_inv, new residual, wt_f32)."""
    wt = whiten_lowrank(W, basisG.U if basisG else None, basisG.e if basisG else None,
                        basisA.U if basisA else None, basisA.e if basisA else None)
    x = to_f32(wt)
    codes, sinv, r = ef_quantize(x, resid_f32, fmt, scaling)
    return codes, sinv, r, x


def reduce_decoded(codes_list, sinv_list, basisG=None, basisA=None, fmt=E4M3, scaling=SCALE_TENSOR,
                   average=True):
    """O5 + O6: returns the unwhitened gradient in float64 (caller rounds to FP32 / BF16)."""
    uhat = reduce(codes_list, sinv_list, fmt, scaling, average)
    return whiten_lowrank(uhat, basisG.U if basisG else None, basisG.ebar if basisG else None,
                          basisA.U if basisA else None, basisA.ebar if basisA else None)
