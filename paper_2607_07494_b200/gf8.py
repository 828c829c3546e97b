"""Thin Python binding of the gf8 C ABI (include/gf8.h): argument marshalling only.

Every step of the codec runs in the CUDA kernels of libgf8.so; torch is used for device memory and
streams.  There is no CPU or eager fallback: if libgf8.so is missing or fails, this module raises.
Function and method names mirror the C entry points (gf8_encode -> Ctx.encode, ...).
"""
import ctypes as C
import os
from dataclasses import dataclass
from typing import List, Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgf8.so")

E4M3, E5M2 = 0, 1
SCALE_TENSOR, SCALE_BLOCK128 = 0, 1
SIDE_NONE, SIDE_IN, SIDE_OUT, SIDE_BOTH = 0, 1, 2, 3
DT_BF16, DT_F32 = 0, 1
PREC_EXACT, PREC_FAST = 0, 1
MAX_RANK, MAX_R = 512, 64

EXPORTS = [
    "gf8_create", "gf8_destroy", "gf8_payload_size", "gf8_status_string", "gf8_last_error", "gf8_launch_count",
    "gf8_sync_check", "gf8_set_stage_timing", "gf8_stage_times",
    "gf8_factor_update", "gf8_refresh_basis", "gf8_encode", "gf8_decode", "gf8_reduce_decoded",
    "gf8_encode_many", "gf8_reduce_decoded_many", "gf8_factor_update_many", "gf8_refresh_basis_many",
    "gf8_encode_ef", "gf8_encode_ef_many", "gf8_resid_size", "gf8_resid_export", "gf8_amax", "gf8_encode_scaled",
    "gf8_step_host", "gf8_get_factor", "gf8_set_factor", "gf8_get_basis", "gf8_set_basis",
    "gf8_whiten_f32", "gf8_quantize_f32", "gf8_reduce_f32",
    "gf8_quantize_f32_noalloc", "gf8_noalloc_last_error",
]


class LayerDesc(C.Structure):
    _fields_ = [("d_out", C.c_int32), ("d_in", C.c_int32), ("rank_in", C.c_int32), ("rank_out", C.c_int32),
                ("side", C.c_int32), ("fmt", C.c_int32), ("scaling", C.c_int32), ("damping", C.c_float),
                ("ema_beta", C.c_float)]


@dataclass
class Layer:
    d_out: int
    d_in: int
    side: int = SIDE_BOTH
    rank_in: int = 0
    rank_out: int = 0
    fmt: int = E4M3
    scaling: int = SCALE_TENSOR
    damping: float = 1e-3
    ema_beta: float = 0.0

    def n_scales(self):
        return 1 if self.scaling == SCALE_TENSOR else ((self.d_out + 127) // 128) * ((self.d_in + 127) // 128)


class Gf8Error(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"gf8 status {status}: {msg}")
        self.status = status


_lib = None


def lib():
    """Load libgf8.so.  Fails loudly when the CUDA library has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2607_07494_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int, C.c_int64
        L.gf8_create.argtypes = [C.POINTER(vp), i32, C.POINTER(LayerDesc), i32, i32]
        L.gf8_destroy.argtypes = [vp]
        L.gf8_payload_size.argtypes = [vp, i32, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
        L.gf8_status_string.restype = C.c_char_p
        L.gf8_status_string.argtypes = [i32]
        L.gf8_last_error.restype = C.c_char_p
        L.gf8_last_error.argtypes = [vp]
        L.gf8_launch_count.restype = i64
        L.gf8_launch_count.argtypes = [vp]
        L.gf8_sync_check.argtypes = [vp, vp]
        L.gf8_set_stage_timing.argtypes = [vp, i32]
        L.gf8_stage_times.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(i32), vp]
        L.gf8_factor_update.argtypes = [vp, i32, vp, vp, i64, i32, vp]
        L.gf8_refresh_basis.argtypes = [vp, i32, i32, vp]
        L.gf8_encode.argtypes = [vp, i32, vp, i32, vp, vp, vp]
        L.gf8_decode.argtypes = [vp, i32, vp, vp, vp, i32, vp]
        L.gf8_reduce_decoded.argtypes = [vp, i32, C.POINTER(vp), C.POINTER(vp), i32, i32, vp, i32, vp]
        L.gf8_encode_many.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(vp), i32, C.POINTER(vp), C.POINTER(vp), vp]
        L.gf8_amax.argtypes = [vp, i32, vp, i32, vp, vp]
        L.gf8_encode_scaled.argtypes = [vp, i32, vp, i32, vp, vp, vp, vp, vp]
        L.gf8_resid_size.argtypes = [vp, i32, C.POINTER(C.c_size_t)]
        L.gf8_resid_export.argtypes = [vp, i32, i32, vp, vp, vp]
        L.gf8_encode_ef.argtypes = [vp, i32, vp, i32, vp, vp, vp, vp]
        L.gf8_encode_ef_many.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(vp), i32, C.POINTER(vp), C.POINTER(vp),
                                         C.POINTER(vp), vp]
        L.gf8_reduce_decoded_many.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(vp), C.POINTER(vp), i32, i32,
                                              C.POINTER(vp), i32, vp]
        L.gf8_factor_update_many.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(vp), C.POINTER(vp), C.POINTER(i64),
                                             i32, vp]
        L.gf8_refresh_basis_many.argtypes = [vp, i32, C.POINTER(i32), i32, vp]
        L.gf8_step_host.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(vp), i32, i32, C.POINTER(vp), i32, vp]
        L.gf8_get_factor.argtypes = [vp, i32, i32, vp, vp]
        L.gf8_set_factor.argtypes = [vp, i32, i32, vp, vp]
        L.gf8_get_basis.argtypes = [vp, i32, i32, vp, vp, C.POINTER(C.c_float), vp]
        L.gf8_set_basis.argtypes = [vp, i32, i32, vp, vp, C.c_float, vp]
        L.gf8_whiten_f32.argtypes = [vp, i32, vp, i32, vp, vp]
        L.gf8_quantize_f32.argtypes = [vp, i32, i32, vp, i64, i64, vp, vp, vp]
        L.gf8_reduce_f32.argtypes = [vp, i32, i32, C.POINTER(vp), C.POINTER(vp), i32, i32, i64, i64, vp, vp]
        L.gf8_quantize_f32_noalloc.argtypes = [i32, i32, vp, i64, i64, vp, vp, vp]
        L.gf8_noalloc_last_error.restype = C.c_char_p
        L.gf8_noalloc_last_error.argtypes = []
        for name in EXPORTS:
            if name not in ("gf8_status_string", "gf8_last_error", "gf8_launch_count", "gf8_noalloc_last_error"):
                getattr(L, name).restype = i32
        _lib = L
    return _lib


def _dt(t: torch.Tensor) -> int:
    if t.dtype == torch.bfloat16:
        return DT_BF16
    if t.dtype == torch.float32:
        return DT_F32
    raise TypeError(f"gf8 takes bfloat16 or float32 gradients, got {t.dtype}")


def _tdt(dt: int):
    return torch.bfloat16 if dt == DT_BF16 else torch.float32


def _ptr(t: Optional[torch.Tensor]):
    if t is None:
        return None
    assert t.is_contiguous(), "gf8 takes contiguous row-major tensors"
    return C.c_void_p(t.data_ptr())


def _ptr_array(ts):
    """ctypes array of device (or host) pointers; an array made earlier by ptr_array() passes through, so a
    training loop that reuses its buffers marshals them once."""
    if isinstance(ts, C.Array):
        return ts
    arr = (C.c_void_p * len(ts))()
    for i, t in enumerate(ts):
        arr[i] = None if t is None else t.data_ptr()
    return arr


def ptr_array(ts: Sequence[Optional[torch.Tensor]]):
    for t in ts:
        assert t is None or t.is_contiguous(), "gf8 takes contiguous row-major tensors"
    return _ptr_array(list(ts))


def int_array(xs):
    return xs if isinstance(xs, C.Array) else (C.c_int * len(xs))(*xs)


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Ctx:
    """gf8_ctx: owns factors, bases, multipliers and scratch of a set of gradient matrices."""

    def __init__(self, layers: List[Layer], precision: int = PREC_EXACT, device: Optional[int] = None):
        L = lib()
        if not torch.cuda.is_available():
            raise RuntimeError("gf8 needs a CUDA device (no CPU fallback)")
        self.device = torch.cuda.current_device() if device is None else int(device)
        self.layers = list(layers)
        self.precision = precision
        descs = (LayerDesc * len(layers))()
        for i, l in enumerate(layers):
            descs[i] = LayerDesc(l.d_out, l.d_in, l.rank_in, l.rank_out, l.side, l.fmt, l.scaling, l.damping, l.ema_beta)
        self._h = C.c_void_p()
        st = L.gf8_create(C.byref(self._h), self.device, descs, len(layers), precision)
        if st != 0:
            self._h = C.c_void_p()
            raise Gf8Error(st, L.gf8_status_string(st).decode())
        self._tdev = torch.device("cuda", self.device)

    def _ck(self, st):
        if st != 0:
            raise Gf8Error(st, lib().gf8_last_error(self._h).decode() or lib().gf8_status_string(st).decode())

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().gf8_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def set_stage_timing(self, enable=True):
        self._ck(lib().gf8_set_stage_timing(self._h, 1 if enable else 0))

    def stage_times(self):
        """(ms[8], launches[8]) of the tensor-core stages since the last call (synchronises the stream)."""
        ms, n = (C.c_float * 8)(), (C.c_int * 8)()
        self._ck(lib().gf8_stage_times(self._h, ms, n, _stream()))
        return list(ms), list(n)

    def launch_count(self) -> int:
        return int(lib().gf8_launch_count(self._h))

    def sync_check(self):
        """Synchronise the current stream and raise if a kernel reported an asynchronous failure."""
        self._ck(lib().gf8_sync_check(self._h, _stream()))

    def payload_size(self, layer):
        a, b = C.c_size_t(), C.c_size_t()
        st = lib().gf8_payload_size(self._h, layer, C.byref(a), C.byref(b))
        if st != 0:
            raise Gf8Error(st, f"layer {layer} out of range")
        return a.value, b.value

    def _payload_buffers(self, layer):
        self.payload_size(layer)                       # range check is the library's (GF8_ERR_INVALID_ARG)
        l = self.layers[layer]
        return (torch.empty((l.d_out, l.d_in), dtype=torch.uint8, device=self._tdev),
                torch.empty((l.n_scales(),), dtype=torch.float32, device=self._tdev))

    # ---- geometry state -------------------------------------------------------------------------
    def factor_update(self, layer, act: Optional[torch.Tensor], gout: Optional[torch.Tensor]):
        ref = act if act is not None else gout
        T = ref.shape[0]
        self._ck(lib().gf8_factor_update(self._h, layer, _ptr(act), _ptr(gout), T, _dt(ref), _stream()))

    def refresh_basis(self, layer, n_iter: int):
        self._ck(lib().gf8_refresh_basis(self._h, layer, n_iter, _stream()))

    def factor_update_many(self, layers, acts, gouts):
        n = len(layers)
        ref = next(t for t in list(acts) + list(gouts) if t is not None)
        Ts = (C.c_int64 * n)(*[(a if a is not None else g).shape[0] for a, g in zip(acts, gouts)])
        self._ck(lib().gf8_factor_update_many(self._h, n, (C.c_int * n)(*layers), _ptr_array(acts), _ptr_array(gouts),
                                              Ts, _dt(ref), _stream()))

    def refresh_basis_many(self, layers, n_iter):
        n = len(layers)
        self._ck(lib().gf8_refresh_basis_many(self._h, n, (C.c_int * n)(*layers), n_iter, _stream()))

    # ---- codec -------------------------------------------------------------------------------------
    def encode(self, layer, grad: torch.Tensor, codes=None, scale_inv=None):
        if codes is None:
            codes, scale_inv = self._payload_buffers(layer)
        self._ck(lib().gf8_encode(self._h, layer, _ptr(grad), _dt(grad), _ptr(codes), _ptr(scale_inv), _stream()))
        return codes, scale_inv

    def decode(self, layer, codes, scale_inv, out=None, dt=DT_BF16):
        l = self.layers[layer]
        if out is None:
            out = torch.empty((l.d_out, l.d_in), dtype=_tdt(dt), device=self._tdev)
        self._ck(lib().gf8_decode(self._h, layer, _ptr(codes), _ptr(scale_inv), _ptr(out), _dt(out), _stream()))
        return out

    def reduce_decoded(self, layer, codes_list, scale_inv_list, average=True, out=None, dt=DT_BF16):
        l = self.layers[layer]
        R = len(codes_list)
        if out is None:
            out = torch.empty((l.d_out, l.d_in), dtype=_tdt(dt), device=self._tdev)
        self._ck(lib().gf8_reduce_decoded(self._h, layer, _ptr_array(codes_list), _ptr_array(scale_inv_list), R,
                                          1 if average else 0, _ptr(out), _dt(out), _stream()))
        return out

    def encode_many(self, layers, grads, codes, scale_invs, dt=None):
        n = len(layers)
        dt = dt if dt is not None else _dt(grads[0])
        self._ck(lib().gf8_encode_many(self._h, n, int_array(layers), _ptr_array(grads), dt,
                                       _ptr_array(codes), _ptr_array(scale_invs), _stream()))

    def amax(self, layer, grad: torch.Tensor):
        """f2: amax (per tensor / per block) of what the quantizer would see for this gradient."""
        out = torch.empty(self.layers[layer].n_scales(), dtype=torch.float32, device=self._tdev)
        self._ck(lib().gf8_amax(self._h, layer, _ptr(grad), _dt(grad), _ptr(out), _stream()))
        return out

    def encode_scaled(self, layer, grad: torch.Tensor, amax_sync: torch.Tensor, hits: Optional[torch.Tensor] = None):
        """f2 / f3: cast with an agreed amax; `hits` (int64[2] on the device, accumulated) counts upper / lower boundary hits."""
        codes, scale_inv = self._payload_buffers(layer)
        assert amax_sync.dtype == torch.float32 and amax_sync.numel() == self.layers[layer].n_scales()
        assert hits is None or (hits.dtype == torch.int64 and hits.numel() == 2)
        self._ck(lib().gf8_encode_scaled(self._h, layer, _ptr(grad), _dt(grad), _ptr(amax_sync), _ptr(codes), _ptr(scale_inv),
                                         _ptr(hits), _stream()))
        return codes, scale_inv

    def resid_new(self, layer):
        """A zeroed error-feedback residual for `layer` (opaque FP32 state, gf8_resid_size floats)."""
        n = C.c_size_t()
        self._ck(lib().gf8_resid_size(self._h, layer, C.byref(n)))
        return torch.zeros(n.value, dtype=torch.float32, device=self._tdev)

    def resid_export(self, layer, resid: torch.Tensor, dt=DT_BF16):
        """The residual as a row-major [d_out][d_in] FP32 tensor (dt: the gradient type the buffer was used with)."""
        l = self.layers[layer]
        out = torch.empty((l.d_out, l.d_in), dtype=torch.float32, device=self._tdev)
        self._ck(lib().gf8_resid_export(self._h, layer, dt, _ptr(resid), _ptr(out), _stream()))
        return out

    def encode_ef(self, layer, grad: torch.Tensor, resid: torch.Tensor, codes=None, scale_inv=None):
        """f1: encode with error feedback; `resid` (from resid_new) is read and overwritten."""
        assert resid.dtype == torch.float32
        if codes is None:
            codes, scale_inv = self._payload_buffers(layer)
        self._ck(lib().gf8_encode_ef(self._h, layer, _ptr(grad), _dt(grad), _ptr(resid), _ptr(codes), _ptr(scale_inv),
                                     _stream()))
        return codes, scale_inv

    def encode_ef_many(self, layers, grads, resids, codes, scale_invs, dt=None):
        n = len(layers)
        dt = dt if dt is not None else _dt(grads[0])
        self._ck(lib().gf8_encode_ef_many(self._h, n, int_array(layers), _ptr_array(grads), dt, _ptr_array(resids),
                                          _ptr_array(codes), _ptr_array(scale_invs), _stream()))

    def reduce_decoded_many(self, layers, codes, scale_invs, R, outs, average=True, dt=None):
        """codes / scale_invs: flat lists of n*R tensors, index [i*R + r]."""
        n = len(layers)
        dt = dt if dt is not None else _dt(outs[0])
        self._ck(lib().gf8_reduce_decoded_many(self._h, n, int_array(layers), _ptr_array(codes),
                                               _ptr_array(scale_invs), R, 1 if average else 0, _ptr_array(outs),
                                               dt, _stream()))

    def step_host(self, layers, grads_host, R, outs_host, average=True):
        """grads_host: flat list of n*R pinned CPU tensors [i*R + r]; outs_host: n pinned CPU tensors."""
        n = len(layers)
        for t in list(grads_host) + list(outs_host):
            assert t.device.type == "cpu" and t.is_contiguous()
        self._ck(lib().gf8_step_host(self._h, n, (C.c_int * n)(*layers), _ptr_array(grads_host), R,
                                     1 if average else 0, _ptr_array(outs_host), _dt(outs_host[0]), _stream()))

    # ---- state access ------------------------------------------------------------------------------
    def _side_dim(self, layer, side):
        l = self.layers[layer]
        return (l.d_in, l.rank_in) if side == SIDE_IN else (l.d_out, l.rank_out)

    def get_factor(self, layer, side):
        d, _ = self._side_dim(layer, side)
        f = torch.empty((d, d), dtype=torch.float32, device=self._tdev)
        self._ck(lib().gf8_get_factor(self._h, layer, side, _ptr(f), _stream()))
        return f

    def set_factor(self, layer, side, f: torch.Tensor):
        assert f.dtype == torch.float32
        self._ck(lib().gf8_set_factor(self._h, layer, side, _ptr(f), _stream()))

    def get_basis(self, layer, side):
        d, k = self._side_dim(layer, side)
        U = torch.empty((d, k), dtype=torch.float32, device=self._tdev)
        mu = torch.empty((k,), dtype=torch.float32, device=self._tdev)
        rho = C.c_float()
        self._ck(lib().gf8_get_basis(self._h, layer, side, _ptr(U), _ptr(mu), C.byref(rho), _stream()))
        return U, mu, rho.value

    def set_basis(self, layer, side, U: torch.Tensor, mu: Optional[torch.Tensor] = None, rho: float = 0.0):
        assert U.dtype == torch.float32 and (mu is None or mu.dtype == torch.float32)
        self._ck(lib().gf8_set_basis(self._h, layer, side, _ptr(U), _ptr(mu), float(rho), _stream()))

    def whiten_f32(self, layer, grad):
        l = self.layers[layer]
        out = torch.empty((l.d_out, l.d_in), dtype=torch.float32, device=self._tdev)
        self._ck(lib().gf8_whiten_f32(self._h, layer, _ptr(grad), _dt(grad), _ptr(out), _stream()))
        return out

    def quantize_f32(self, x: torch.Tensor, fmt=E4M3, scaling=SCALE_TENSOR):
        assert x.dtype == torch.float32 and x.dim() == 2
        m, n = x.shape
        ns = 1 if scaling == SCALE_TENSOR else ((m + 127) // 128) * ((n + 127) // 128)
        codes = torch.empty((m, n), dtype=torch.uint8, device=self._tdev)
        sinv = torch.empty((ns,), dtype=torch.float32, device=self._tdev)
        self._ck(lib().gf8_quantize_f32(self._h, fmt, scaling, _ptr(x), m, n, _ptr(codes), _ptr(sinv), _stream()))
        return codes, sinv

    def reduce_f32(self, codes_list, scale_inv_list, fmt=E4M3, scaling=SCALE_TENSOR, average=True):
        R = len(codes_list)
        m, n = codes_list[0].shape
        out = torch.empty((m, n), dtype=torch.float32, device=self._tdev)
        self._ck(lib().gf8_reduce_f32(self._h, fmt, scaling, _ptr_array(codes_list), _ptr_array(scale_inv_list), R,
                                      1 if average else 0, m, n, _ptr(out), _stream()))
        return out


def create(layers: List[Layer], precision: int = PREC_EXACT, device: Optional[int] = None) -> Ctx:
    return Ctx(layers, precision, device)


def quantize_f32_noalloc(x: torch.Tensor, codes: torch.Tensor, scale_inv: torch.Tensor, fmt=E4M3, scaling=SCALE_TENSOR):
    """gf8_quantize_f32_noalloc: the quantizer without a context and without any allocation (static device scratch);
    the caller passes the output buffers.  Runs on x's device, on torch's current stream."""
    assert x.dtype == torch.float32 and x.dim() == 2 and x.is_cuda and codes.dtype == torch.uint8 and scale_inv.dtype == torch.float32
    m, n = x.shape
    with torch.cuda.device(x.device):
        st = lib().gf8_quantize_f32_noalloc(fmt, scaling, _ptr(x), m, n, _ptr(codes), _ptr(scale_inv), _stream())
    if st != 0:
        raise Gf8Error(st, lib().gf8_noalloc_last_error().decode())
    return codes, scale_inv
