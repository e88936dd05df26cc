"""Thin ctypes binding of libsubmatrix.so (include/submatrix.h).

Argument marshalling only: every step of the path (PAPER.md:110 steps 1-3, Eq. 13/14) runs in the
CUDA kernels behind the C ABI.  PyTorch provides device memory and the current stream.  There is no
CPU fallback: if the library cannot be loaded, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from types import SimpleNamespace

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libsubmatrix.so")
if not os.path.exists(_SO):
    raise ImportError(
        f"{_SO} is missing: build it with `python -m paper_2205_14741_b200.build` "
        "(or __graft_entry__.build()); there is no CPU fallback")
_lib = C.CDLL(_SO)

SM_OK, SM_ERR_ARG, SM_ERR_SPACE, SM_ERR_PATTERN, SM_ERR_CUDA, SM_ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5
SM_WARN_NOT_CONVERGED = 1
SM_F64, SM_F32, SM_BF16, SM_F16 = 0, 1, 2, 3
SM_SCALE_NONE, SM_SCALE_GERSHGORIN, SM_SCALE_POWER, SM_SCALE_GLOBAL = 0, 1, 2, 3

DTYPES = {"f64": SM_F64, "f32": SM_F32, "bf16": SM_BF16, "f16": SM_F16}
TORCH_DTYPE = {SM_F64: torch.float64, SM_F32: torch.float32, SM_BF16: torch.bfloat16, SM_F16: torch.float16}
SCALES = {"none": SM_SCALE_NONE, "gershgorin": SM_SCALE_GERSHGORIN, "power": SM_SCALE_POWER, "global": SM_SCALE_GLOBAL}
EXPORTS = ["sm_last_cuda_error", "sm_pattern_sizes", "sm_build_pattern", "sm_plan_columns",
           "sm_gather_ws_bytes", "sm_gather", "sm_sign_ws_bytes", "sm_sign_ns", "sm_sign_status",
           "sm_scatter", "sm_symmetrise", "sm_density_ws_bytes", "sm_density", "sm_density_from_sign",
           "sm_mu_search", "sm_launch_count", "sm_profile_enable", "sm_profile_read", "sm_sign_ws_bytes_ex",
           "sm_sign_ns_ex", "sm_set_option", "sm_get_option", "sm_build_info", "sm_last_device_error",
           "sm_inv_sqrt_ws_bytes", "sm_inv_sqrt", "sm_density_nonorth_ws_bytes", "sm_density_nonorth", "sm_density_ex",
           "sm_density_ws_bytes_ex", "sm_sign_ns_static_capacity", "sm_sign_ns_static"]
SM_SIGN_NONSYMMETRIC, SM_SIGN_ORDER3 = 1, 2      # sm_sign_ns_ex flags


class SmError(RuntimeError):
    def __init__(self, fn, status):
        self.status = status
        extra = (f" (cuda error {_lib.sm_last_cuda_error()}, device protocol code {_lib.sm_last_device_error()})"
                 if status == SM_ERR_CUDA else "")
        super().__init__(f"{fn} returned status {status}{extra}")


class _Bcsr(C.Structure):
    _fields_ = [("n_blk", C.c_int32), ("nnzb", C.c_int32), ("blk_size", C.c_void_p),
                ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p), ("val_ptr", C.c_void_p)]


class _Sizes(C.Structure):
    _fields_ = [("nbr_len", C.c_int64), ("gmap_len", C.c_int64), ("packed_elems", C.c_int64),
                ("build_ws_bytes", C.c_int64), ("max_dim", C.c_int32), ("max_dim_pad", C.c_int32),
                ("max_nbr", C.c_int32), ("reserved", C.c_int32)]


class _Pattern(C.Structure):
    _fields_ = [("n_blk", C.c_int32), ("nnzb", C.c_int32), ("pad_to", C.c_int32), ("max_dim", C.c_int32),
                ("max_dim_pad", C.c_int32), ("max_nbr", C.c_int32), ("packed_elems", C.c_int64),
                ("gmap_len", C.c_int64)] + [(k, C.c_void_p) for k in (
                    "nbr_ptr", "nbr_idx", "own_pos", "dim", "dim_pad", "row_off", "sub_off", "gmap_ptr",
                    "gmap", "tmap", "order")]


_lib.sm_launch_count.restype = C.c_int64
_lib.sm_gather_ws_bytes.restype = C.c_int64
_lib.sm_sign_ws_bytes.restype = C.c_int64
_lib.sm_sign_ws_bytes_ex.restype = C.c_int64
_lib.sm_inv_sqrt_ws_bytes.restype = C.c_int64
_lib.sm_density_nonorth_ws_bytes.restype = C.c_int64
_lib.sm_density_ws_bytes.restype = C.c_int64
_lib.sm_density_ws_bytes_ex.restype = C.c_int64
_lib.sm_sign_ns_static_capacity.restype = C.c_int64


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _check(fn, status, allow_warn=False):
    if status < 0 or (status > 0 and not allow_warn):
        raise SmError(fn, status)
    return status


def set_option(name: str, value: int) -> None:
    _check("sm_set_option", _lib.sm_set_option(C.c_char_p(name.encode()), C.c_int32(int(value))))


def get_option(name: str) -> int:
    v = C.c_int32(0)
    _check("sm_get_option", _lib.sm_get_option(C.c_char_p(name.encode()), C.byref(v)))
    return int(v.value)


def build_info() -> int:
    return int(_lib.sm_build_info())


def last_device_error() -> int:
    return int(_lib.sm_last_device_error())


def launch_count() -> int:
    return int(_lib.sm_launch_count())


def profile_enable(on: bool) -> None:
    _check("sm_profile_enable", _lib.sm_profile_enable(C.c_int32(1 if on else 0)))


def profile_read():
    """(summed duration in ms, number of launches) of the tensor-core NS kernel since enable/read."""
    ms, n = C.c_double(0.0), C.c_int64(0)
    _check("sm_profile_read", _lib.sm_profile_read(C.byref(ms), C.byref(n)))
    return ms.value, int(n.value)


class Bcsr:
    """Device copy of a block-CSR pattern (+ optional values)."""

    def __init__(self, wl, device="cuda", val_dtype="f64"):
        dev = torch.device(device)
        self.n_blk, self.nnzb = int(wl.n_blk), int(wl.nnzb)
        self.blk_size = torch.as_tensor(np.ascontiguousarray(wl.blk_size, dtype=np.int32), device=dev)
        self.row_ptr = torch.as_tensor(np.ascontiguousarray(wl.row_ptr, dtype=np.int32), device=dev)
        self.col_idx = torch.as_tensor(np.ascontiguousarray(wl.col_idx, dtype=np.int32), device=dev)
        self.val_ptr = torch.as_tensor(np.ascontiguousarray(wl.val_ptr, dtype=np.int64), device=dev)
        self.n_vals = int(wl.val_ptr[-1])
        self.val_dtype = DTYPES[val_dtype]
        self.vals = None
        if getattr(wl, "vals", None) is not None:
            self.vals = torch.as_tensor(np.ascontiguousarray(wl.vals), device=dev).to(TORCH_DTYPE[self.val_dtype])
        self.c = _Bcsr(self.n_blk, self.nnzb, self.blk_size.data_ptr(), self.row_ptr.data_ptr(),
                       self.col_idx.data_ptr(), self.val_ptr.data_ptr())
        self.device = dev


def sm_pattern_sizes(A: Bcsr, pad_to: int):
    out = _Sizes()
    scratch = torch.zeros(64, dtype=torch.int64, device=A.device)
    _check("sm_pattern_sizes", _lib.sm_pattern_sizes(C.byref(A.c), C.c_int32(pad_to), C.byref(out),
                                                     _ptr(scratch), _stream()))
    return out


class Pattern:
    """Device arrays of sm_pattern_t, allocated by torch."""
    INT32 = ("nbr_ptr", "nbr_idx", "own_pos", "dim", "dim_pad", "row_off", "gmap", "tmap", "order")
    INT64 = ("sub_off", "gmap_ptr")

    def __init__(self, A: Bcsr, pad_to: int, sizes):
        n, dev = A.n_blk, A.device
        lens = dict(nbr_ptr=n + 1, nbr_idx=sizes.nbr_len, own_pos=n, dim=n, dim_pad=n, row_off=sizes.nbr_len,
                    sub_off=n + 1, gmap_ptr=n + 1, gmap=sizes.gmap_len, tmap=A.nnzb, order=n)
        for k in self.INT32:
            setattr(self, k, torch.empty(max(int(lens[k]), 1), dtype=torch.int32, device=dev))
        for k in self.INT64:
            setattr(self, k, torch.empty(max(int(lens[k]), 1), dtype=torch.int64, device=dev))
        self.n_blk, self.nnzb, self.pad_to = n, A.nnzb, pad_to
        self.max_dim, self.max_dim_pad, self.max_nbr = sizes.max_dim, sizes.max_dim_pad, sizes.max_nbr
        self.packed_elems, self.gmap_len = int(sizes.packed_elems), int(sizes.gmap_len)
        self.c = _Pattern(n, A.nnzb, pad_to, sizes.max_dim, sizes.max_dim_pad, sizes.max_nbr,
                          sizes.packed_elems, sizes.gmap_len,
                          *[getattr(self, k).data_ptr() for k in (
                              "nbr_ptr", "nbr_idx", "own_pos", "dim", "dim_pad", "row_off", "sub_off",
                              "gmap_ptr", "gmap", "tmap", "order")])
        self.device = dev
        self._h_dim_pad = None

    @property
    def h_dim_pad(self) -> np.ndarray:
        if self._h_dim_pad is None:
            self._h_dim_pad = self.dim_pad.cpu().numpy().astype(np.int32)
        return self._h_dim_pad


def sm_build_pattern(A: Bcsr, pad_to: int, sizes=None) -> Pattern:
    """a1.  `sizes`: the result of an earlier sm_pattern_sizes call on the same geometry (e.g. `P.sizes` of a previous
    build); sm_pattern_sizes validates the pattern and reads the sizes back, i.e. synchronises, so a caller that
    evaluates the same geometry repeatedly passes them in and the build itself stays asynchronous."""
    if sizes is None:
        sizes = sm_pattern_sizes(A, pad_to)
    P = Pattern(A, pad_to, sizes)
    P.sizes = sizes
    ws = torch.empty(int(sizes.build_ws_bytes), dtype=torch.uint8, device=A.device)
    _check("sm_build_pattern", _lib.sm_build_pattern(C.byref(A.c), C.c_int32(pad_to), C.byref(P.c), _ptr(ws),
                                                     C.c_int64(ws.numel()), _stream()))
    P._ws = ws
    return P


def _cols_tensor(P: Pattern, cols):
    if cols is None:
        return None
    if isinstance(cols, torch.Tensor):
        return cols.to(device=P.device, dtype=torch.int32).contiguous()
    return torch.as_tensor(np.ascontiguousarray(cols, dtype=np.int32), device=P.device)


def sm_plan_columns(P: Pattern, cols):
    """(cols tensor or None, col_off tensor, n_cols)."""
    ct = _cols_tensor(P, cols)
    if ct is None:
        return None, P.sub_off, P.n_blk
    n = int(ct.numel())
    col_off = torch.empty(n + 1, dtype=torch.int64, device=P.device)
    _check("sm_plan_columns", _lib.sm_plan_columns(C.byref(P.c), _ptr(ct), C.c_int32(n), _ptr(col_off), _stream()))
    return ct, col_off, n


def packed_elems(P: Pattern, cols) -> int:
    if cols is None:
        return P.packed_elems
    hp = P.h_dim_pad[np.asarray(cols.cpu() if isinstance(cols, torch.Tensor) else cols)].astype(np.int64)
    return int((hp * hp).sum())


def sm_gather(A: Bcsr, P: Pattern, cols, col_off, n_cols, mu, scale_mode, x_dtype, X=None, A_vals=None):
    x_dt = DTYPES[x_dtype] if isinstance(x_dtype, str) else x_dtype
    sc = SCALES[scale_mode] if isinstance(scale_mode, str) else scale_mode
    vals = A.vals if A_vals is None else A_vals
    if X is None:
        X = torch.empty(packed_elems(P, cols), dtype=TORCH_DTYPE[x_dt], device=A.device)
    scale = torch.empty(n_cols, dtype=torch.float64, device=A.device)
    wsb = int(_lib.sm_gather_ws_bytes(C.byref(A.c), C.byref(P.c), C.c_int32(n_cols)))
    ws = torch.empty(wsb, dtype=torch.uint8, device=A.device)
    _check("sm_gather", _lib.sm_gather(C.byref(A.c), _ptr(vals), C.c_int32(A.val_dtype), C.byref(P.c), _ptr(cols),
                                       C.c_int32(n_cols), _ptr(col_off), C.c_double(mu), C.c_int32(sc),
                                       C.c_int32(x_dt), _ptr(X), _ptr(scale), _ptr(ws), C.c_int64(wsb), _stream()))
    return X, scale


def sm_sign_ws_bytes(P: Pattern, n_cols, n_elems, x_dtype, flags=0) -> int:
    x_dt = DTYPES[x_dtype] if isinstance(x_dtype, str) else x_dtype
    if flags:
        b = int(_lib.sm_sign_ws_bytes_ex(C.byref(P.c), C.c_int32(n_cols), C.c_int64(n_elems), C.c_int32(x_dt),
                                         C.c_int32(flags)))
    else:
        b = int(_lib.sm_sign_ws_bytes(C.byref(P.c), C.c_int32(n_cols), C.c_int64(n_elems), C.c_int32(x_dt)))
    if b < 0:
        raise SmError("sm_sign_ws_bytes", b)
    return b


def sm_sign_ns(P: Pattern, cols, col_off, n_cols, n_elems, x_dtype, X, max_iter, tol, ws=None,
               iters=None, residual=None, flags=0, switch_iter=-1):
    """flags / switch_iter non-default: sm_sign_ns_ex (non-symmetric matrices, third-order iteration, bf16 -> fp16 schedule)."""
    x_dt = DTYPES[x_dtype] if isinstance(x_dtype, str) else x_dtype
    if ws is None:
        ws = torch.empty(sm_sign_ws_bytes(P, n_cols, n_elems, x_dt, flags), dtype=torch.uint8, device=P.device)
    if iters is None:
        iters = torch.empty(n_cols, dtype=torch.int32, device=P.device)
    if residual is None:
        residual = torch.empty(n_cols, dtype=torch.float64, device=P.device)
    if flags or switch_iter >= 0:
        _check("sm_sign_ns_ex", _lib.sm_sign_ns_ex(C.byref(P.c), _ptr(cols), C.c_int32(n_cols), _ptr(col_off),
                                                   C.c_int64(n_elems), C.c_int32(x_dt), _ptr(X), _ptr(ws),
                                                   C.c_int64(ws.numel()), C.c_int32(max_iter), C.c_double(tol),
                                                   C.c_int32(flags), C.c_int32(switch_iter),
                                                   _ptr(iters), _ptr(residual), _stream()))
    else:
        _check("sm_sign_ns", _lib.sm_sign_ns(C.byref(P.c), _ptr(cols), C.c_int32(n_cols), _ptr(col_off),
                                             C.c_int64(n_elems), C.c_int32(x_dt), _ptr(X), _ptr(ws),
                                             C.c_int64(ws.numel()), C.c_int32(max_iter), C.c_double(tol),
                                             _ptr(iters), _ptr(residual), _stream()))
    return iters, residual


def sm_sign_ns_static_capacity() -> int:
    return int(_lib.sm_sign_ns_static_capacity())


def sm_sign_ns_static(P: Pattern, cols, col_off, n_cols, n_elems, x_dtype, X, max_iter, tol, iters, residual):
    """sm_sign_ns on the library's static 16 MiB workspace: allocates nothing (iters / residual are the caller's)."""
    x_dt = DTYPES[x_dtype] if isinstance(x_dtype, str) else x_dtype
    _check("sm_sign_ns_static", _lib.sm_sign_ns_static(C.byref(P.c), _ptr(cols), C.c_int32(n_cols), _ptr(col_off),
                                                       C.c_int64(n_elems), C.c_int32(x_dt), _ptr(X), C.c_int32(max_iter),
                                                       C.c_double(tol), _ptr(iters), _ptr(residual), _stream()))
    return iters, residual


def sm_sign_status(residual, tol) -> int:
    scratch = torch.zeros(16, dtype=torch.int32, device=residual.device)
    return _check("sm_sign_status", _lib.sm_sign_status(_ptr(residual), C.c_int32(residual.numel()),
                                                        C.c_double(tol), _ptr(scratch), _stream()), allow_warn=True)


def sm_scatter(A: Bcsr, P: Pattern, cols, col_off, n_cols, x_dtype, S, r_dtype="f64", R=None, symmetrise=False):
    x_dt = DTYPES[x_dtype] if isinstance(x_dtype, str) else x_dtype
    r_dt = DTYPES[r_dtype] if isinstance(r_dtype, str) else r_dtype
    if R is None:
        R = torch.zeros(A.n_vals, dtype=TORCH_DTYPE[r_dt], device=A.device)
    _check("sm_scatter", _lib.sm_scatter(C.byref(A.c), C.byref(P.c), _ptr(cols), C.c_int32(n_cols), _ptr(col_off),
                                         C.c_int32(x_dt), _ptr(S), C.c_int32(r_dt), _ptr(R),
                                         C.c_int32(1 if symmetrise else 0), _stream()))
    return R


def sm_symmetrise(A: Bcsr, P: Pattern, R, r_dtype="f64"):
    r_dt = DTYPES[r_dtype] if isinstance(r_dtype, str) else r_dtype
    _check("sm_symmetrise", _lib.sm_symmetrise(C.byref(A.c), C.byref(P.c), C.c_int32(r_dt), _ptr(R), _stream()))
    return R


def sm_density_from_sign(A: Bcsr, P: Pattern, RD, d_dtype="f64"):
    d_dt = DTYPES[d_dtype] if isinstance(d_dtype, str) else d_dtype
    trace = torch.zeros(1, dtype=torch.float64, device=A.device)
    _check("sm_density_from_sign", _lib.sm_density_from_sign(C.byref(A.c), C.byref(P.c), C.c_int32(d_dt),
                                                             _ptr(RD), _ptr(trace), _stream()))
    return RD, trace


class DensityPlan:
    """Buffers for repeated sm_density calls on one geometry (allocated once)."""

    def __init__(self, A: Bcsr, P: Pattern, x_dtype, max_chunk_elems=None, d_dtype="f64", order=2):
        self.x_dt = DTYPES[x_dtype] if isinstance(x_dtype, str) else x_dtype
        self.d_dt = DTYPES[d_dtype] if isinstance(d_dtype, str) else d_dtype
        self.max_chunk_elems = int(max_chunk_elems or P.packed_elems)
        self.order = order          # workspace sized for sm_density(..., order=this)
        wsb = int(_lib.sm_density_ws_bytes_ex(C.byref(A.c), C.byref(P.c), C.c_int32(self.x_dt),
                                              C.c_int64(self.max_chunk_elems),
                                              C.c_int32(SM_SIGN_ORDER3 if order == 3 else 0)))
        if wsb < 0:
            raise SmError("sm_density_ws_bytes", wsb)
        dev = A.device
        self.ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
        self.D = torch.zeros(A.n_vals, dtype=TORCH_DTYPE[self.d_dt], device=dev)
        self.trace = torch.zeros(1, dtype=torch.float64, device=dev)
        self.iters = torch.zeros(A.n_blk, dtype=torch.int32, device=dev)
        self.residual = torch.zeros(A.n_blk, dtype=torch.float64, device=dev)
        self.scale = torch.zeros(A.n_blk, dtype=torch.float64, device=dev)
        self.h_dim_pad = np.ascontiguousarray(P.h_dim_pad, dtype=np.int32)


def sm_density(A: Bcsr, P: Pattern, plan: DensityPlan, mu=0.0, scale_mode="gershgorin", max_iter=100,
               tol=0.0, symmetrise=False, A_vals=None, switch_iter=-1, order=2):
    """Whole path; returns the plan (D, trace, iters, residual, scale live in it; the per-column
    arrays are indexed by position in P.order).  switch_iter >= 0: bf16 -> fp16 schedule; order = 3: third-order
    iteration in a3 (both through sm_density_ex)."""
    sc = SCALES[scale_mode] if isinstance(scale_mode, str) else scale_mode
    vals = A.vals if A_vals is None else A_vals
    if order not in (2, 3):
        raise ValueError("order must be 2 or 3")
    if order == 3 and plan.order != 3:
        raise ValueError("the plan's workspace was sized for order 2: DensityPlan(..., order=3)")
    if switch_iter >= 0 or order == 3:
        _check("sm_density_ex", _lib.sm_density_ex(
            C.byref(A.c), _ptr(vals), C.c_int32(A.val_dtype), C.c_double(mu), C.c_int32(plan.x_dt), C.c_int32(sc),
            C.c_int32(max_iter), C.c_double(tol), C.c_int32(switch_iter), C.c_int32(SM_SIGN_ORDER3 if order == 3 else 0),
            C.c_int32(1 if symmetrise else 0), C.byref(P.c),
            plan.h_dim_pad.ctypes.data_as(C.c_void_p), C.c_int64(plan.max_chunk_elems), _ptr(plan.ws),
            C.c_int64(plan.ws.numel()), C.c_int32(plan.d_dt), _ptr(plan.D), _ptr(plan.trace), _ptr(plan.iters),
            _ptr(plan.residual), _ptr(plan.scale), _stream()))
        return plan
    _check("sm_density", _lib.sm_density(
        C.byref(A.c), _ptr(vals), C.c_int32(A.val_dtype), C.c_double(mu), C.c_int32(plan.x_dt), C.c_int32(sc),
        C.c_int32(max_iter), C.c_double(tol), C.c_int32(1 if symmetrise else 0), C.byref(P.c),
        plan.h_dim_pad.ctypes.data_as(C.c_void_p), C.c_int64(plan.max_chunk_elems), _ptr(plan.ws),
        C.c_int64(plan.ws.numel()), C.c_int32(plan.d_dt), _ptr(plan.D), _ptr(plan.trace), _ptr(plan.iters),
        _ptr(plan.residual), _ptr(plan.scale), _stream()))
    return plan


def _doubled_elems(P: Pattern):
    """Elements of the doubled images (dimension 2 m_i rounded up to pad_to): buffer sizing only."""
    m2 = 2 * P.dim.cpu().numpy().astype(np.int64)
    p2 = (m2 + P.pad_to - 1) // P.pad_to * P.pad_to
    return int((p2 * p2).sum()), int((p2 * p2).max())


def sm_inv_sqrt(S: Bcsr, P: Pattern, x_dtype, max_iter=100, tol=0.0, max_chunk_elems2=None, z_dtype="f64", want_sqrt=False):
    """f2 (Eq. 12): returns (Z ~ S^-1/2, Y ~ S^1/2 or None, iters, residual, scale), per-column arrays by position in P.order."""
    x_dt, z_dt = DTYPES[x_dtype], DTYPES[z_dtype]
    total2, largest2 = _doubled_elems(P)
    mce = int(max_chunk_elems2 or total2)
    mce = max(mce, largest2)
    wsb = int(_lib.sm_inv_sqrt_ws_bytes(C.byref(S.c), C.byref(P.c), C.c_int32(x_dt), C.c_int64(mce)))
    if wsb < 0:
        raise SmError("sm_inv_sqrt_ws_bytes", wsb)
    dev = S.device
    ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
    Z = torch.zeros(S.n_vals, dtype=TORCH_DTYPE[z_dt], device=dev)
    Y = torch.zeros(S.n_vals, dtype=TORCH_DTYPE[z_dt], device=dev) if want_sqrt else None
    iters = torch.zeros(S.n_blk, dtype=torch.int32, device=dev)
    residual = torch.zeros(S.n_blk, dtype=torch.float64, device=dev)
    scale = torch.zeros(S.n_blk, dtype=torch.float64, device=dev)
    h_dim = np.ascontiguousarray(P.dim.cpu().numpy(), dtype=np.int32)
    _check("sm_inv_sqrt", _lib.sm_inv_sqrt(
        C.byref(S.c), _ptr(S.vals), C.c_int32(S.val_dtype), C.c_int32(x_dt), C.c_int32(max_iter), C.c_double(tol),
        C.byref(P.c), h_dim.ctypes.data_as(C.c_void_p), C.c_int64(mce), _ptr(ws), C.c_int64(ws.numel()), C.c_int32(z_dt),
        _ptr(Z), _ptr(Y), _ptr(iters), _ptr(residual), _ptr(scale), _stream()))
    return Z, Y, iters, residual, scale


def sm_density_nonorth(A: Bcsr, S_vals, P: Pattern, x_dtype, mu=0.0, max_iter=100, tol=0.0, symmetrise=False,
                       max_chunk_elems2=None):
    """f2 (Eq. 14 with S != I): returns (P_vals, Tr(P S), iters, residual, scale); P_vals in the arithmetic type for
    fp64 / fp32, fp64 for the 16-bit types."""
    x_dt = DTYPES[x_dtype]
    d_dt = x_dt if x_dt in (SM_F64, SM_F32) else SM_F64
    total2, largest2 = _doubled_elems(P)
    mce = max(int(max_chunk_elems2 or total2), largest2)
    wsb = int(_lib.sm_density_nonorth_ws_bytes(C.byref(A.c), C.byref(P.c), C.c_int32(x_dt), C.c_int64(mce)))
    if wsb < 0:
        raise SmError("sm_density_nonorth_ws_bytes", wsb)
    dev = A.device
    ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
    Pv = torch.zeros(A.n_vals, dtype=TORCH_DTYPE[d_dt], device=dev)
    tr = torch.zeros(1, dtype=torch.float64, device=dev)
    iters = torch.zeros(A.n_blk, dtype=torch.int32, device=dev)
    residual = torch.zeros(A.n_blk, dtype=torch.float64, device=dev)
    scale = torch.zeros(A.n_blk, dtype=torch.float64, device=dev)
    h_dim = np.ascontiguousarray(P.dim.cpu().numpy(), dtype=np.int32)
    _check("sm_density_nonorth", _lib.sm_density_nonorth(
        C.byref(A.c), _ptr(A.vals), _ptr(S_vals), C.c_int32(A.val_dtype), C.c_double(mu), C.c_int32(x_dt),
        C.c_int32(max_iter), C.c_double(tol), C.c_int32(1 if symmetrise else 0), C.byref(P.c),
        h_dim.ctypes.data_as(C.c_void_p), C.c_int64(mce), _ptr(ws), C.c_int64(ws.numel()), C.c_int32(d_dt), _ptr(Pv),
        _ptr(tr), _ptr(iters), _ptr(residual), _ptr(scale), _stream()))
    return Pv, tr, iters, residual, scale


def sm_mu_search(A: Bcsr, P: Pattern, plan: DensityPlan, n_target, mu_lo, mu_hi, tol_n=1e-6, mu_tol=1e-12,
                 max_trials=60, scale_mode="gershgorin", max_iter=100, tol=0.0, symmetrise=False, A_vals=None):
    """Bisection on Tr D(mu) = n_target; returns (mu, trace, trials); D etc. of the last trial live in the plan."""
    sc = SCALES[scale_mode] if isinstance(scale_mode, str) else scale_mode
    vals = A.vals if A_vals is None else A_vals
    mu, tr, nt = C.c_double(0.0), C.c_double(0.0), C.c_int32(0)
    _check("sm_mu_search", _lib.sm_mu_search(
        C.byref(A.c), _ptr(vals), C.c_int32(A.val_dtype), C.c_double(n_target), C.c_double(mu_lo),
        C.c_double(mu_hi), C.c_double(tol_n), C.c_double(mu_tol), C.c_int32(max_trials), C.c_int32(plan.x_dt),
        C.c_int32(sc), C.c_int32(max_iter), C.c_double(tol), C.c_int32(1 if symmetrise else 0), C.byref(P.c),
        plan.h_dim_pad.ctypes.data_as(C.c_void_p), C.c_int64(plan.max_chunk_elems), _ptr(plan.ws),
        C.c_int64(plan.ws.numel()), C.c_int32(plan.d_dt), _ptr(plan.D), _ptr(plan.trace), _ptr(plan.iters),
        _ptr(plan.residual), _ptr(plan.scale), C.byref(mu), C.byref(tr), C.byref(nt), _stream()))
    return mu.value, tr.value, nt.value


def pattern_to_host(P: Pattern) -> SimpleNamespace:
    return SimpleNamespace(**{k: getattr(P, k).cpu().numpy() for k in Pattern.INT32 + Pattern.INT64})
