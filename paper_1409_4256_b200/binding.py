"""Thin ctypes binding of libemc (include/emc.h): same names, argument marshalling only.

PyTorch provides device memory and streams; every step of the path runs in the library's CUDA
kernels.  There is no CPU fallback: if libemc.so cannot be loaded or a call fails, an EmcError is
raised.  Nothing here imports the oracle.
"""
from __future__ import annotations

import ctypes
import pathlib
from ctypes import POINTER, Structure, c_char_p, c_double, c_int, c_size_t, c_uint, c_uint64, c_void_p

import torch

from . import build as _build

EMC_OK = 0
EMC_ERR_ARG, EMC_ERR_UNSUPPORTED, EMC_ERR_WORKSPACE, EMC_ERR_CUDA, EMC_ERR_COUNT_RANGE, EMC_ERR_VALUE_RANGE = -1, -2, -3, -4, -5, -6
EMC_ERR_STATIC_SCRATCH = -7
EMC_STATIC_SCRATCH_BYTES = 4 << 20
EMC_I32, EMC_U16, EMC_U8 = 0, 1, 2
EMC_MAX_COUNT = 2048
EMC_COMPRESS_WEIGHTED = 0x1
EMC_ACCUMULATE = 0x2
EMC_UPDATE_RAW = 0x4
EMC_PATTERNS_ON_HOST = 0x10
EMC_PROFILE_STAGES = 0x20
EMC_SPARSE_PHOTONS = 0x40
EMC_DEBUG_SIMT = 0x100
EMC_GEMM_1CTA = 0x200
EMC_MAX_SPANS = 4096
EMC_VIEW_LOGLIK, EMC_VIEW_S, EMC_VIEW_WNEW = 0, 1, 2
STAGES = ("expand", "pack", "loglik", "normalize", "update", "compress")

# every symbol include/emc.h declares (tests check the library exports all of them)
SYMBOLS = ("emc_context_create", "emc_context_destroy", "emc_workspace_bytes", "emc_workspace_bytes_geometry", "emc_expand", "emc_loglik",
           "emc_normalize", "emc_normalize_static", "emc_normalize_static_bytes", "emc_update", "emc_compress", "emc_iterate", "emc_iterate_rot_chunked",
           "emc_workspace_bytes_rot_chunked", "emc_workspace_view", "emc_shard_stats", "emc_shard_update", "emc_shard_finish", "emc_iterate_gaussian", "emc_loglik_gaussian", "emc_refine", "emc_check",
           "emc_profile_read", "emc_profile_dropped", "emc_launch_count", "emc_strerror", "emc_last_cuda_error", "emc_version")


class EmcError(RuntimeError):
    def __init__(self, status, where):
        lib = load()
        msg = lib.emc_strerror(status).decode()
        if status == EMC_ERR_CUDA:
            msg += ": " + lib.emc_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({status})")
        self.status = status


class _Model(Structure):
    _fields_ = [("n", c_int), ("model", c_void_p)]


class _Detector(Structure):
    _fields_ = [("n_pix", c_int), ("q", c_void_p), ("mask", c_void_p), ("row_len", c_int)]


class _Rotations(Structure):
    _fields_ = [("n_rot", c_int), ("quat", c_void_p), ("weight", c_void_p)]


class _Patterns(Structure):
    _fields_ = [("n_pat", c_int), ("counts", c_void_p), ("type", c_int)]


_LIB = None


def load(path: str | pathlib.Path | None = None) -> ctypes.CDLL:
    """dlopen libemc.so (built in-tree by build.py) and declare the prototypes of include/emc.h."""
    global _LIB
    if _LIB is not None and path is None:
        return _LIB
    p = pathlib.Path(path) if path else _build.LIB
    if not p.exists():
        p = _build.build()          # needs nvcc; raises if it cannot be built -- no fallback
    lib = ctypes.CDLL(str(p))
    vp, sz, ci, cu = c_void_p, c_size_t, c_int, c_uint
    lib.emc_context_create.restype = ci
    lib.emc_context_create.argtypes = [POINTER(vp)]
    lib.emc_context_destroy.restype = ci
    lib.emc_context_destroy.argtypes = [vp]
    lib.emc_workspace_bytes.restype = sz
    lib.emc_workspace_bytes.argtypes = [ci, ci, ci, ci, cu]
    lib.emc_workspace_bytes_geometry.restype = sz
    lib.emc_workspace_bytes_geometry.argtypes = [ci, ci, ci]
    lib.emc_expand.restype = ci
    lib.emc_expand.argtypes = [POINTER(_Model), POINTER(_Detector), POINTER(_Rotations), vp, vp, vp, sz, vp]
    lib.emc_loglik.restype = ci
    lib.emc_loglik.argtypes = [vp, vp, POINTER(_Detector), POINTER(_Patterns), ci, vp, ci, cu, vp, sz, vp]
    lib.emc_normalize.restype = ci
    lib.emc_normalize.argtypes = [vp, POINTER(_Rotations), ci, ci, vp, vp, vp, cu, vp, sz, vp]
    lib.emc_normalize_static_bytes.restype = sz
    lib.emc_normalize_static_bytes.argtypes = [ci, ci, ci]
    lib.emc_normalize_static.restype = ci
    lib.emc_normalize_static.argtypes = [vp, POINTER(_Rotations), ci, ci, vp, vp, vp, cu, vp]
    lib.emc_update.restype = ci
    lib.emc_update.argtypes = [vp, ci, vp, POINTER(_Detector), POINTER(_Patterns), ci, vp, cu, vp, sz, vp]
    lib.emc_compress.restype = ci
    lib.emc_compress.argtypes = [vp, vp, POINTER(_Detector), POINTER(_Rotations), ci, vp, vp, cu, vp, sz, vp]
    lib.emc_iterate.restype = ci
    lib.emc_iterate.argtypes = [POINTER(_Model), POINTER(_Detector), POINTER(_Rotations), POINTER(_Patterns),
                                ci, ci, vp, vp, ci, vp, cu, vp, sz, vp, vp]
    lib.emc_workspace_view.restype = ci
    lib.emc_workspace_view.argtypes = [vp, ci, ci, ci, ci, cu, ci, POINTER(vp), POINTER(c_int)]
    lib.emc_workspace_bytes_rot_chunked.restype = sz
    lib.emc_workspace_bytes_rot_chunked.argtypes = [ci, ci, ci, ci, ci]
    lib.emc_iterate_rot_chunked.restype = ci
    lib.emc_iterate_rot_chunked.argtypes = [POINTER(_Model), POINTER(_Detector), POINTER(_Rotations), POINTER(_Patterns),
                                            ci, ci, vp, vp, cu, vp, sz, vp, vp]
    lib.emc_loglik_gaussian.restype = ci
    lib.emc_loglik_gaussian.argtypes = [vp, POINTER(_Detector), POINTER(_Patterns), ci, ctypes.c_float, vp, vp, ci, cu, vp, sz, vp]
    lib.emc_shard_stats.restype = ci
    lib.emc_shard_stats.argtypes = [POINTER(_Model), POINTER(_Detector), POINTER(_Rotations), POINTER(_Patterns), ci, vp, cu,
                                    vp, sz, vp]
    lib.emc_shard_update.restype = ci
    lib.emc_shard_update.argtypes = [POINTER(_Model), POINTER(_Detector), POINTER(_Rotations), POINTER(_Patterns), ci, vp, ci,
                                     vp, vp, vp, cu, vp, sz, vp]
    lib.emc_shard_finish.restype = ci
    lib.emc_shard_finish.argtypes = [vp, ci, vp, vp]
    lib.emc_iterate_gaussian.restype = ci
    lib.emc_iterate_gaussian.argtypes = [POINTER(_Model), POINTER(_Detector), POINTER(_Rotations), POINTER(_Patterns),
                                         ci, ci, ctypes.c_float, vp, vp, ci, vp, cu, vp, sz, vp, vp]
    lib.emc_refine.restype = ci
    lib.emc_refine.argtypes = [POINTER(_Model), POINTER(_Detector), POINTER(_Rotations), ci, POINTER(_Patterns), ci,
                               c_double, ci, vp, vp, vp, POINTER(ctypes.c_int32), cu, vp, sz, vp, vp]
    lib.emc_check.restype = ci
    lib.emc_check.argtypes = [vp, vp]
    lib.emc_profile_read.restype = ci
    lib.emc_profile_read.argtypes = [vp, POINTER(c_double), POINTER(c_int)]
    lib.emc_profile_dropped.restype = ci
    lib.emc_profile_dropped.argtypes = [vp]
    lib.emc_launch_count.restype = c_uint64
    lib.emc_launch_count.argtypes = []
    for name in ("emc_strerror", "emc_last_cuda_error", "emc_version"):
        getattr(lib, name).restype = c_char_p
    lib.emc_strerror.argtypes = [ci]
    if path is None:
        _LIB = lib
    return lib


# ---------------------------------------------------------------------------- marshalling helpers

_COUNT_TYPES = {torch.int32: EMC_I32, torch.uint16: EMC_U16, torch.uint8: EMC_U8}


def _dev(t: torch.Tensor, dtype, name: str) -> int:
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of {dtype}")
    return t.data_ptr()


def _opt(t, dtype, name):
    return None if t is None else _dev(t, dtype, name)


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _check(status: int, where: str):
    if status != EMC_OK:
        raise EmcError(status, where)


def ld_for(n_pat: int) -> int:
    """Row pitch (floats) the binding uses for L and P: N rounded up to 64."""
    return (n_pat + 63) // 64 * 64


def _detector(q, mask):
    """q is [P, 3], or [rows, row_len, 3] for a row-major 2-D detector (emc_detector.row_len, a locality hint)."""
    row_len = q.shape[1] if q.dim() == 3 else 0
    n_pix = q.numel() // 3
    if mask is not None and mask.numel() != n_pix:
        raise ValueError("mask length != number of pixels")
    return _Detector(n_pix, _dev(q, torch.float32, "q"), _opt(mask, torch.uint8, "mask"), row_len)


def _rotations(quat, weight):
    if weight is not None and weight.shape[0] != quat.shape[0]:
        raise ValueError("weight length != number of rotations")
    return _Rotations(quat.shape[0], _dev(quat, torch.float32, "quat"), _opt(weight, torch.float32, "weight"))


def _patterns(counts, n_pix, on_host=False):
    if counts.dtype not in _COUNT_TYPES or counts.dim() != 2 or counts.shape[1] != n_pix or not counts.is_contiguous():
        raise TypeError("counts: expected a contiguous [N, P] tensor of int32, uint16 or uint8")
    if on_host:
        if counts.is_cuda or not counts.is_pinned():
            raise TypeError("counts: EMC_PATTERNS_ON_HOST needs a pinned host tensor")
    elif not counts.is_cuda:
        raise TypeError("counts: expected a CUDA tensor")
    return _Patterns(counts.shape[0], counts.data_ptr(), _COUNT_TYPES[counts.dtype])


def emc_workspace_bytes(n: int, n_pix: int, n_rot: int, n_pat_chunk: int, flags: int = 0) -> int:
    return load().emc_workspace_bytes(n, n_pix, n_rot, n_pat_chunk, flags)


def make_workspace(n, n_pix, n_rot, n_pat_chunk, flags=0, device="cuda") -> torch.Tensor:
    nbytes = emc_workspace_bytes(n, n_pix, n_rot, n_pat_chunk, flags)
    if nbytes == 0:
        raise EmcError(EMC_ERR_UNSUPPORTED, "emc_workspace_bytes")
    return torch.empty(nbytes, dtype=torch.uint8, device=device)


def make_geometry_workspace(n, n_pix, n_rot, device="cuda") -> torch.Tensor:
    """Workspace for emc_expand / emc_compress alone (emc_workspace_bytes_geometry)."""
    nbytes = load().emc_workspace_bytes_geometry(n, n_pix, n_rot)
    if nbytes == 0:
        raise EmcError(EMC_ERR_UNSUPPORTED, "emc_workspace_bytes_geometry")
    return torch.empty(nbytes, dtype=torch.uint8, device=device)


def _ws(ws, n, n_pix, n_rot, n_chunk, flags=0):
    if ws is None:
        ws = make_workspace(n, n_pix, n_rot, n_chunk, flags)
    return ws, ws.data_ptr(), ws.numel()


# ---------------------------------------------------------------------------- context

class EmcContext:
    """emc_context (include/emc.h): the copy stream and event pool the library may use on the caller's behalf.
    One context serves one stream at a time."""

    def __init__(self):
        h = c_void_p()
        _check(load().emc_context_create(ctypes.byref(h)), "emc_context_create")
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            load().emc_context_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


_DEFAULT_CTX = None


def default_context() -> EmcContext:
    """The binding's own context, created on first use (outside any libemc hot call)."""
    global _DEFAULT_CTX
    if _DEFAULT_CTX is None:
        _DEFAULT_CTX = EmcContext()
    return _DEFAULT_CTX


def _ctx(ctx, flags):
    if ctx is None and flags & (EMC_PATTERNS_ON_HOST | EMC_PROFILE_STAGES):
        ctx = default_context()
    return ctx.handle if ctx is not None else None


# ---------------------------------------------------------------------------- the six calls

def emc_expand(model, q, quat, want_idx=True, use_ws=True):
    """Stage 1 (eq. 2.9).  Returns (W [R,P] float32, idx [R,P] int32 or None).  use_ws=False takes the
    library's plain-gather kernel instead of the blocked-copy one."""
    n = model.shape[0]
    m = _Model(n, _dev(model, torch.float32, "model"))
    det = _detector(q, None)
    rot = _rotations(quat, None)
    w = torch.empty((rot.n_rot, det.n_pix), dtype=torch.float32, device=model.device)
    idx = torch.empty((rot.n_rot, det.n_pix), dtype=torch.int32, device=model.device) if want_idx else None
    ws = make_geometry_workspace(n, det.n_pix, rot.n_rot) if use_ws else None
    _check(load().emc_expand(m, det, rot, w.data_ptr(), idx.data_ptr() if want_idx else None,
                             ws.data_ptr() if use_ws else None, ws.numel() if use_ws else 0, _stream()), "emc_expand")
    return w, idx


def emc_loglik(w, idx, q, mask, counts, flags=0, ws=None):
    """Stage 2.  Returns L as a [R, N] view of a [R, ld_n] float32 tensor."""
    n_rot, n_pix = w.shape
    det = _detector(q, mask)
    pat = _patterns(counts, n_pix)
    ld = ld_for(pat.n_pat)
    big_l = torch.empty((n_rot, ld), dtype=torch.float32, device=w.device)
    ws, wp, wb = _ws(ws, 2, n_pix, n_rot, pat.n_pat)
    _check(load().emc_loglik(_dev(w, torch.float32, "W"), _opt(idx, torch.int32, "idx"), det, pat, n_rot,
                             big_l.data_ptr(), ld, flags, wp, wb, _stream()), "emc_loglik")
    return big_l[:, :pat.n_pat]


def _pitched(x, name):
    """(base pointer, pitch) of a [R, N] float32 view whose rows are `pitch` floats apart."""
    if x.dtype != torch.float32 or not x.is_cuda or x.dim() != 2 or x.stride(1) != 1:
        raise TypeError(f"{name}: expected a 2-D CUDA float32 tensor with unit column stride")
    return x.data_ptr(), x.stride(0)


def emc_normalize(big_l, quat, weight, flags=0, s=None, loglik=None, ws=None):
    """Stage 3.  Returns (P [R,N] view, s [R], loglik 1-element float64 tensor)."""
    n_rot, n_pat = big_l.shape
    lp, ld = _pitched(big_l, "L")
    rot = _rotations(quat, weight)
    p = torch.empty((n_rot, ld), dtype=torch.float32, device=big_l.device)
    if s is None:
        s = torch.zeros(n_rot, dtype=torch.float32, device=big_l.device)
    if loglik is None:
        loglik = torch.zeros(1, dtype=torch.float64, device=big_l.device)
    ws, wp, wb = _ws(ws, 2, 1, n_rot, n_pat)
    _check(load().emc_normalize(lp, rot, n_pat, ld, p.data_ptr(), s.data_ptr(), loglik.data_ptr(), flags, wp, wb,
                                _stream()), "emc_normalize")
    return p[:, :n_pat], s, loglik


def emc_normalize_static(big_l, quat, weight, p_out, s_out=None, loglik_out=None, flags=0):
    """Stage 3 without a workspace, for callers that cannot allocate device memory (include/emc.h,
    emc_normalize_static): the scratch is an array built into libemc.  Unlike the other wrappers this one creates no
    tensor: the caller passes L and every output -- p_out a [R, N] float32 view with the row pitch of L, s_out [R]
    float32 or None, loglik_out one float64 or None -- and gets nothing back.  Raises EmcError
    (EMC_ERR_STATIC_SCRATCH) when the sizes exceed the built-in array.  Calls that may overlap on the GPU race on
    that array: keep them on one stream."""
    n_rot, n_pat = big_l.shape
    lp, ld = _pitched(big_l, "L")
    pp, ldp = _pitched(p_out, "P")
    if tuple(p_out.shape) != (n_rot, n_pat) or ldp != ld:
        raise ValueError("p_out: expected the shape and row pitch of L")
    rot = _rotations(quat, weight)
    _check(load().emc_normalize_static(lp, rot, n_pat, ld, pp, _opt(s_out, torch.float32, "s"),
                                       _opt(loglik_out, torch.float64, "loglik"), flags, _stream()), "emc_normalize_static")


def emc_update(p, s, q, mask, counts, flags=0, wnew=None, ws=None):
    """Stage 4 (eq. 2.5 / 2.11).  Returns W' [R,P] float32."""
    n_rot, n_pat = p.shape
    pp, ld = _pitched(p, "P")
    det = _detector(q, mask)
    pat = _patterns(counts, det.n_pix)
    if pat.n_pat != n_pat:
        raise ValueError("P columns != number of patterns")
    if wnew is None:
        wnew = torch.empty((n_rot, det.n_pix), dtype=torch.float32, device=p.device)
    ws, wp, wb = _ws(ws, 2, det.n_pix, n_rot, n_pat)
    _check(load().emc_update(pp, ld, _opt(s, torch.float32, "s"), det, pat, n_rot,
                             _dev(wnew, torch.float32, "Wnew"), flags, wp, wb, _stream()), "emc_update")
    return wnew


def emc_compress(wnew, slice_w, q, mask, quat, n, flags=0, want_den=False, ws=None):
    """Stage 5 (eq. 2.10 / 2.12).  Returns (model' [n,n,n] float32, den [n^3] or None)."""
    n_rot, n_pix = wnew.shape
    det = _detector(q, mask)
    rot = _rotations(quat, None)
    model = torch.empty((n, n, n), dtype=torch.float32, device=wnew.device)
    den = torch.empty(n * n * n, dtype=torch.float32, device=wnew.device) if want_den else None
    if ws is None:
        ws = make_geometry_workspace(n, n_pix, n_rot)
    wp, wb = ws.data_ptr(), ws.numel()
    _check(load().emc_compress(_dev(wnew, torch.float32, "Wnew"), _opt(slice_w, torch.float32, "slice_w"), det, rot,
                               n, model.data_ptr(), den.data_ptr() if want_den else None, flags, wp, wb, _stream()),
           "emc_compress")
    return model, den


def emc_iterate(model, q, mask, quat, weight, counts, n_iter=1, n_pat_chunk=0, flags=0, want_p=False, ws=None,
                model_out=None, loglik=None, ctx=None):
    """Algorithm 1: n_iter iterations of stages 1-5.  Returns dict(model, loglik [n_iter] float64, P or None)."""
    n = model.shape[0]
    m = _Model(n, _dev(model, torch.float32, "model"))
    det = _detector(q, mask)
    rot = _rotations(quat, weight)
    on_host = bool(flags & EMC_PATTERNS_ON_HOST)
    pat = _patterns(counts, det.n_pix, on_host)
    chunk = pat.n_pat if (n_pat_chunk == 0 or n_pat_chunk > pat.n_pat) else n_pat_chunk
    dev = model.device
    if model_out is None:
        model_out = torch.empty_like(model)
    if loglik is None:
        loglik = torch.zeros(n_iter, dtype=torch.float64, device=dev)
    ld = ld_for(pat.n_pat)
    p = torch.empty((rot.n_rot, ld), dtype=torch.float32, device=dev) if want_p else None
    ws, wp, wb = _ws(ws, n, det.n_pix, rot.n_rot, chunk, flags)
    _check(load().emc_iterate(m, det, rot, pat, n_iter, n_pat_chunk, _dev(model_out, torch.float32, "model_out"),
                              p.data_ptr() if want_p else None, ld, loglik.data_ptr(), flags, wp, wb, _stream(),
                              _ctx(ctx, flags)), "emc_iterate")
    return dict(model=model_out, loglik=loglik, P=p[:, :pat.n_pat] if want_p else None, ws=ws)


def emc_workspace_view(ws, n, n_pix, n_rot, n_pat_chunk, what, flags=0):
    """A tensor view (no copy) of what the emc_iterate call that used `ws` left in it (include/emc.h, emc_workspace_view):
    EMC_VIEW_LOGLIK -> L [R, n_pat_chunk] float32 (rows ld_n apart), EMC_VIEW_S -> s [R], EMC_VIEW_WNEW -> W' [R, P].
    Synchronise the stream of that call first."""
    ptr, ld = c_void_p(), c_int()
    _check(load().emc_workspace_view(ws.data_ptr(), n, n_pix, n_rot, n_pat_chunk, flags, what, ctypes.byref(ptr), ctypes.byref(ld)),
           "emc_workspace_view")
    off = ptr.value - ws.data_ptr()
    pitch = ld.value if what != EMC_VIEW_S else 1
    rows = n_rot if what != EMC_VIEW_S else 1
    cols = {EMC_VIEW_LOGLIK: n_pat_chunk, EMC_VIEW_S: n_rot, EMC_VIEW_WNEW: n_pix}[what]
    flat = ws[off: off + 4 * ((rows - 1) * pitch + cols)].view(torch.float32)
    if what == EMC_VIEW_S:
        return flat
    return flat.as_strided((rows, cols), (pitch, 1))


def emc_iterate_rot_chunked(model, q, mask, quat, weight, counts, n_rot_chunk, n_iter=1, flags=0, ws=None, ctx=None):
    """Algorithm 1 with the rotation list streamed in chunks.  Returns dict(model, loglik, ws)."""
    n = model.shape[0]
    m = _Model(n, _dev(model, torch.float32, "model"))
    det = _detector(q, mask)
    rot = _rotations(quat, weight)
    pat = _patterns(counts, det.n_pix)
    model_out = torch.empty_like(model)
    loglik = torch.zeros(n_iter, dtype=torch.float64, device=model.device)
    if ws is None:
        nbytes = load().emc_workspace_bytes_rot_chunked(n, det.n_pix, rot.n_rot, n_rot_chunk, pat.n_pat)
        if nbytes == 0:
            raise EmcError(EMC_ERR_UNSUPPORTED, "emc_workspace_bytes_rot_chunked")
        ws = torch.empty(nbytes, dtype=torch.uint8, device=model.device)
    _check(load().emc_iterate_rot_chunked(m, det, rot, pat, n_iter, n_rot_chunk, model_out.data_ptr(), loglik.data_ptr(),
                                          flags, ws.data_ptr(), ws.numel(), _stream(), _ctx(ctx, flags)),
           "emc_iterate_rot_chunked")
    return dict(model=model_out, loglik=loglik, ws=ws)


def emc_loglik_gaussian(w, q, mask, counts, sigma, flags=0, ws=None):
    """E-step exponent and fluence of the Gaussian model (eqs. 2.2, 2.3, 2.6).  Returns (Q, phi) as [R, N] views."""
    n_rot, n_pix = w.shape
    det = _detector(q, mask)
    pat = _patterns(counts, n_pix)
    ld = ld_for(pat.n_pat)
    big_q = torch.empty((n_rot, ld), dtype=torch.float32, device=w.device)
    phi = torch.empty((n_rot, ld), dtype=torch.float32, device=w.device)
    ws, wp, wb = _ws(ws, 2, n_pix, n_rot, pat.n_pat)
    _check(load().emc_loglik_gaussian(_dev(w, torch.float32, "W"), det, pat, n_rot, float(sigma), big_q.data_ptr(), phi.data_ptr(),
                                      ld, flags, wp, wb, _stream()), "emc_loglik_gaussian")
    return big_q[:, :pat.n_pat], phi[:, :pat.n_pat]


def emc_shard_stats(model, q, mask, quat_local, weight_local, counts, n_rot_total, flags=0, ws=None):
    """A rank's Expand, log-likelihood and per-pattern statistics (rotation shards, include/emc.h).
    Returns (stats [3, ld_n] float32, ws): ws carries L to emc_shard_update."""
    n = model.shape[0]
    m = _Model(n, _dev(model, torch.float32, "model"))
    det = _detector(q, mask)
    rot = _rotations(quat_local, weight_local)
    pat = _patterns(counts, det.n_pix)
    stats = torch.empty((3, ld_for(pat.n_pat)), dtype=torch.float32, device=model.device)
    ws, wp, wb = _ws(ws, n, det.n_pix, rot.n_rot, pat.n_pat, flags)
    _check(load().emc_shard_stats(m, det, rot, pat, n_rot_total, stats.data_ptr(), flags, wp, wb, _stream()), "emc_shard_stats")
    return stats, ws


def emc_shard_update(model, q, mask, quat_local, weight_local, counts, n_rot_total, stats_all, ws, flags=0):
    """Merges the ranks' statistics [world, 3, ld_n] and runs the rank's P, update and Compress scatter.
    Returns (numden [2, n, n, n] float32, loglik 1-element float64, s [R_local])."""
    n = model.shape[0]
    m = _Model(n, _dev(model, torch.float32, "model"))
    det = _detector(q, mask)
    rot = _rotations(quat_local, weight_local)
    pat = _patterns(counts, det.n_pix)
    world = stats_all.shape[0]
    if tuple(stats_all.shape[1:]) != (3, ld_for(pat.n_pat)):
        raise ValueError("stats_all: expected [world, 3, ld_n]")
    numden = torch.empty((2, n, n, n), dtype=torch.float32, device=model.device)
    loglik = torch.zeros(1, dtype=torch.float64, device=model.device)
    s = torch.empty(rot.n_rot, dtype=torch.float32, device=model.device)
    _check(load().emc_shard_update(m, det, rot, pat, n_rot_total, _dev(stats_all, torch.float32, "stats_all"), world,
                                   numden.data_ptr(), loglik.data_ptr(), s.data_ptr(), flags, ws.data_ptr(), ws.numel(),
                                   _stream()), "emc_shard_update")
    return numden, loglik, s


def emc_shard_finish(numden):
    """model' = num / den from the all-reduced grids."""
    n = numden.shape[1]
    model = torch.empty((n, n, n), dtype=torch.float32, device=numden.device)
    _check(load().emc_shard_finish(_dev(numden, torch.float32, "numden"), n, model.data_ptr(), _stream()), "emc_shard_finish")
    return model


def emc_iterate_gaussian(model, q, mask, quat, weight, counts, sigma, n_iter=1, n_pat_chunk=0, flags=0, want_p=False, ws=None,
                         ctx=None):
    """Algorithm 1 with the paper's Gaussian likelihood and fluence (eqs. 2.2-2.6).  Returns dict(model, loglik, P)."""
    n = model.shape[0]
    m = _Model(n, _dev(model, torch.float32, "model"))
    det = _detector(q, mask)
    rot = _rotations(quat, weight)
    pat = _patterns(counts, det.n_pix, bool(flags & EMC_PATTERNS_ON_HOST))
    dev = model.device
    model_out = torch.empty_like(model)
    loglik = torch.zeros(n_iter, dtype=torch.float64, device=dev)
    ld = ld_for(pat.n_pat)
    p = torch.empty((rot.n_rot, ld), dtype=torch.float32, device=dev) if want_p else None
    chunk = pat.n_pat if (n_pat_chunk == 0 or n_pat_chunk > pat.n_pat) else n_pat_chunk
    ws, wp, wb = _ws(ws, n, det.n_pix, rot.n_rot, chunk, flags)
    _check(load().emc_iterate_gaussian(m, det, rot, pat, n_iter, n_pat_chunk, float(sigma), model_out.data_ptr(),
                                       p.data_ptr() if want_p else None, ld, loglik.data_ptr(), flags, wp, wb, _stream(),
                                       _ctx(ctx, flags)), "emc_iterate_gaussian")
    return dict(model=model_out, loglik=loglik, P=p[:, :pat.n_pat] if want_p else None, ws=ws)


def emc_refine(model, q, mask, levels, counts, n_iter, threshold=0.01, n_pat_chunk=0, flags=0, ws=None, ctx=None):
    """Adaptive EMC (section 3.4, eq. 3.1).  `levels` = [(quat [R,4], weight [R] or None), ...] from coarse to
    fine.  Returns dict(model, loglik [n_iter] float64 tensor, level = list of the list index of every iteration)."""
    n = model.shape[0]
    m = _Model(n, _dev(model, torch.float32, "model"))
    det = _detector(q, mask)
    rots = (_Rotations * len(levels))(*[_rotations(qt, w) for qt, w in levels])
    pat = _patterns(counts, det.n_pix, bool(flags & EMC_PATTERNS_ON_HOST))
    chunk = pat.n_pat if (n_pat_chunk == 0 or n_pat_chunk > pat.n_pat) else n_pat_chunk
    model_out, model_tmp = torch.empty_like(model), torch.empty_like(model)
    loglik = torch.zeros(n_iter, dtype=torch.float64, device=model.device)
    level = (ctypes.c_int32 * n_iter)()
    ws, wp, wb = _ws(ws, n, det.n_pix, max(r.n_rot for r in rots), chunk, flags)
    _check(load().emc_refine(m, det, rots, len(levels), pat, n_iter, float(threshold), n_pat_chunk,
                             model_out.data_ptr(), model_tmp.data_ptr(), loglik.data_ptr(), level, flags, wp, wb,
                             _stream(), _ctx(ctx, flags)), "emc_refine")
    return dict(model=model_out, loglik=loglik, level=list(level), ws=ws)


def emc_check(ws):
    """Synchronises and raises EmcError(EMC_ERR_COUNT_RANGE) if a count exceeded EMC_MAX_COUNT."""
    _check(load().emc_check(ws.data_ptr(), _stream()), "emc_check")


def emc_profile_read(ctx=None) -> dict:
    """Per-stage device milliseconds and span counts recorded under EMC_PROFILE_STAGES in `ctx` (default: the
    binding's own context); resets."""
    ms = (c_double * len(STAGES))()
    spans = (c_int * len(STAGES))()
    _check(load().emc_profile_read((ctx or default_context()).handle, ms, spans), "emc_profile_read")
    return {name: (ms[i], spans[i]) for i, name in enumerate(STAGES)}


def emc_profile_dropped(ctx=None) -> int:
    """Spans dropped because the context's pool of EMC_MAX_SPANS event pairs was exhausted; resets the count."""
    return load().emc_profile_dropped((ctx or default_context()).handle)


def emc_launch_count() -> int:
    return load().emc_launch_count()


def emc_version() -> str:
    return load().emc_version().decode()


__all__ = sorted(n for n in dir() if n.startswith(("emc_", "EMC_", "Emc"))) + [
    "STAGES", "SYMBOLS", "ld_for", "load", "make_workspace", "make_geometry_workspace", "default_context"]
