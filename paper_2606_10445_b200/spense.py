"""Thin ctypes binding of libspense.so (include/spense.h).  Argument marshalling only: every step
of the path runs in the CUDA kernels.  PyTorch supplies device memory and streams, nothing else.

There is no fallback: if the shared library is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, c_char_p, c_float, c_int, c_int32, c_int64, c_size_t, c_void_p

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libspense.so")

SPENSE_F32, SPENSE_BF16 = 0, 1
SPENSE_PER_TENSOR, SPENSE_PER_ROW = 0, 1

STATUS = {0: "SPENSE_OK", -1: "SPENSE_ERR_ARG", -2: "SPENSE_ERR_ALIGN", -3: "SPENSE_ERR_SHAPE",
          -4: "SPENSE_ERR_BUFFER_TOO_SMALL", -5: "SPENSE_ERR_NOT_2_4", -6: "SPENSE_ERR_NAN_WEIGHT",
          -7: "SPENSE_ERR_BAD_PERM", -8: "SPENSE_ERR_ARCH", -9: "SPENSE_ERR_CUDA", -10: "SPENSE_ERR_BAD_BLOB",
          -11: "SPENSE_ERR_TIMEOUT", -12: "SPENSE_ERR_STATIC_SCRATCH"}

EXPORTS = ["spense_version", "spense_strerror", "spense_device_status", "spense_schedule", "spense_perm_from_dense_idx", "spense_pack_sizes", "spense_pack",
           "spense_workspace_size", "spense_workspace_init", "spense_gate_up", "spense_down", "spense_mlp",
           "spense_mlp_dyn", "spense_mlp_host", "spense_mlp_stack_host", "spense_quantize_e4m3", "spense_prune_2to4_magnitude", "spense_dense_idx_last", "spense_select_workspace_size",
           "spense_select_dense", "spense_linear_pack_sizes", "spense_pack_linear", "spense_linear_workspace_size",
           "spense_linear_out_split", "spense_linear_in_split", "spense_prune_obs_workspace_size", "spense_prune_obs_2to4",
           "spense_quantize_e4m3_static", "spense_probe_read"]

SPENSE_SPLIT_OUT, SPENSE_SPLIT_IN = 0, 1
SPENSE_QUANTIZE_STATIC_MAX_ROWS = 65536


class SpenseError(RuntimeError):
    def __init__(self, status: int, where=None):
        self.status = status
        self.code = STATUS.get(status, str(status))
        self.where = where
        super().__init__(f"{self.code} ({lib().spense_strerror(status).decode()})" + (f" at {where}" if where else ""))


class Shape(ctypes.Structure):
    _fields_ = [("H", c_int32), ("I", c_int32), ("I_dense", c_int32)]


class Canon(ctypes.Structure):
    _fields_ = [(n, c_void_p) for n in ("perm", "gate_sp_val", "up_sp_val", "gate_sp_meta", "up_sp_meta",
                                        "gate_dn", "up_dn", "down_sp_val", "down_sp_meta", "down_dn")]


class LinearShape(ctypes.Structure):
    _fields_ = [("N", c_int32), ("K", c_int32), ("n_dense", c_int32), ("split", c_int32)]


class LinearCanon(ctypes.Structure):
    _fields_ = [(n, c_void_p) for n in ("perm", "sp_val", "sp_meta", "dn")]


_lib = None


def lib() -> ctypes.CDLL:
    """Load libspense.so (built in-tree by paper_2606_10445_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_2606_10445_b200.build` "
                               "(there is no CPU / PyTorch fallback for the Spense path)")
        L = ctypes.CDLL(LIB_PATH)
        L.spense_version.restype = c_int
        L.spense_strerror.restype = c_char_p
        L.spense_strerror.argtypes = [c_int]
        L.spense_device_status.argtypes = [c_int]
        L.spense_schedule.argtypes = [POINTER(Shape), c_int32, c_int32, c_int32, POINTER(c_int32), POINTER(c_int32)]
        L.spense_perm_from_dense_idx.argtypes = [c_int32, POINTER(c_int32), c_int32, POINTER(c_int32)]
        L.spense_pack_sizes.argtypes = [POINTER(Shape), POINTER(c_size_t), POINTER(c_size_t)]
        L.spense_pack.argtypes = [POINTER(Shape), c_void_p, c_void_p, c_void_p, POINTER(c_float), c_void_p, c_void_p,
                                  c_size_t, POINTER(Canon), c_void_p, c_size_t, POINTER(c_int64), c_void_p]
        L.spense_workspace_size.argtypes = [POINTER(Shape), c_int32, POINTER(c_size_t)]
        L.spense_workspace_init.argtypes = [c_void_p, c_size_t, c_void_p]
        L.spense_gate_up.argtypes = [POINTER(Shape), c_void_p, c_void_p, c_void_p, c_int32, c_void_p, c_int32,
                                     c_void_p, c_void_p, c_void_p, c_size_t, c_void_p]
        L.spense_down.argtypes = [POINTER(Shape), c_void_p, c_void_p, c_void_p, c_int32, c_int32, c_void_p, c_int32,
                                  c_void_p, c_size_t, c_void_p, c_void_p]
        L.spense_mlp.argtypes = [POINTER(Shape), c_void_p, c_void_p, c_void_p, c_int32, c_void_p, c_int32, c_void_p,
                                 c_void_p, c_void_p, c_int32, c_void_p, c_size_t, c_void_p, c_void_p]
        L.spense_mlp_dyn.argtypes = [POINTER(Shape), c_void_p, c_void_p, c_void_p, c_int32, c_void_p, c_void_p, c_void_p,
                                     c_void_p, c_int32, c_void_p, c_size_t, c_void_p, c_void_p]
        L.spense_mlp_host.argtypes = [POINTER(Shape), c_void_p, c_void_p, c_void_p, c_int32, c_void_p, c_int32,
                                      c_void_p, c_int32, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_size_t,
                                      c_void_p, c_void_p]
        L.spense_mlp_stack_host.argtypes = [POINTER(Shape), POINTER(c_void_p), c_int32, c_void_p, c_void_p, c_int32, c_void_p,
                                            c_int32, c_void_p, c_int32, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p,
                                            c_size_t, c_void_p]
        L.spense_select_workspace_size.argtypes = [POINTER(Shape), POINTER(c_size_t)]
        L.spense_select_dense.argtypes = [POINTER(Shape), c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_float, c_void_p,
                                          c_void_p, c_void_p, c_void_p, c_size_t, c_void_p]
        L.spense_prune_2to4_magnitude.argtypes = [POINTER(Shape), c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
        L.spense_dense_idx_last.argtypes = [c_int32, c_int32, POINTER(c_int32)]
        L.spense_quantize_e4m3.argtypes = [c_void_p, c_int64, c_int64, c_int32, c_void_p, c_void_p, c_void_p,
                                           c_size_t, c_void_p]
        L.spense_quantize_e4m3_static.argtypes = [c_void_p, c_int64, c_int64, c_int32, c_void_p, c_void_p, c_void_p]
        L.spense_probe_read.argtypes = [c_void_p, c_size_t, c_void_p, c_void_p]
        L.spense_linear_pack_sizes.argtypes = [POINTER(LinearShape), POINTER(c_size_t), POINTER(c_size_t)]
        L.spense_pack_linear.argtypes = [POINTER(LinearShape), c_void_p, c_float, c_void_p, c_void_p, c_size_t, POINTER(LinearCanon),
                                         c_void_p, c_size_t, POINTER(c_int64), c_void_p]
        L.spense_linear_workspace_size.argtypes = [POINTER(LinearShape), c_int32, POINTER(c_size_t)]
        for f in (L.spense_linear_out_split, L.spense_linear_in_split):
            f.argtypes = [POINTER(LinearShape), c_void_p, c_void_p, c_void_p, c_int32, c_int32, c_void_p, c_int32, c_void_p,
                          c_size_t, c_void_p]
        L.spense_prune_obs_workspace_size.argtypes = [c_int32, c_int32, POINTER(c_size_t)]
        L.spense_prune_obs_2to4.argtypes = [c_int32, c_int32, c_int32, c_void_p, c_void_p, c_void_p, c_size_t, c_void_p]
        for name in EXPORTS:
            if name not in ("spense_strerror",):
                getattr(L, name).restype = c_int
        _lib = L
    return _lib


def _check(st: int, where=None):
    if st != 0:
        raise SpenseError(st, where)


def _ptr(t):
    return None if t is None else c_void_p(t.data_ptr())


def _stream():
    return c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t: torch.Tensor, dtype=None):
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"expected dtype {dtype}, got {t.dtype}")
    return t


def spense_version() -> int:
    return lib().spense_version()


def spense_device_status(clear: bool = False) -> str:
    """The first device-side error an earlier launch recorded (synchronise first), as its status name."""
    return STATUS[lib().spense_device_status(1 if clear else 0)]


def spense_schedule(H: int, I: int, I_dense: int, M: int, mode: int, sms: int = 148):
    """(span boundaries, info) of the launch geometry for M tokens; see include/spense.h."""
    sb = (c_int32 * 161)()
    info = (c_int32 * 6)()
    n = lib().spense_schedule(ctypes.byref(Shape(H, I, I_dense)), M, mode, sms, sb, info)
    if n < 0:
        raise SpenseError(n)
    return list(sb[:n + 1]), dict(zip(("stages", "blocks_per_launch", "n_pad", "ring", "blocks", "ctas_per_span"), info))


def spense_perm_from_dense_idx(I: int, dense_idx) -> torch.Tensor:
    idx = (c_int32 * len(dense_idx))(*[int(v) for v in dense_idx])
    out = (c_int32 * I)()
    _check(lib().spense_perm_from_dense_idx(I, idx, len(dense_idx), out))
    return torch.tensor(list(out), dtype=torch.int32)


def spense_dense_idx_last(I: int, n_dense: int) -> torch.Tensor:
    out = (c_int32 * max(n_dense, 1))()
    _check(lib().spense_dense_idx_last(I, n_dense, out))
    return torch.tensor(list(out[:n_dense]), dtype=torch.int32)


def spense_prune_2to4_magnitude(wgate, wup, wdown, perm, I_dense: int):
    """In place magnitude 2:4 pruning of the sparse region (permuted order) of fp32 CUDA weights in original order."""
    for t in (wgate, wup, wdown):
        _dev(t, torch.float32)
    if perm is not None:
        _dev(perm, torch.int32)
    I, H = wgate.shape
    _check(lib().spense_prune_2to4_magnitude(ctypes.byref(Shape(H, I, I_dense)), _ptr(wgate), _ptr(wup), _ptr(wdown), _ptr(perm), _stream()))
    return wgate, wup, wdown


def spense_pack_sizes(H: int, I: int, I_dense: int):
    b, w = c_size_t(), c_size_t()
    _check(lib().spense_pack_sizes(ctypes.byref(Shape(H, I, I_dense)), ctypes.byref(b), ctypes.byref(w)))
    return b.value, w.value


class PackedLayer:
    """A packed Spense layer: the opaque device blob plus (optionally) the canonical arrays."""

    def __init__(self, H, I, I_dense, blob, canon=None):
        self.H, self.I, self.I_dense, self.blob, self.canon = H, I, I_dense, blob, canon
        self.shape = Shape(H, I, I_dense)


def spense_pack(wgate, wup, wdown, w_scale, perm, I_dense: int, want_canon: bool = False) -> PackedLayer:
    """wgate, wup uint8 [I, H]; wdown uint8 [H, I] (CUDA, original index order); perm int32 [I] or None."""
    _dev(wgate, torch.uint8), _dev(wup, torch.uint8), _dev(wdown, torch.uint8)
    I, H = wgate.shape
    dev = wgate.device
    blob_bytes, ws_bytes = spense_pack_sizes(H, I, I_dense)
    blob = torch.empty(blob_bytes, dtype=torch.uint8, device=dev)
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
    I_s = I - I_dense
    canon, cstruct = None, None
    if want_canon:
        e = lambda *s: torch.empty(*s, dtype=torch.uint8, device=dev)
        canon = dict(perm=torch.empty(I, dtype=torch.int32, device=dev),
                     gate_sp_val=e(I_s, H // 2), up_sp_val=e(I_s, H // 2), gate_sp_meta=e(I_s, H // 8),
                     up_sp_meta=e(I_s, H // 8), gate_dn=e(I_dense, H), up_dn=e(I_dense, H),
                     down_sp_val=e(H, I_s // 2), down_sp_meta=e(H, I_s // 8), down_dn=e(H, I_dense))
        cstruct = Canon(**{k: v.data_ptr() for k, v in canon.items()})
    if perm is not None:
        _dev(perm, torch.int32)
    scales = (c_float * 3)(*[float(s) for s in w_scale])
    where = (c_int64 * 4)(-1, -1, -1, -1)
    st = lib().spense_pack(ctypes.byref(Shape(H, I, I_dense)), _ptr(wgate), _ptr(wup), _ptr(wdown), scales, _ptr(perm),
                           _ptr(blob), blob_bytes, ctypes.byref(cstruct) if cstruct else None, _ptr(ws), ws_bytes,
                           where, _stream())
    _check(st, tuple(where))
    return PackedLayer(H, I, I_dense, blob, canon)


def spense_workspace_size(H: int, I: int, I_dense: int, M: int) -> int:
    b = c_size_t()
    _check(lib().spense_workspace_size(ctypes.byref(Shape(H, I, I_dense)), M, ctypes.byref(b)))
    return b.value


def spense_workspace(layer: PackedLayer, M: int) -> torch.Tensor:
    """Allocate and initialise a GEMM workspace for up to M tokens."""
    n = spense_workspace_size(layer.H, layer.I, layer.I_dense, M)
    ws = torch.empty(n, dtype=torch.uint8, device=layer.blob.device)
    _check(lib().spense_workspace_init(_ptr(ws), n, _stream()))
    return ws


def spense_gate_up(layer: PackedLayer, x, s_x, s_h, ws, hq=None, h_f32=None):
    """x uint8 [M, H], s_x f32 [M], s_h f32 [1] or [M].  Returns hq uint8 [M, I] (permuted order)."""
    _dev(x, torch.uint8), _dev(s_x, torch.float32), _dev(s_h, torch.float32)
    M = x.shape[0]
    if hq is None:
        hq = torch.empty(M, layer.I, dtype=torch.uint8, device=x.device)
    stride = 0 if s_h.numel() == 1 else 1
    _check(lib().spense_gate_up(ctypes.byref(layer.shape), _ptr(layer.blob), _ptr(x), _ptr(s_x), M, _ptr(s_h), stride,
                                _ptr(hq), _ptr(h_f32), _ptr(ws), ws.numel(), _stream()))
    return hq


def _next(next_layer):
    return None if next_layer is None else c_void_p(next_layer.blob.data_ptr())


def spense_down(layer: PackedLayer, hq, s_h, ws, y=None, dtype=torch.float32, next_layer=None):
    _dev(hq, torch.uint8), _dev(s_h, torch.float32)
    M = hq.shape[0]
    if y is None:
        y = torch.empty(M, layer.H, dtype=dtype, device=hq.device)
    stride = 0 if s_h.numel() == 1 else 1
    _check(lib().spense_down(ctypes.byref(layer.shape), _ptr(layer.blob), _ptr(hq), _ptr(s_h), stride, M, _ptr(y),
                             SPENSE_F32 if y.dtype == torch.float32 else SPENSE_BF16, _ptr(ws), ws.numel(),
                             _next(next_layer), _stream()))
    return y


def spense_mlp(layer: PackedLayer, x, s_x, s_h, ws, hq_scratch=None, y=None, h_f32=None, dtype=torch.float32,
               next_layer=None):
    """next_layer: the PackedLayer that runs next on this stream (same shape) or None -- L2 prefetch hint."""
    _dev(x, torch.uint8), _dev(s_x, torch.float32), _dev(s_h, torch.float32)
    M = x.shape[0]
    if hq_scratch is None:
        hq_scratch = torch.empty(M, layer.I, dtype=torch.uint8, device=x.device)
    if y is None:
        y = torch.empty(M, layer.H, dtype=dtype, device=x.device)
    stride = 0 if s_h.numel() == 1 else 1
    _check(lib().spense_mlp(ctypes.byref(layer.shape), _ptr(layer.blob), _ptr(x), _ptr(s_x), M, _ptr(s_h), stride,
                            _ptr(hq_scratch), _ptr(h_f32), _ptr(y),
                            SPENSE_F32 if y.dtype == torch.float32 else SPENSE_BF16, _ptr(ws), ws.numel(),
                            _next(next_layer), _stream()))
    return y


def spense_mlp_dyn(layer: PackedLayer, x, s_x, ws, s_h=None, hq_scratch=None, h_scratch=None, y=None,
                   dtype=torch.float32, next_layer=None):
    """The layer with dynamic per-token requant: returns (y, s_h [M], hq [M, I], h fp32 [M, I])."""
    _dev(x, torch.uint8), _dev(s_x, torch.float32)
    M = x.shape[0]
    dev = x.device
    s_h = torch.empty(M, dtype=torch.float32, device=dev) if s_h is None else s_h
    hq_scratch = torch.empty(M, layer.I, dtype=torch.uint8, device=dev) if hq_scratch is None else hq_scratch
    h_scratch = torch.empty(M, layer.I, dtype=torch.float32, device=dev) if h_scratch is None else h_scratch
    y = torch.empty(M, layer.H, dtype=dtype, device=dev) if y is None else y
    _check(lib().spense_mlp_dyn(ctypes.byref(layer.shape), _ptr(layer.blob), _ptr(x), _ptr(s_x), M, _ptr(s_h),
                                _ptr(hq_scratch), _ptr(h_scratch), _ptr(y),
                                SPENSE_F32 if y.dtype == torch.float32 else SPENSE_BF16, _ptr(ws), ws.numel(),
                                _ptr(next_layer.blob) if next_layer is not None else None, _stream()))
    return y, s_h, hq_scratch, h_scratch


def spense_mlp_host(layer: PackedLayer, h_x, h_sx, h_sh, h_y, staging, ws, next_layer=None):
    """HOST (pinned) x uint8 [M, H], s_x [M], s_h [1|M] -> HOST y [M, H].  staging = dict of device
    buffers d_x, d_scales, d_hq, d_y.  Synchronises the stream."""
    M = h_x.shape[0]
    stride = 0 if h_sh.numel() == 1 else 1
    _check(lib().spense_mlp_host(ctypes.byref(layer.shape), _ptr(layer.blob), _ptr(h_x), _ptr(h_sx), M, _ptr(h_sh),
                                 stride, _ptr(h_y), SPENSE_F32 if h_y.dtype == torch.float32 else SPENSE_BF16,
                                 _ptr(staging["d_x"]), _ptr(staging["d_scales"]), _ptr(staging["d_hq"]),
                                 _ptr(staging["d_y"]), _ptr(ws), ws.numel(), _next(next_layer), _stream()))
    return h_y


def spense_mlp_stack_host(layers, h_x, h_sx, h_sh, h_y, staging, ws):
    """HOST (pinned) x, s_x, s_h through every PackedLayer of `layers` (same shape) -> HOST y of the last one: one H2D
    copy, len(layers) x spense_mlp, one D2H copy, one synchronise."""
    M = h_x.shape[0]
    stride = 0 if h_sh.numel() == 1 else 1
    blobs = (c_void_p * len(layers))(*[l.blob.data_ptr() for l in layers])
    _check(lib().spense_mlp_stack_host(ctypes.byref(layers[0].shape), blobs, len(layers), _ptr(h_x), _ptr(h_sx), M, _ptr(h_sh),
                                       stride, _ptr(h_y), SPENSE_F32 if h_y.dtype == torch.float32 else SPENSE_BF16,
                                       _ptr(staging["d_x"]), _ptr(staging["d_scales"]), _ptr(staging["d_hq"]),
                                       _ptr(staging["d_y"]), _ptr(ws), ws.numel(), _stream()))
    return h_y


def spense_quantize_e4m3(x: torch.Tensor, mode: int):
    _dev(x, torch.float32)
    rows, cols = x.shape
    out = torch.empty(rows, cols, dtype=torch.uint8, device=x.device)
    scales = torch.empty(rows if mode == SPENSE_PER_ROW else 1, dtype=torch.float32, device=x.device)
    ws = torch.empty((rows + 1) * 4, dtype=torch.uint8, device=x.device)
    _check(lib().spense_quantize_e4m3(_ptr(x), rows, cols, mode, _ptr(out), _ptr(scales), _ptr(ws), ws.numel(), _stream()))
    return out, scales


def spense_quantize_e4m3_static(x: torch.Tensor, mode: int, out: torch.Tensor, scales: torch.Tensor):
    """spense_quantize_e4m3 without a scratch buffer, for callers that must not allocate device memory when they call
    (an engine that already gave all of HBM to its cache pool, a host callback, a latency-critical loop): the scratch is a
    fixed 256 KB array inside libspense.so, so at most SPENSE_QUANTIZE_STATIC_MAX_ROWS rows.  Unlike the other wrappers
    this one creates no tensor either: `out` [rows, cols] uint8 and `scales` [rows] or [1] fp32 are the caller's.
    All calls on a device share that array: keep them ordered on one stream.  Make the first call on a device outside
    stream capture (it looks up the array's address).  Returns (out, scales)."""
    _dev(x, torch.float32)
    rows, cols = x.shape
    n_scales = rows if mode == SPENSE_PER_ROW else 1
    if out.dtype != torch.uint8 or tuple(out.shape) != (rows, cols) or not out.is_contiguous() or out.device != x.device:
        raise ValueError("out must be a contiguous [rows, cols] uint8 tensor on x's device")
    if scales.dtype != torch.float32 or scales.numel() != n_scales or not scales.is_contiguous() or scales.device != x.device:
        raise ValueError("scales must be a contiguous fp32 tensor of rows (per row) or 1 (per tensor) elements on x's device")
    _check(lib().spense_quantize_e4m3_static(_ptr(x), rows, cols, mode, _ptr(out), _ptr(scales), _stream()))
    return out, scales


def spense_probe_read(buf: torch.Tensor, sink: torch.Tensor = None):
    """Stream `buf` (uint8, CUDA, a multiple of 32768 bytes) through the SMs the way the GEMM streams weights and discard
    it; time it with events for the read-only HBM ceiling.  Returns the 256-word sink (XOR of one word per chunk, per CTA)."""
    _dev(buf, torch.uint8)
    if sink is None:
        sink = torch.zeros(256, dtype=torch.int32, device=buf.device)
    _check(lib().spense_probe_read(_ptr(buf), buf.numel(), _ptr(sink), _stream()))
    return sink


def spense_select_dense(wgate, wup, wdown, hdiag_x, hdiag_h, I_dense: int, eps: float = 1e-8):
    """SpenseGPT+ dense-index selection on fp32 weights (CUDA).  Returns (score [I], dense_idx [I_dense], perm [I])."""
    for t in (wgate, wup, wdown, hdiag_x, hdiag_h):
        _dev(t, torch.float32)
    I, H = wgate.shape
    dev = wgate.device
    shape = Shape(H, I, I_dense)
    b = c_size_t()
    _check(lib().spense_select_workspace_size(ctypes.byref(shape), ctypes.byref(b)))
    ws = torch.empty(b.value, dtype=torch.uint8, device=dev)
    score = torch.empty(I, dtype=torch.float32, device=dev)
    dense_idx = torch.empty(I_dense, dtype=torch.int32, device=dev)
    perm = torch.empty(I, dtype=torch.int32, device=dev)
    _check(lib().spense_select_dense(ctypes.byref(shape), _ptr(wgate), _ptr(wup), _ptr(wdown), _ptr(hdiag_x), _ptr(hdiag_h),
                                     c_float(eps), _ptr(score), _ptr(dense_idx) if I_dense else None, _ptr(perm), _ptr(ws),
                                     b.value, _stream()))
    return score, dense_idx, perm


class PackedLinear:
    """One packed Spense linear W [N, K] (out-split or in-split): the opaque device blob plus (optionally) the canonical arrays."""

    def __init__(self, N, K, n_dense, split, blob, canon=None):
        self.N, self.K, self.n_dense, self.split, self.blob, self.canon = N, K, n_dense, split, blob, canon
        self.shape = LinearShape(N, K, n_dense, split)


def spense_pack_linear(w, w_scale: float, perm, n_dense: int, split: int, want_canon: bool = False) -> PackedLinear:
    """w uint8 [N, K] (CUDA, original order); perm int32 over N (out-split) or K (in-split) or None."""
    _dev(w, torch.uint8)
    N, K = w.shape
    dev = w.device
    shape = LinearShape(N, K, n_dense, split)
    b, wsb = c_size_t(), c_size_t()
    _check(lib().spense_linear_pack_sizes(ctypes.byref(shape), ctypes.byref(b), ctypes.byref(wsb)))
    blob = torch.empty(b.value, dtype=torch.uint8, device=dev)
    ws = torch.empty(wsb.value, dtype=torch.uint8, device=dev)
    canon, cstruct = None, None
    if want_canon:
        e = lambda *sh: torch.empty(*sh, dtype=torch.uint8, device=dev)
        if split == SPENSE_SPLIT_OUT:
            n_s = N - n_dense
            canon = dict(perm=torch.empty(N, dtype=torch.int32, device=dev), sp_val=e(n_s, K // 2), sp_meta=e(n_s, K // 8), dn=e(n_dense, K))
        else:
            k_s = K - n_dense
            canon = dict(perm=torch.empty(K, dtype=torch.int32, device=dev), sp_val=e(N, k_s // 2), sp_meta=e(N, k_s // 8), dn=e(N, n_dense))
        cstruct = LinearCanon(**{k: v.data_ptr() for k, v in canon.items()})
    if perm is not None:
        _dev(perm, torch.int32)
    where = (c_int64 * 4)(-1, -1, -1, -1)
    st = lib().spense_pack_linear(ctypes.byref(shape), _ptr(w), c_float(float(w_scale)), _ptr(perm), _ptr(blob), b.value,
                                  ctypes.byref(cstruct) if cstruct else None, _ptr(ws), wsb.value, where, _stream())
    _check(st, tuple(where))
    return PackedLinear(N, K, n_dense, split, blob, canon)


def spense_linear_workspace(lin: PackedLinear, M: int) -> torch.Tensor:
    b = c_size_t()
    _check(lib().spense_linear_workspace_size(ctypes.byref(lin.shape), M, ctypes.byref(b)))
    ws = torch.empty(b.value, dtype=torch.uint8, device=lin.blob.device)
    _check(lib().spense_workspace_init(_ptr(ws), b.value, _stream()))
    return ws


def spense_linear(lin: PackedLinear, x, s_x, ws, y=None, dtype=torch.float32):
    """x uint8 [M, K], s_x f32 [1] or [M] -> y [M, N] = (x W'^T) * s_x * s_w (out-split: permuted row order)."""
    _dev(x, torch.uint8), _dev(s_x, torch.float32)
    M = x.shape[0]
    if y is None:
        y = torch.empty(M, lin.N, dtype=dtype, device=x.device)
    f = lib().spense_linear_out_split if lin.split == SPENSE_SPLIT_OUT else lib().spense_linear_in_split
    _check(f(ctypes.byref(lin.shape), _ptr(lin.blob), _ptr(x), _ptr(s_x), 0 if s_x.numel() == 1 else 1, M, _ptr(y),
             SPENSE_F32 if y.dtype == torch.float32 else SPENSE_BF16, _ptr(ws), ws.numel(), _stream()))
    return y


def spense_prune_obs_2to4(w, u, k_sparse: int):
    """SparseGPT 2:4 column sweep in place on w fp32 [N, K] (CUDA, permuted column order, sparse columns first) with
    u fp32 [K, K] = the upper Cholesky factor of the inverse input Hessian (H^-1 = u^T u).  Returns w."""
    _dev(w, torch.float32), _dev(u, torch.float32)
    N, K = w.shape
    b = c_size_t()
    _check(lib().spense_prune_obs_workspace_size(N, K, ctypes.byref(b)))
    ws = torch.empty(b.value, dtype=torch.uint8, device=w.device)
    _check(lib().spense_prune_obs_2to4(N, K, k_sparse, _ptr(w), _ptr(u), _ptr(ws), b.value, _stream()))
    return w
