"""Thin ctypes binding of libstrata_na3d.so (include/strata_na3d.h): argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels; nothing here computes.  PyTorch
supplies device memory and streams.  There is no CPU fallback: if the library is missing or a call
fails, this raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional, Sequence, Tuple

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libstrata_na3d.so")

STRATA_OK = 0
STRATA_ERR_STATIC_SCRATCH = 5
STATIC_SCRATCH_BYTES = 1 << 20          # STRATA_STATIC_SCRATCH_BYTES of include/strata_na3d.h
DTYPE_F32, DTYPE_BF16 = 0, 1
ROPE_INTERLEAVED, ROPE_HALF = 0, 1
IMPL_AUTO, IMPL_SIMT, IMPL_TCGEN05, IMPL_TCGEN05_TILE = 0, 1, 2, 3

EXPORTS = ("strata_na3d_workspace_bytes", "strata_na3d_host_workspace_bytes", "strata_na3d_impl_selected",
           "strata_na3d_fwd", "strata_na3d_bwd", "strata_na3d_fwd_host", "strata_na3d_bwd_host",
           "strata_na3d_fwd_static",
           "strata_na3d_normgate_workspace_bytes", "strata_na3d_normgate_fwd", "strata_na3d_normgate_bwd",
           "strata_na3d_last_launch_count", "strata_na3d_set_profiling", "strata_na3d_profile_read",
           "strata_na3d_window_start", "strata_na3d_inverse_window", "strata_stereo_coords",
           "strata_wind_to_tile_frame", "strata_tile_stitch", "strata_status_string", "strata_version")


class StrataError(RuntimeError):
    pass


class _CDesc(ctypes.Structure):
    _fields_ = [("batch", ctypes.c_int32), ("heads", ctypes.c_int32), ("head_dim", ctypes.c_int32),
                ("grid", ctypes.c_int32 * 3), ("window", ctypes.c_int32 * 3),
                ("rope_axes", ctypes.c_int32), ("rope_pairing", ctypes.c_int32),
                ("dtype", ctypes.c_int32), ("impl", ctypes.c_int32), ("scale", ctypes.c_float)]


@dataclass(frozen=True)
class NA3DDesc:
    """Mirror of strata_na3d_desc_t."""
    batch: int
    heads: int
    head_dim: int
    grid: Tuple[int, int, int]
    window: Tuple[int, int, int]
    rope_axes: int = 2
    rope_pairing: int = ROPE_INTERLEAVED
    dtype: int = DTYPE_BF16
    impl: int = IMPL_AUTO
    scale: float = 0.0

    def c(self) -> _CDesc:
        return _CDesc(self.batch, self.heads, self.head_dim, (ctypes.c_int32 * 3)(*self.grid),
                      (ctypes.c_int32 * 3)(*self.window), self.rope_axes, self.rope_pairing,
                      self.dtype, self.impl, self.scale)

    @property
    def tensor_shape(self):
        return (self.batch,) + tuple(self.grid) + (self.heads, self.head_dim)

    @property
    def lse_shape(self):
        return (self.batch, self.heads) + tuple(self.grid)

    @property
    def torch_dtype(self):
        return torch.float32 if self.dtype == DTYPE_F32 else torch.bfloat16


_LIB = None


def lib() -> ctypes.CDLL:
    """Load the C-ABI library; fail loudly if it has not been built."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise StrataError(f"{LIB_PATH} is missing: run `python -m paper_2606_31248_b200.build` "
                              "(there is no fallback path)")
        L = ctypes.CDLL(LIB_PATH)
        vp, sz, i32 = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int
        dp = ctypes.POINTER(_CDesc)
        L.strata_na3d_workspace_bytes.restype = sz
        L.strata_na3d_workspace_bytes.argtypes = [dp, i32]
        L.strata_na3d_host_workspace_bytes.restype = sz
        L.strata_na3d_host_workspace_bytes.argtypes = [dp, i32]
        L.strata_na3d_impl_selected.restype = i32
        L.strata_na3d_impl_selected.argtypes = [dp, i32]
        for name in ("strata_na3d_fwd", "strata_na3d_fwd_host"):
            f = getattr(L, name)
            f.restype = i32
            f.argtypes = [dp] + [vp] * 8 + [sz, vp]
        for name in ("strata_na3d_bwd", "strata_na3d_bwd_host"):
            f = getattr(L, name)
            f.restype = i32
            f.argtypes = [dp] + [vp] * 12 + [sz, vp]
        L.strata_na3d_fwd_static.restype = i32
        L.strata_na3d_fwd_static.argtypes = [dp] + [vp] * 7 + [vp]
        L.strata_na3d_normgate_workspace_bytes.restype = sz
        L.strata_na3d_normgate_workspace_bytes.argtypes = [dp, i32]
        L.strata_na3d_normgate_fwd.restype = i32
        L.strata_na3d_normgate_fwd.argtypes = [dp] + [vp] * 6 + [ctypes.c_float] + [vp] * 3 + [sz, vp]
        L.strata_na3d_normgate_bwd.restype = i32
        L.strata_na3d_normgate_bwd.argtypes = [dp] + [vp] * 9 + [ctypes.c_float] + [vp] * 5 + [sz, vp]
        L.strata_na3d_last_launch_count.restype = i32
        L.strata_na3d_set_profiling.restype = None
        L.strata_na3d_set_profiling.argtypes = [i32]
        L.strata_na3d_profile_read.restype = i32
        L.strata_na3d_profile_read.argtypes = [ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_char_p), i32]
        L.strata_na3d_window_start.restype = i32
        L.strata_na3d_window_start.argtypes = [i32, i32, i32]
        L.strata_na3d_inverse_window.restype = i32
        L.strata_na3d_inverse_window.argtypes = [i32, i32, i32, ctypes.POINTER(i32), ctypes.POINTER(i32)]
        L.strata_stereo_coords.restype = i32
        L.strata_stereo_coords.argtypes = [vp, vp, ctypes.c_longlong, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                           vp, i32, vp]
        L.strata_wind_to_tile_frame.restype = i32
        L.strata_wind_to_tile_frame.argtypes = [vp, vp, vp, vp, ctypes.c_longlong, ctypes.c_double, ctypes.c_double,
                                                vp, vp, vp]
        L.strata_tile_stitch.restype = i32
        L.strata_tile_stitch.argtypes = [vp, vp, i32, i32, i32, i32, vp, vp, vp, i32, i32, vp]
        L.strata_status_string.restype = ctypes.c_char_p
        L.strata_status_string.argtypes = [i32]
        L.strata_version.restype = i32
        _LIB = L
    return _LIB


def _check(status: int, what: str):
    if status != STRATA_OK:
        raise StrataError(f"{what}: {lib().strata_status_string(status).decode()} (status {status})")


def _ptr(t) -> Optional[int]:
    """Raw address of a torch tensor (device or host) or None."""
    if t is None:
        return None
    if not isinstance(t, torch.Tensor):
        raise TypeError("expected a torch.Tensor")
    if not t.is_contiguous():
        raise ValueError("tensors must be contiguous")
    return t.data_ptr()


def _stream_handle(stream) -> Optional[int]:
    if stream is None:
        stream = torch.cuda.current_stream()
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream or None
    return int(stream) or None


# ------------------------------------------------------------------ 1:1 wrappers of the C entry points
def strata_version() -> int:
    return int(lib().strata_version())


def strata_na3d_window_start(i: int, k: int, n: int) -> int:
    return int(lib().strata_na3d_window_start(int(i), int(k), int(n)))


def strata_na3d_inverse_window(j: int, k: int, n: int):
    """(lo, hi) inclusive, or None on invalid arguments."""
    lo, hi = ctypes.c_int(0), ctypes.c_int(0)
    if lib().strata_na3d_inverse_window(int(j), int(k), int(n), ctypes.byref(lo), ctypes.byref(hi)) != 0:
        return None
    return lo.value, hi.value


def strata_na3d_workspace_bytes(desc: NA3DDesc, backward: bool = False) -> int:
    return int(lib().strata_na3d_workspace_bytes(ctypes.byref(desc.c()), int(backward)))


def strata_na3d_host_workspace_bytes(desc: NA3DDesc, backward: bool = False) -> int:
    return int(lib().strata_na3d_host_workspace_bytes(ctypes.byref(desc.c()), int(backward)))


def strata_na3d_impl_selected(desc: NA3DDesc, backward: bool = False) -> int:
    return int(lib().strata_na3d_impl_selected(ctypes.byref(desc.c()), int(backward)))


def strata_na3d_last_launch_count() -> int:
    return int(lib().strata_na3d_last_launch_count())


def strata_na3d_set_profiling(enable: bool) -> None:
    lib().strata_na3d_set_profiling(int(bool(enable)))


def strata_na3d_profile_read(capacity: int = 4096):
    """[(kernel name, milliseconds)] of every kernel since profiling was enabled; sync the stream first."""
    ms = (ctypes.c_float * capacity)()
    names = (ctypes.c_char_p * capacity)()
    n = int(lib().strata_na3d_profile_read(ms, names, capacity))
    if n < 0:
        raise StrataError("strata_na3d_profile_read: event query failed")
    return [(names[i].decode(), float(ms[i])) for i in range(min(n, capacity))]


def strata_na3d_fwd_status(desc, q, k, v, coords, freqs, o, lse, workspace, stream=None, host=False) -> int:
    """Raw status code (tests of the error paths use this)."""
    fn = lib().strata_na3d_fwd_host if host else lib().strata_na3d_fwd
    ws_bytes = workspace.numel() * workspace.element_size() if workspace is not None else 0
    return int(fn(ctypes.byref(desc.c()), _ptr(q), _ptr(k), _ptr(v), _ptr(coords), _ptr(freqs), _ptr(o),
                  _ptr(lse), _ptr(workspace), ws_bytes, _stream_handle(stream)))


def strata_na3d_bwd_status(desc, q, k, v, o, d_o, lse, coords, freqs, dq, dk, dv, workspace, stream=None,
                           host=False) -> int:
    fn = lib().strata_na3d_bwd_host if host else lib().strata_na3d_bwd
    ws_bytes = workspace.numel() * workspace.element_size() if workspace is not None else 0
    return int(fn(ctypes.byref(desc.c()), _ptr(q), _ptr(k), _ptr(v), _ptr(o), _ptr(d_o), _ptr(lse),
                  _ptr(coords), _ptr(freqs), _ptr(dq), _ptr(dk), _ptr(dv), _ptr(workspace), ws_bytes,
                  _stream_handle(stream)))


def strata_na3d_fwd(desc, q, k, v, coords, freqs, o, lse, workspace, stream=None):
    _check(strata_na3d_fwd_status(desc, q, k, v, coords, freqs, o, lse, workspace, stream), "strata_na3d_fwd")


def strata_na3d_fwd_static_status(desc, q, k, v, coords, freqs, o, lse, stream=None) -> int:
    """Raw status of strata_na3d_fwd_static (no workspace argument: the library's own fixed array is the scratch)."""
    return int(lib().strata_na3d_fwd_static(ctypes.byref(desc.c()), _ptr(q), _ptr(k), _ptr(v), _ptr(coords), _ptr(freqs),
                                            _ptr(o), _ptr(lse), _stream_handle(stream)))


def strata_na3d_fwd_static(desc, q, k, v, coords, freqs, o, lse, stream=None):
    """The forward for a caller that cannot allocate device memory (it lives inside a host whose pool owns the GPU, or
    may not disturb a running loop with cudaMalloc's synchronisation): same kernels and results as strata_na3d_fwd,
    scratch in a 1 MiB array inside the library.  Raises StrataError (status 5) when the problem needs more than
    STATIC_SCRATCH_BYTES of scratch; calls that may overlap on one GPU race on the array -- keep them on one stream."""
    _check(strata_na3d_fwd_static_status(desc, q, k, v, coords, freqs, o, lse, stream), "strata_na3d_fwd_static")


def strata_na3d_bwd(desc, q, k, v, o, d_o, lse, coords, freqs, dq, dk, dv, workspace, stream=None):
    _check(strata_na3d_bwd_status(desc, q, k, v, o, d_o, lse, coords, freqs, dq, dk, dv, workspace, stream),
           "strata_na3d_bwd")


def strata_na3d_normgate_workspace_bytes(desc, backward: bool) -> int:
    return int(lib().strata_na3d_normgate_workspace_bytes(ctypes.byref(desc.c()), 1 if backward else 0))


def strata_na3d_normgate_fwd(desc, q, k, v, coords, freqs, gate, eps, o, lse, workspace, stream=None):
    """QK-RMSNorm -> StereoRoPE + NA3D -> sigmoid head gate (gate: float32 [B,L,Y,X,H] logits or None)."""
    ws_bytes = workspace.numel() * workspace.element_size() if workspace is not None else 0
    _check(int(lib().strata_na3d_normgate_fwd(ctypes.byref(desc.c()), _ptr(q), _ptr(k), _ptr(v), _ptr(coords), _ptr(freqs),
                                              _ptr(gate), float(eps), _ptr(o), _ptr(lse), _ptr(workspace), ws_bytes,
                                              _stream_handle(stream))), "strata_na3d_normgate_fwd")


def strata_na3d_normgate_bwd(desc, q, k, v, o, d_o, lse, coords, freqs, gate, eps, dq, dk, dv, dgate, workspace,
                             stream=None):
    ws_bytes = workspace.numel() * workspace.element_size() if workspace is not None else 0
    _check(int(lib().strata_na3d_normgate_bwd(ctypes.byref(desc.c()), _ptr(q), _ptr(k), _ptr(v), _ptr(o), _ptr(d_o),
                                              _ptr(lse), _ptr(coords), _ptr(freqs), _ptr(gate), float(eps), _ptr(dq),
                                              _ptr(dk), _ptr(dv), _ptr(dgate), _ptr(workspace), ws_bytes,
                                              _stream_handle(stream))), "strata_na3d_normgate_bwd")


def strata_na3d_fwd_host(desc, q, k, v, coords, freqs, o, lse, workspace, stream=None):
    _check(strata_na3d_fwd_status(desc, q, k, v, coords, freqs, o, lse, workspace, stream, host=True),
           "strata_na3d_fwd_host")


def strata_na3d_bwd_host(desc, q, k, v, o, d_o, lse, coords, freqs, dq, dk, dv, workspace, stream=None):
    _check(strata_na3d_bwd_status(desc, q, k, v, o, d_o, lse, coords, freqs, dq, dk, dv, workspace, stream,
                                  host=True), "strata_na3d_bwd_host")


# ------------------------------------------------------------------ geometry
def strata_stereo_coords(lat, lon, lat0: float, lon0: float, n_total: float, coords, stride: int = 2, stream=None):
    """Eq. (1) on the device: lat, lon float64 CUDA tensors of n points -> coords[i * stride + {0, 1}] (float32)."""
    n = lat.numel()
    if lon.numel() != n or lat.dtype != torch.float64 or lon.dtype != torch.float64 or coords.dtype != torch.float32:
        raise TypeError("lat, lon: float64 tensors of equal size; coords: float32")
    if coords.numel() < n * stride:
        raise ValueError("coords too small")
    _check(lib().strata_stereo_coords(_ptr(lat), _ptr(lon), n, float(lat0), float(lon0), float(n_total), _ptr(coords),
                                      int(stride), _stream_handle(stream)), "strata_stereo_coords")


def strata_wind_to_tile_frame(u, v, lat, lon, lat0: float, lon0: float, u_loc, v_loc, stream=None):
    """Eq. (2) on the device: winds (u, v) float32 at (lat, lon) float64 -> (u_loc, v_loc) float32."""
    n = u.numel()
    for t, dt in ((u, torch.float32), (v, torch.float32), (u_loc, torch.float32), (v_loc, torch.float32),
                  (lat, torch.float64), (lon, torch.float64)):
        if t.numel() != n or t.dtype != dt:
            raise TypeError("u, v, u_loc, v_loc: float32; lat, lon: float64; all of one size")
    _check(lib().strata_wind_to_tile_frame(_ptr(u), _ptr(v), _ptr(lat), _ptr(lon), n, float(lat0), float(lon0),
                                           _ptr(u_loc), _ptr(v_loc), _stream_handle(stream)), "strata_wind_to_tile_frame")


def strata_tile_stitch(tiles, origins, wy, wx, out, stream=None):
    """Eq. (5) on the device: tiles [T,C,th,tw] f32, origins [T,2] int32, windows wy [th], wx [tw], out [C,gh,gw] f32."""
    T, C, th, tw = tiles.shape
    if origins.dtype != torch.int32 or tuple(origins.shape) != (T, 2) or wy.numel() != th or wx.numel() != tw:
        raise TypeError("origins: int32 [T, 2]; wy [th]; wx [tw]")
    for t in (tiles, wy, wx, out):
        if t.dtype != torch.float32:
            raise TypeError("tiles, windows and out are float32")
    _check(lib().strata_tile_stitch(_ptr(tiles), _ptr(origins), T, C, th, tw, _ptr(wy), _ptr(wx), _ptr(out), out.shape[1],
                                    out.shape[2], _stream_handle(stream)), "strata_tile_stitch")


# ------------------------------------------------------------------ convenience: allocate + call
def desc_for(q: torch.Tensor, window: Sequence[int], rope_axes: int, rope_pairing: int = ROPE_INTERLEAVED,
             scale: float = 0.0, impl: int = IMPL_AUTO) -> NA3DDesc:
    if q.dim() != 6:
        raise ValueError("q must be [B, L, Y, X, H, d]")
    if q.dtype not in (torch.float32, torch.bfloat16):
        raise TypeError("dtype must be float32 or bfloat16")
    B, L, Y, X, H, D = q.shape
    return NA3DDesc(B, H, D, (L, Y, X), tuple(int(w) for w in window), rope_axes, rope_pairing,
                    DTYPE_F32 if q.dtype == torch.float32 else DTYPE_BF16, impl, float(scale))


def fixup_stats(workspace: torch.Tensor):
    """(rows listed for the exact fix-up kernel, take-all flag) that the last tensor-core FORWARD left at the head of
    `workspace` (include/strata_na3d.h, "exponent range"); synchronises.  Meaningless after a SIMT call."""
    head = workspace[:16].view(torch.int64).cpu()
    return int(head[0]), bool(head[1] != 0)


def alloc_workspace(nbytes: int, device) -> torch.Tensor:
    return torch.empty(max(int(nbytes), 16), dtype=torch.uint8, device=device)


def na3d_forward(q, k, v, coords, freqs, window, rope_pairing=ROPE_INTERLEAVED, scale=0.0, impl=IMPL_AUTO,
                 workspace=None, stream=None):
    """StereoRoPE + NA3D forward on device tensors.  Returns (o, lse).
    A workspace allocated here (workspace=None) comes from torch's caching allocator on the CURRENT torch stream:
    pass your own workspace when `stream` is another stream."""
    if not q.is_cuda:
        raise StrataError("na3d_forward needs CUDA tensors (there is no CPU path)")
    rope_axes = 0 if coords is None else coords.shape[-1]
    desc = desc_for(q, window, rope_axes, rope_pairing, scale, impl)
    o = torch.empty_like(q)
    lse = torch.empty(desc.lse_shape, dtype=torch.float32, device=q.device)
    if workspace is None:
        workspace = alloc_workspace(strata_na3d_workspace_bytes(desc, False), q.device)
    strata_na3d_fwd(desc, q, k, v, coords, freqs, o, lse, workspace, stream)
    return o, lse


def na3d_backward(q, k, v, o, d_o, lse, coords, freqs, window, rope_pairing=ROPE_INTERLEAVED, scale=0.0,
                  impl=IMPL_AUTO, workspace=None, stream=None):
    """StereoRoPE + NA3D backward on device tensors.  Returns (dq, dk, dv)."""
    if not q.is_cuda:
        raise StrataError("na3d_backward needs CUDA tensors (there is no CPU path)")
    rope_axes = 0 if coords is None else coords.shape[-1]
    desc = desc_for(q, window, rope_axes, rope_pairing, scale, impl)
    dq, dk, dv = torch.empty_like(q), torch.empty_like(q), torch.empty_like(q)
    if workspace is None:
        workspace = alloc_workspace(strata_na3d_workspace_bytes(desc, True), q.device)
    strata_na3d_bwd(desc, q, k, v, o, d_o, lse, coords, freqs, dq, dk, dv, workspace, stream)
    return dq, dk, dv
