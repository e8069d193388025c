"""CPU float64 ORACLE for StereoRoPE + 3D neighbourhood attention -- TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs
may import this package.  The product (`paper_2606_31248_b200`) never does, and this package never
imports the product's CUDA path; the only shared module is the seeded input generator
`paper_2606_31248_b200.workloads`, which the callers use, not this package.

The arithmetic lives in `na3d_oracle.c` (plain C, float64, the paper's definition written out;
see that file's header for the passages it follows); this file only marshals numpy arrays.
Parity status: every function below is pinned by tests/test_oracle_pins.py (no "parity unpinned"
function); the *conventions* the paper does not state (readings R4-R11: frequency
schedule, pair-to-axis map, N_total, cube-face orientation) cannot be pinned against the authors'
code, which is not available -- they live in the input generator, not here.
"""
from __future__ import annotations

import ctypes
from typing import Optional, Sequence, Tuple

import numpy as np

from . import build as _build
from . import geometry  # noqa: F401
from . import normgate as _normgate
from . import stitch  # noqa: F401

_LIB = None

DT_F64, DT_F32, DT_BF16 = 0, 1, 2


class _Desc(ctypes.Structure):
    _fields_ = [("B", ctypes.c_int32), ("H", ctypes.c_int32), ("D", ctypes.c_int32),
                ("L", ctypes.c_int32), ("Y", ctypes.c_int32), ("X", ctypes.c_int32),
                ("kL", ctypes.c_int32), ("kY", ctypes.c_int32), ("kX", ctypes.c_int32),
                ("A", ctypes.c_int32), ("pairing", ctypes.c_int32), ("dtype", ctypes.c_int32),
                ("scale", ctypes.c_double)]


def lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(_build.build())
        _LIB.oracle_window_start.restype = ctypes.c_int
        _LIB.oracle_num_threads.restype = ctypes.c_int
    return _LIB


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def window_start(i: int, k: int, n: int) -> int:
    return int(lib().oracle_window_start(int(i), int(k), int(n)))


def _tag(x: np.ndarray) -> int:
    if x.dtype == np.float64:
        return DT_F64
    if x.dtype == np.float32:
        return DT_F32
    if x.dtype == np.uint16:
        return DT_BF16
    raise TypeError(f"oracle input dtype {x.dtype}: want float64, float32 or uint16 (bf16 bits)")


def _ptr(x: np.ndarray):
    return x.ctypes.data_as(ctypes.c_void_p)


def _prep(q, k, v, coords, freqs, window, scale, pairing, extra=()):
    q = np.ascontiguousarray(q)
    tag = _tag(q)
    arrs = [np.ascontiguousarray(t) for t in (k, v) + tuple(extra)]
    for t in arrs:
        if _tag(t) != tag or t.shape != q.shape:
            raise ValueError("q, k, v (, do) must share dtype and shape")
    B, L, Y, X, H, D = q.shape
    coords = np.ascontiguousarray(coords, dtype=np.float32)
    freqs = np.ascontiguousarray(freqs, dtype=np.float32)
    A = coords.shape[-1] if coords.size else 0
    if A:
        assert coords.shape == (B, L, Y, X, A) and freqs.shape == (A, D // 2)
    for kk, n in zip(window, (L, Y, X)):
        if not 1 <= kk <= n:
            raise ValueError("window must satisfy 1 <= k_a <= n_a")
    d = _Desc(B, H, D, L, Y, X, int(window[0]), int(window[1]), int(window[2]), A, int(pairing), tag,
              float(scale) if scale else 0.0)
    return d, q, arrs, coords, freqs


def rope_rotate(x, coords, freqs, pairing: int = 0, sign: float = 1.0) -> np.ndarray:
    """A1 + A2: rotate every head vector of x [B,L,Y,X,H,D] by the angles of its token."""
    x = np.ascontiguousarray(x)
    B, L, Y, X, H, D = x.shape
    coords = np.ascontiguousarray(coords, dtype=np.float32)
    freqs = np.ascontiguousarray(freqs, dtype=np.float32)
    A = coords.shape[-1] if coords.size else 0
    d = _Desc(B, H, D, L, Y, X, 1, 1, 1, A, int(pairing), _tag(x), 0.0)
    out = np.empty(x.shape, dtype=np.float64)
    lib().oracle_rope_rotate(ctypes.byref(d), _ptr(x), _ptr(coords), _ptr(freqs),
                             ctypes.c_double(sign), _ptr(out))
    return out


def na3d_fwd(q, k, v, coords, freqs, window: Sequence[int], scale: Optional[float] = None,
             pairing: int = 0) -> Tuple[np.ndarray, np.ndarray]:
    """A1-A6 on the whole tensor.  Returns (o [B,L,Y,X,H,D], lse [B,H,L,Y,X]) in float64."""
    d, q, (k, v), coords, freqs = _prep(q, k, v, coords, freqs, window, scale, pairing)
    o = np.empty(q.shape, dtype=np.float64)
    lse = np.empty((d.B, d.H, d.L, d.Y, d.X), dtype=np.float64)
    rc = lib().oracle_na3d_fwd(ctypes.byref(d), _ptr(q), _ptr(k), _ptr(v), _ptr(coords), _ptr(freqs),
                               _ptr(o), _ptr(lse))
    if rc:
        raise MemoryError("oracle_na3d_fwd")
    return o, lse


def na3d_fwd_queries(q, k, v, coords, freqs, window, idx, scale=None, pairing: int = 0):
    """A1-A6 for the (b, token, h) rows idx (flat index (b*N + token)*H + h).
    Returns (o [n, D], lse [n]) in float64."""
    d, q, (k, v), coords, freqs = _prep(q, k, v, coords, freqs, window, scale, pairing)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    o = np.empty((idx.size, d.D), dtype=np.float64)
    lse = np.empty((idx.size,), dtype=np.float64)
    lib().oracle_na3d_fwd_queries(ctypes.byref(d), _ptr(q), _ptr(k), _ptr(v), _ptr(coords),
                                  _ptr(freqs), ctypes.c_longlong(idx.size), _ptr(idx), _ptr(o), _ptr(lse))
    return o, lse


def na3d_bwd(q, k, v, d_o, coords, freqs, window, scale=None, pairing: int = 0):
    """B1-B4 on the whole tensor.  Returns (dq, dk, dv) in float64."""
    d, q, (k, v, d_o), coords, freqs = _prep(q, k, v, coords, freqs, window, scale, pairing, (d_o,))
    dq = np.empty(q.shape, dtype=np.float64)
    dk = np.empty(q.shape, dtype=np.float64)
    dv = np.empty(q.shape, dtype=np.float64)
    rc = lib().oracle_na3d_bwd(ctypes.byref(d), _ptr(q), _ptr(k), _ptr(v), _ptr(d_o), _ptr(coords),
                               _ptr(freqs), _ptr(dq), _ptr(dk), _ptr(dv))
    if rc:
        raise MemoryError("oracle_na3d_bwd")
    return dq, dk, dv


def na3d_bwd_rows(q, k, v, d_o, coords, freqs, window, idx, scale=None, pairing: int = 0):
    """B1-B4 for sampled rows idx (flat (b, token, h)): dq of the row as a query, dk / dv of the
    row as a key (brute force over all queries).  Returns (dq, dk, dv) each [n, D] float64."""
    d, q, (k, v, d_o), coords, freqs = _prep(q, k, v, coords, freqs, window, scale, pairing, (d_o,))
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    outs = [np.empty((idx.size, d.D), dtype=np.float64) for _ in range(3)]
    lib().oracle_na3d_bwd_rows(ctypes.byref(d), _ptr(q), _ptr(k), _ptr(v), _ptr(d_o), _ptr(coords),
                               _ptr(freqs), ctypes.c_longlong(idx.size), _ptr(idx),
                               _ptr(outs[0]), _ptr(outs[1]), _ptr(outs[2]))
    return tuple(outs)


def na3d_normgate_fwd(q, k, v, gate, coords, freqs, window, eps: float = 1e-6, scale=None, pairing: int = 0):
    """QK-RMSNorm -> StereoRoPE + NA3D -> sigmoid head gate.  Returns (o, lse, a) (oracle/normgate.py)."""
    return _normgate.fwd(na3d_fwd, q, k, v, gate, coords, freqs, window, eps, scale, pairing)


def na3d_normgate_bwd(q, k, v, gate, d_o, coords, freqs, window, eps: float = 1e-6, scale=None, pairing: int = 0):
    """Gradients of the above wrt q, k, v and the gate logits: (dq, dk, dv, dgate)."""
    return _normgate.bwd(na3d_fwd, na3d_bwd, q, k, v, gate, d_o, coords, freqs, window, eps, scale, pairing)
