"""ORACLE (test infrastructure only): QK-RMSNorm and the head-specific sigmoid gate around the attention,
PAPER.md:390 (App. B.5): "QK RMSNorm [55], which applies RMSNorm (without learnable scale) to the query and key
vectors before their dot product" and "gated attention [56], which applies a head-specific sigmoid gate to the
attention output".  Plain numpy float64 around the C oracle's attention (oracle.na3d_fwd / na3d_bwd).

Readings (R23, R24): RMSNorm over the head_dim channels of one (token, head) vector,
x^ = x / sqrt(mean_c x_c^2 + eps), applied BEFORE StereoRoPE (the rotation is orthogonal, so the order does not change
the result); the gate is one logit per (token, head), o = sigmoid(g) * a, a the attention output; LSE is that of the
normalised logits.  Backward: plain chain rule, written out.
"""
from __future__ import annotations

import numpy as np


def _f64(x):
    """Exact float64 values of a float64 / float32 / bf16-bit-pattern (uint16) array."""
    x = np.asarray(x)
    if x.dtype == np.uint16:
        return (x.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)
    return x.astype(np.float64)


def rmsnorm(x, eps):
    x = _f64(x)
    return x / np.sqrt(np.mean(x * x, axis=-1, keepdims=True) + eps)


def sigmoid(g):
    g = np.asarray(g, dtype=np.float64)
    return 1.0 / (1.0 + np.exp(-g))


def fwd(na3d_fwd, q, k, v, gate, coords, freqs, window, eps=1e-6, scale=None, pairing=0):
    """Returns (o, lse, a): gated output, LSE, un-gated attention output (float64).  gate: [B,L,Y,X,H] logits or None."""
    qh, kh = rmsnorm(q, eps), rmsnorm(k, eps)
    a, lse = na3d_fwd(qh, kh, _f64(v), coords, freqs, window, scale=scale, pairing=pairing)
    o = a if gate is None else sigmoid(gate)[..., None] * a
    return o, lse, a


def bwd(na3d_fwd, na3d_bwd, q, k, v, gate, d_o, coords, freqs, window, eps=1e-6, scale=None, pairing=0):
    """Returns (dq, dk, dv, dgate) in float64 (dgate None without a gate)."""
    q, k, v, d_o = _f64(q), _f64(k), _f64(v), _f64(d_o)
    rq = 1.0 / np.sqrt(np.mean(q * q, axis=-1, keepdims=True) + eps)
    rk = 1.0 / np.sqrt(np.mean(k * k, axis=-1, keepdims=True) + eps)
    qh, kh = q * rq, k * rk
    if gate is None:
        da, dgate = d_o, None
    else:
        a, _ = na3d_fwd(qh, kh, v, coords, freqs, window, scale=scale, pairing=pairing)
        s = sigmoid(gate)
        da = s[..., None] * d_o                                    # o = s a
        dgate = s * (1.0 - s) * np.sum(d_o * a, axis=-1)
    dqh, dkh, dv = na3d_bwd(qh, kh, v, da, coords, freqs, window, scale=scale, pairing=pairing)
    # x^ = x r, r = (mean x^2 + eps)^(-1/2):  dx_c = r (dx^_c - x^_c mean_j(x^_j dx^_j))
    dq = rq * (dqh - qh * np.mean(qh * dqh, axis=-1, keepdims=True))
    dk = rk * (dkh - kh * np.mean(kh * dkh, axis=-1, keepdims=True))
    return dq, dk, dv, dgate
