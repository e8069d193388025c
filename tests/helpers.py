"""Shared test plumbing: numpy <-> torch device tensors, the parity tolerances."""
from __future__ import annotations

import numpy as np
import torch

from paper_2606_31248_b200 import binding, workloads as wl


def to_device(x: np.ndarray, dtype: str, device="cuda") -> torch.Tensor:
    if dtype == "bf16":
        return torch.from_numpy(x.view(np.int16)).to(device).view(torch.bfloat16)
    return torch.from_numpy(x).to(device)


def to_f64(t: torch.Tensor) -> np.ndarray:
    return t.detach().to("cpu", torch.float64).numpy()


def device_inputs(w: wl.Workload, inp, device="cuda"):
    d = {n: to_device(inp[n], w.dtype, device) for n in ("q", "k", "v", "do") if n in inp}
    d["coords"] = torch.from_numpy(inp["coords"]).to(device) if w.rope_axes else None
    d["freqs"] = torch.from_numpy(inp["freqs"]).to(device) if w.rope_axes else None
    return d


def desc_of(w: wl.Workload, impl=binding.IMPL_AUTO, scale=0.0) -> binding.NA3DDesc:
    return binding.NA3DDesc(w.batch, w.heads, w.head_dim, w.grid, w.window, w.rope_axes, w.rope_pairing,
                            binding.DTYPE_F32 if w.dtype == "f32" else binding.DTYPE_BF16, impl, scale)


# BASELINE.json north_star: fp32 max-abs 1e-4; bf16 |err| <= 2e-2 + 1e-2 |ref|.
# On top of that DESIGN.md §6 derives a relative-RMS bound that an all-zero output cannot pass:
# fp32 path 1e-5, bf16 path 1e-2 (bf16 rounding of qrot, krot, P and of the output, 2^-9 each).
def assert_parity(got: np.ndarray, ref: np.ndarray, dtype: str, what: str, rms_bound=None):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape, (what, got.shape, ref.shape)
    assert np.all(np.isfinite(got)), f"{what}: non-finite values"
    err = np.abs(got - ref)
    if dtype == "f32":
        assert err.max() <= 1e-4, f"{what}: max abs err {err.max():.3e} > 1e-4"
        bound = 1e-5 if rms_bound is None else rms_bound
    else:
        viol = err - (2e-2 + 1e-2 * np.abs(ref))
        assert viol.max() <= 0, f"{what}: allclose(2e-2, 1e-2) violated by {viol.max():.3e} (max abs err {err.max():.3e})"
        bound = 1e-2 if rms_bound is None else rms_bound
    denom = np.sqrt(np.mean(ref ** 2))
    rel_rms = np.sqrt(np.mean(err ** 2)) / max(denom, 1e-300)
    assert rel_rms <= bound, f"{what}: relative RMS err {rel_rms:.3e} > {bound:g}"
    return float(err.max()), float(rel_rms)
