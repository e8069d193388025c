"""GPU parity: the CUDA path through the C ABI against the CPU float64 oracle, element by element."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2606_31248_b200 import binding, workloads as wl
from helpers import assert_parity, desc_of, device_inputs, to_f64

pytestmark = pytest.mark.gpu

IMPLS = [binding.IMPL_SIMT, binding.IMPL_AUTO, binding.IMPL_TCGEN05_TILE]


def run_fwd(w, inp, impl=binding.IMPL_AUTO, scale=0.0):
    d = device_inputs(w, inp)
    desc = desc_of(w, impl, scale)
    o = torch.empty_like(d["q"])
    lse = torch.empty(desc.lse_shape, dtype=torch.float32, device="cuda")
    ws = binding.alloc_workspace(binding.strata_na3d_workspace_bytes(desc, False), "cuda")
    binding.strata_na3d_fwd(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], o, lse, ws)
    torch.cuda.synchronize()
    return d, o, lse


def run_bwd(w, inp, d, o, lse, impl=binding.IMPL_AUTO, scale=0.0):
    desc = desc_of(w, impl, scale)
    dq, dk, dv = (torch.empty_like(d["q"]) for _ in range(3))
    ws = binding.alloc_workspace(binding.strata_na3d_workspace_bytes(desc, True), "cuda")
    binding.strata_na3d_bwd(desc, d["q"], d["k"], d["v"], o, d["do"], lse, d["coords"], d["freqs"], dq, dk, dv, ws)
    torch.cuda.synchronize()
    return dq, dk, dv


def check_full(oracle_mod, w, impl, backward=True, scale=0.0):
    inp = wl.make_inputs(w, with_do=True)
    d, o, lse = run_fwd(w, inp, impl, scale)
    coords = inp["coords"] if w.rope_axes else np.zeros((w.batch,) + w.grid + (0,), np.float32)
    o_ref, lse_ref = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], coords, inp["freqs"], w.window,
                                         scale=scale or None, pairing=w.rope_pairing)
    assert_parity(to_f64(o), o_ref, w.dtype, f"{w.name} O")
    assert_parity(to_f64(lse), lse_ref, "f32" if w.dtype == "f32" else "bf16", f"{w.name} LSE", rms_bound=1e-2)
    if backward:
        dq, dk, dv = run_bwd(w, inp, d, o, lse, impl, scale)
        rq, rk, rv = oracle_mod.na3d_bwd(inp["q"], inp["k"], inp["v"], inp["do"], coords, inp["freqs"], w.window,
                                         scale=scale or None, pairing=w.rope_pairing)
        # the GPU backward starts from the GPU's rounded O (bf16): allow 2e-2 relative RMS there
        rb = None if w.dtype == "f32" else 2e-2
        assert_parity(to_f64(dq), rq, w.dtype, f"{w.name} dQ", rms_bound=rb)
        assert_parity(to_f64(dk), rk, w.dtype, f"{w.name} dK", rms_bound=rb)
        assert_parity(to_f64(dv), rv, w.dtype, f"{w.name} dV", rms_bound=rb)


# ------------------------------------------------------------------ BASELINE.json configs
@pytest.mark.parametrize("impl", IMPLS[:2])
def test_config0_tiny_fp32_fwd_bwd(oracle_mod, impl):
    check_full(oracle_mod, wl.config(0), impl)


@pytest.mark.parametrize("impl", IMPLS)
def test_config1_bf16_fwd_full(oracle_mod, impl):
    check_full(oracle_mod, wl.config(1), impl, backward=False)


def test_config4_bf16_bwd_full(oracle_mod):
    w = wl.config(4)
    inp = wl.make_inputs(w, with_do=True)
    d, o, lse = run_fwd(w, inp)
    dq, dk, dv = run_bwd(w, inp, d, o, lse)
    rq, rk, rv = oracle_mod.na3d_bwd(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window)
    for got, ref, nm in ((dq, rq, "dQ"), (dk, rk, "dK"), (dv, rv, "dV")):
        assert_parity(to_f64(got), ref, "bf16", f"cfg4 {nm}", rms_bound=2e-2)


def _full_fwd_by_sample(oracle_mod, w):
    """Every element of O and LSE of a big config: one GPU call, the oracle one batch element at a time."""
    inp = wl.make_inputs(w)
    d, o, lse = run_fwd(w, inp)
    assert bool(torch.isfinite(o.float()).all()) and bool(torch.isfinite(lse).all())
    worst = (0.0, 0.0)
    for b in range(w.batch):
        sl = slice(b, b + 1)
        o_ref, lse_ref = oracle_mod.na3d_fwd(inp["q"][sl], inp["k"][sl], inp["v"][sl], inp["coords"][sl], inp["freqs"],
                                             w.window)
        e = assert_parity(to_f64(o[sl]), o_ref, w.dtype, f"{w.name} O[{b}]")
        assert_parity(to_f64(lse[sl]), lse_ref, "bf16", f"{w.name} LSE[{b}]", rms_bound=1e-2)
        worst = (max(worst[0], e[0]), max(worst[1], e[1]))
        del o_ref, lse_ref
    print(f"{w.name}: every element of {w.batch} samples, O max-abs err {worst[0]:.3e}, rel-rms {worst[1]:.3e}")


def test_config2_bf16_wide_head_full(oracle_mod):
    _full_fwd_by_sample(oracle_mod, wl.config(2))


def test_config3_bf16_global_rollout_full(oracle_mod):
    _full_fwd_by_sample(oracle_mod, wl.config(3))


# ------------------------------------------------------------------ shape / option sweep
SWEEP = [
    dict(grid=(3, 6, 7), window=(3, 3, 3), heads=2, head_dim=32),
    dict(grid=(5, 9, 11), window=(3, 5, 7), heads=3, head_dim=64, batch=2),
    dict(grid=(2, 10, 9), window=(2, 4, 6), heads=1, head_dim=32),                 # even windows
    dict(grid=(4, 5, 6), window=(4, 5, 6), heads=2, head_dim=32),                  # window = grid: dense
    dict(grid=(3, 5, 5), window=(1, 1, 1), heads=2, head_dim=32),                  # k = 1
    dict(grid=(1, 12, 13), window=(1, 5, 5), heads=2, head_dim=64),                # 2D
    dict(grid=(1, 1, 40), window=(1, 1, 9), heads=2, head_dim=32),                 # 1D
    dict(grid=(9, 17, 19), window=(5, 9, 9), heads=2, head_dim=128),               # wide head, ragged tiles
    dict(grid=(3, 6, 7), window=(3, 3, 3), heads=2, head_dim=32, rope_pairing=1),  # HALF pairing
    dict(grid=(3, 6, 7), window=(3, 3, 3), heads=2, head_dim=64, rope_pairing=1),
    dict(grid=(4, 6, 7), window=(3, 3, 3), heads=2, head_dim=32, rope_axes=3),     # level axis rotated too
    dict(grid=(3, 6, 7), window=(3, 3, 3), heads=2, head_dim=32, rope_axes=0),     # no RoPE
    dict(grid=(8, 18, 21), window=(3, 7, 7), heads=2, head_dim=64, batch=2),       # several tiles + ragged tail
    dict(grid=(5, 13, 10), window=(3, 5, 5), heads=2, head_dim=64),                # tcgen05 (3,5,5), odd L
    dict(grid=(3, 7, 7), window=(3, 7, 7), heads=1, head_dim=64),                  # tcgen05, window = grid < tile
    dict(grid=(7, 9, 23), window=(3, 3, 3), heads=3, head_dim=64, rope_pairing=1), # tcgen05 (3,3,3), HALF
    dict(grid=(6, 16, 16), window=(5, 9, 9), heads=2, head_dim=128, batch=2),      # tcgen05 d=128, exact tiles
    dict(grid=(2, 40, 9), window=(1, 7, 7), heads=1, head_dim=64),                 # (1,7,7): SIMT fallback
    dict(grid=(8, 24, 32), window=(3, 7, 7), heads=2, head_dim=64, rope_axes=3),   # tcgen05 + 3-axis RoPE
    dict(grid=(4, 9, 10), window=(3, 5, 5), heads=2, head_dim=64),                 # level sweep, 2 tiles
    dict(grid=(6, 17, 9), window=(3, 3, 3), heads=2, head_dim=64, batch=2),        # level sweep, 3 tiles
    dict(grid=(10, 20, 12), window=(3, 7, 7), heads=1, head_dim=64),               # level sweep, 5 tiles
    dict(grid=(3, 8, 8), window=(3, 7, 7), heads=2, head_dim=64),                  # level sweep, L = k_L
    dict(grid=(12, 7, 30), window=(3, 7, 7), heads=1, head_dim=64),                # level sweep, Y = k_Y
    dict(grid=(4, 20, 20), window=(3, 7, 7), heads=2, head_dim=64),                # tcgen05 bwd: inverse halo wider than one chunk
    dict(grid=(7, 12, 20), window=(3, 5, 5), heads=1, head_dim=64, batch=2),       # tcgen05 bwd (3,5,5), odd L, ragged y
    dict(grid=(8, 18, 21), window=(3, 7, 7), heads=2, head_dim=64, rope_axes=0),   # tcgen05 without RoPE (fused fwd, bwd without table)
    dict(grid=(5, 9, 12), window=(3, 3, 3), heads=2, head_dim=64, rope_axes=0, rope_pairing=1),
    dict(grid=(6, 16, 16), window=(5, 9, 9), heads=1, head_dim=128, rope_axes=0),  # d=128 tile kernel without RoPE
]


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("case", range(len(SWEEP)))
def test_shape_sweep_fwd_bwd(oracle_mod, case, dtype):
    w = wl.small(name=f"sweep{case}_{dtype}", dtype=dtype, **SWEEP[case])
    check_full(oracle_mod, w, binding.IMPL_AUTO)


@pytest.mark.parametrize("rope_axes", [0, 2, 3])
def test_tile_kernel_forced(oracle_mod, rope_axes):
    """IMPL_TCGEN05_TILE: the one-tile-per-CTA forward on pre-rotated operands, where AUTO takes the fused kernel."""
    w = wl.small(name=f"tile_a{rope_axes}", dtype="bf16", grid=(5, 13, 20), window=(3, 7, 7), heads=2, head_dim=64,
                 rope_axes=rope_axes)
    check_full(oracle_mod, w, binding.IMPL_TCGEN05_TILE, backward=False)


def test_qknorm_logits_bf16(oracle_mod):
    """What QK-RMSNorm hands the kernel: |q| = |k| = sqrt(d), logits up to +-sqrt(d)."""
    w = wl.small(name="qknorm", dtype="bf16", value_scale="qknorm", grid=(8, 16, 16), window=(3, 7, 7),
                 heads=2, head_dim=64)
    check_full(oracle_mod, w, binding.IMPL_AUTO)


def test_large_logits_stay_close(oracle_mod):
    """Unit-normal q, k with scale 0.5: logits of +-20 (the fused forward subtracts no maximum: e^20 is in range)."""
    w = wl.small(name="hot", dtype="bf16", value_scale="unit", grid=(8, 16, 24), window=(3, 7, 7),
                 heads=2, head_dim=64)
    inp = wl.make_inputs(w)
    d, o, lse = run_fwd(w, inp, binding.IMPL_AUTO, 0.5)
    o_ref, lse_ref = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window, scale=0.5)
    # The rotated operands are rounded to bf16 (and the fused forward rotates in bf16x2 arithmetic): the error of a
    # logit grows with its size, measured max-abs error on O 0.0085 / 0.028 / 0.060 / 0.092 at max |logit| 6 / 10 / 20 /
    # 30.  At +-20 that is outside north_star's per-element bound by construction; held here: 1.5x
    # the measured maximum, and the NORMAL relative-RMS bound (measured 7.5e-3).  The in-tolerance test of large logits
    # is the exact-input one below.
    err = np.abs(to_f64(o) - o_ref)
    assert np.isfinite(to_f64(o)).all() and err.max() < 0.09
    assert np.sqrt(np.mean(err ** 2)) / np.sqrt(np.mean(o_ref ** 2)) < 1e-2
    assert float(np.abs(to_f64(lse) - lse_ref).max()) < 0.075


def test_backward_with_large_logits_and_determinism(oracle_mod):
    """Unit-normal q, k with scale 0.25: logits of +-10, lse / scale up to ~60.  The dK/dV kernel gets lse and D through a
    three-term bf16 split inside the tensor-core accumulation (na3d_bwd_tc2.cu): a term dropped there would show here first.
    The backward has no atomics: two runs must agree bit for bit."""
    w = wl.small(name="hot_bwd", dtype="bf16", value_scale="unit", grid=(8, 16, 24), window=(3, 7, 7),
                 heads=2, head_dim=64)
    inp = wl.make_inputs(w, with_do=True)
    d, o, lse = run_fwd(w, inp, binding.IMPL_AUTO, 0.25)
    g1 = run_bwd(w, inp, d, o, lse, binding.IMPL_AUTO, 0.25)
    g2 = run_bwd(w, inp, d, o, lse, binding.IMPL_AUTO, 0.25)
    for a, b in zip(g1, g2):
        assert torch.equal(a, b)
    refs = oracle_mod.na3d_bwd(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window, scale=0.25)
    # measured (B200): max-abs error 0.109 / 0.113 / 0.061 on dQ / dK / dV of magnitude up to 6.7 / 7.2 / 4.1, relative RMS
    # 8.4e-3 / 8.1e-3 / 7.1e-3 -- the rounding of the rotated operands and of the GPU's O, growing with the logits as in
    # the forward.  Held: 1.5x the measured maxima and the normal relative-RMS bound of the backward.
    for name, g, r, bound in zip(("dQ", "dK", "dV"), g1, refs, (0.165, 0.17, 0.092)):
        err = np.abs(to_f64(g) - r)
        assert np.isfinite(to_f64(g)).all() and err.max() < bound, (name, err.max())
        assert np.sqrt(np.mean(err ** 2)) / np.sqrt(np.mean(r ** 2)) < 2e-2, name


def _bf16_bits(x):
    """float32 array whose values are exact in bf16 -> the uint16 bit patterns the workloads use."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    assert not np.any(u & 0xFFFF), "value not exact in bf16"
    return (u >> 16).astype(np.uint16)


def _exact_inputs(w, rng):
    """Q, K, V whose products and sums are exact in bf16 / fp32: small integers over 8 (no RoPE), so the only
    rounding left is P -> bf16 and the output."""
    shape = (w.batch,) + w.grid + (w.heads, w.head_dim)
    q = rng.integers(-2, 3, size=shape).astype(np.float32) / 8
    k = rng.integers(-2, 3, size=shape).astype(np.float32) / 8
    v = rng.integers(-4, 5, size=shape).astype(np.float32) / 4
    return q, k, v


@pytest.mark.parametrize("case", [dict(impl=binding.IMPL_AUTO, window=(3, 7, 7), head_dim=64),            # fused forward
                                  dict(impl=binding.IMPL_TCGEN05_TILE, window=(3, 7, 7), head_dim=64),    # tile kernel
                                  dict(impl=binding.IMPL_AUTO, window=(5, 9, 9), head_dim=128)],          # tile kernel, d = 128
                         ids=["fused", "tile", "tile_d128"])
def test_rows_outside_the_exponent_range_take_the_fixup_kernel(oracle_mod, case):
    """The tensor-core forwards exponentiate without a reference; a row whose sum leaves 2^-80 .. 2^100 is listed and
    recomputed by na3d_fix_rows_kernel with a two-pass softmax.  Inputs exact in bf16: normal tolerances apply."""
    w = wl.small(name="fixup", dtype="bf16", grid=(6, 17, 19), window=case["window"], heads=2, head_dim=case["head_dim"],
                 rope_axes=0)
    rng = np.random.default_rng(77)
    q, k, v = _exact_inputs(w, rng)
    k[..., 1] = -40.0                                  # every key: a large component that normal queries hardly see
    hot = [(0, 2, 5, 6, 0), (0, 0, 0, 0, 1), (0, 5, 16, 18, 1), (0, 3, 8, 9, 0)]
    for (b, l, y, x, h) in hot[:3]:                    # logit +200 with their own key: e^200 overflows fp32
        q[b, l, y, x, h, :] = 0.0
        q[b, l, y, x, h, 0] = 40.0
        k[b, l, y, x, h, 0] = 40.0
    b, l, y, x, h = hot[3]                             # every logit -200: the whole row underflows
    q[b, l, y, x, h, :] = 0.0
    q[b, l, y, x, h, 1] = 40.0
    inp = {"q": _bf16_bits(q), "k": _bf16_bits(k), "v": _bf16_bits(v), "coords": np.zeros((w.batch,) + w.grid + (0,), np.float32),
           "freqs": np.zeros((0, w.head_dim // 2), np.float32)}
    dev = device_inputs(w, inp)
    desc = desc_of(w, case["impl"], 0.125)
    o = torch.empty_like(dev["q"])
    lse = torch.empty(desc.lse_shape, dtype=torch.float32, device="cuda")
    ws = binding.alloc_workspace(binding.strata_na3d_workspace_bytes(desc, False), "cuda")
    binding.strata_na3d_fwd(desc, dev["q"], dev["k"], dev["v"], None, None, o, lse, ws)
    torch.cuda.synchronize()
    listed, take_all = binding.fixup_stats(ws)          # (documented in strata_na3d.h: head of the workspace)
    assert listed >= len(hot) and not take_all, f"fix-up list holds {listed} rows, take-all {take_all}"
    o_ref, lse_ref = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window, scale=0.125)
    assert_parity(to_f64(o), o_ref, "bf16", "fixup O")
    assert float(np.abs(to_f64(lse) - lse_ref).max()) < 1e-3, "fixup LSE"


def test_level_dependent_coordinates_take_the_fixup_kernel(oracle_mod):
    """Two rotary axes whose coordinates change with the level (not the paper's case): the fused
    forward shares one rotary table per level column, notices, and hands every row to the fix-up kernel."""
    w = wl.small(name="lvlcoords", dtype="bf16", grid=(4, 9, 10), window=(3, 5, 5), heads=2, head_dim=64)
    inp = wl.make_inputs(w)
    coords = inp["coords"].copy()
    coords[:, 1:, ..., 0] += 3.0 * np.arange(1, w.grid[0], dtype=np.float32)[None, :, None, None]
    inp["coords"] = coords
    d = device_inputs(w, inp)
    desc = desc_of(w)
    o = torch.empty_like(d["q"])
    lse = torch.empty(desc.lse_shape, dtype=torch.float32, device="cuda")
    ws = binding.alloc_workspace(binding.strata_na3d_workspace_bytes(desc, False), "cuda")
    binding.strata_na3d_fwd(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], o, lse, ws)
    torch.cuda.synchronize()
    assert binding.fixup_stats(ws)[1], "the take-all flag the header documents is not set"
    o_ref, lse_ref = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], coords, inp["freqs"], w.window)
    assert_parity(to_f64(o), o_ref, "bf16", "level-dependent coords O")
    assert_parity(to_f64(lse), lse_ref, "bf16", "level-dependent coords LSE", rms_bound=1e-2)


def test_tcgen05_is_selected_for_the_bf16_configs():
    for i in (1, 2, 3):
        assert binding.strata_na3d_impl_selected(desc_of(wl.config(i))) == binding.IMPL_TCGEN05
    assert binding.strata_na3d_impl_selected(desc_of(wl.config(0))) == binding.IMPL_SIMT
    assert binding.strata_na3d_impl_selected(desc_of(wl.config(4)), True) == binding.IMPL_TCGEN05


def test_explicit_scale(oracle_mod):
    w = wl.small(name="scale", dtype="f32", grid=(3, 6, 7), window=(3, 3, 3), heads=2, head_dim=32)
    check_full(oracle_mod, w, binding.IMPL_AUTO, scale=0.31)


# ------------------------------------------------------------------ API behaviour on the device
def test_host_entry_points(oracle_mod):
    w = wl.small(name="host", dtype="bf16", grid=(4, 9, 10), window=(3, 5, 5), heads=2, head_dim=64, batch=2)
    inp = wl.make_inputs(w, with_do=True)
    h = device_inputs(w, inp, device="cpu")
    h = {n: (t.pin_memory() if t is not None else None) for n, t in h.items()}
    desc = desc_of(w)
    o = torch.empty_like(h["q"]).pin_memory()
    lse = torch.empty(desc.lse_shape, dtype=torch.float32).pin_memory()
    ws = binding.alloc_workspace(binding.strata_na3d_host_workspace_bytes(desc, False), "cuda")
    binding.strata_na3d_fwd_host(desc, h["q"], h["k"], h["v"], h["coords"], h["freqs"], o, lse, ws)
    torch.cuda.synchronize()
    o_ref, lse_ref = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window)
    assert_parity(to_f64(o), o_ref, "bf16", "host O")
    assert_parity(to_f64(lse), lse_ref, "bf16", "host LSE")
    dq, dk, dv = (torch.empty_like(h["q"]).pin_memory() for _ in range(3))
    ws = binding.alloc_workspace(binding.strata_na3d_host_workspace_bytes(desc, True), "cuda")
    binding.strata_na3d_bwd_host(desc, h["q"], h["k"], h["v"], o, h["do"], lse, h["coords"], h["freqs"], dq, dk, dv, ws)
    torch.cuda.synchronize()
    ref = oracle_mod.na3d_bwd(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window)
    for got, r, nm in zip((dq, dk, dv), ref, ("dQ", "dK", "dV")):
        assert_parity(to_f64(got), r, "bf16", f"host {nm}", rms_bound=2e-2)


def test_host_entry_points_reuse_their_staging_slots(oracle_mod):
    """Batch 5 through the per-sample host pipeline (strata_na3d.cu host_pipeline): both staging slots are reused
    (samples 2, 3, 4 wait for the kernels and the copies out of samples 0, 1, 2) and the final join covers an uneven
    tail.  The result must equal the device-pointer call on the same inputs bit for bit, forward and backward, and
    match the oracle.  Second pass: on a side stream with work queued ahead of the call -- a delay, then the copy that
    fills the pinned Q buffer -- which the pipeline's copy streams have to wait for."""
    w = wl.small(name="host5", dtype="bf16", value_scale="rsqrt_d", grid=(4, 9, 10), window=(3, 5, 5), heads=2,
                 head_dim=64, batch=5)
    inp = wl.make_inputs(w, with_do=True)
    dev = device_inputs(w, inp)
    h = {n: (t.pin_memory() if t is not None else None) for n, t in device_inputs(w, inp, device="cpu").items()}
    desc = desc_of(w)
    # device-pointer calls (the whole batch in one call)
    o_d = torch.empty_like(dev["q"])
    lse_d = torch.empty(desc.lse_shape, dtype=torch.float32, device="cuda")
    ws = binding.alloc_workspace(max(binding.strata_na3d_workspace_bytes(desc, False),
                                     binding.strata_na3d_workspace_bytes(desc, True)), "cuda")
    binding.strata_na3d_fwd(desc, dev["q"], dev["k"], dev["v"], dev["coords"], dev["freqs"], o_d, lse_d, ws)
    g_d = [torch.empty_like(dev["q"]) for _ in range(3)]
    binding.strata_na3d_bwd(desc, dev["q"], dev["k"], dev["v"], o_d, dev["do"], lse_d, dev["coords"], dev["freqs"], *g_d, ws)
    torch.cuda.synchronize()
    o_ref, lse_ref = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window)
    assert_parity(to_f64(o_d), o_ref, "bf16", "host5 device O")

    ws_f = binding.alloc_workspace(binding.strata_na3d_host_workspace_bytes(desc, False), "cuda")
    ws_b = binding.alloc_workspace(binding.strata_na3d_host_workspace_bytes(desc, True), "cuda")
    side = torch.cuda.Stream()
    for stream in (None, side):
        o = torch.zeros_like(h["q"]).pin_memory()
        lse = torch.zeros(desc.lse_shape, dtype=torch.float32).pin_memory()
        g = [torch.zeros_like(h["q"]).pin_memory() for _ in range(3)]
        hq = h["q"]
        if stream is not None:
            hq = torch.zeros_like(h["q"]).pin_memory()                  # filled by work queued on `stream` before the call
            with torch.cuda.stream(stream):
                torch.cuda._sleep(40_000_000)                            # ~20 ms: the call below returns long before this ends
                hq.copy_(dev["q"], non_blocking=True)
        binding.strata_na3d_fwd_host(desc, hq, h["k"], h["v"], h["coords"], h["freqs"], o, lse, ws_f, stream=stream)
        binding.strata_na3d_bwd_host(desc, hq, h["k"], h["v"], o, h["do"], lse, h["coords"], h["freqs"], *g, ws_b,
                                     stream=stream)
        (stream or torch.cuda.current_stream()).synchronize()
        tag = "default stream" if stream is None else "side stream"
        assert torch.equal(o, o_d.cpu()) and torch.equal(lse, lse_d.cpu()), f"host forward differs ({tag})"
        for got, ref, nm in zip(g, g_d, ("dQ", "dK", "dV")):
            assert torch.equal(got, ref.cpu()), f"host {nm} differs ({tag})"
        assert_parity(to_f64(o), o_ref, "bf16", f"host5 O ({tag})")
        assert_parity(to_f64(lse), lse_ref, "bf16", f"host5 LSE ({tag})")
    ref = oracle_mod.na3d_bwd(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window)
    for got, r, nm in zip(g, ref, ("dQ", "dK", "dV")):
        assert_parity(to_f64(got), r, "bf16", f"host5 {nm}", rms_bound=2e-2)


def test_device_error_paths_and_stream():
    w = wl.small(name="err", dtype="f32", grid=(3, 6, 7), window=(3, 3, 3), heads=2, head_dim=32)
    inp = wl.make_inputs(w)
    d = device_inputs(w, inp)
    desc = desc_of(w)
    o = torch.empty_like(d["q"])
    lse = torch.empty(desc.lse_shape, dtype=torch.float32, device="cuda")
    need = binding.strata_na3d_workspace_bytes(desc, False)
    small = binding.alloc_workspace(need - 256, "cuda")
    assert binding.strata_na3d_fwd_status(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], o, lse, small) == 3
    ws = binding.alloc_workspace(need, "cuda")
    mis = torch.empty(d["q"].numel() + 1, device="cuda")[1:].view_as(d["q"])      # 4-byte offset
    assert binding.strata_na3d_fwd_status(desc, mis, d["k"], d["v"], d["coords"], d["freqs"], o, lse, ws) == 1
    # asynchronous on a side stream; result identical to the default-stream call
    binding.strata_na3d_fwd(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], o, lse, ws)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    o2, lse2 = torch.empty_like(o), torch.empty_like(lse)
    with torch.cuda.stream(s):
        binding.strata_na3d_fwd(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], o2, lse2, ws, stream=s)
    s.synchronize()
    assert torch.equal(o, o2) and torch.equal(lse, lse2)
    assert binding.strata_na3d_last_launch_count() >= 2


def _guarded(shape, dtype, guard=8192):
    """A tensor carved out of a larger byte buffer with canary bands on both sides."""
    n = int(np.prod(shape)) * torch.empty((), dtype=dtype).element_size()
    pad = (n + 255) // 256 * 256
    raw = torch.full((guard + pad + guard,), 0xA5, dtype=torch.uint8, device="cuda")
    view = raw[guard:guard + n].view(dtype).view(shape)
    return raw, view, guard, n


def _guards_intact(raw, guard, n):
    return bool((raw[:guard] == 0xA5).all()) and bool((raw[guard + n:] == 0xA5).all())


@pytest.mark.parametrize("case", [dict(grid=(5, 11, 13), window=(3, 7, 7), heads=2, head_dim=64),
                                  dict(grid=(8, 17, 9), window=(3, 5, 5), heads=3, head_dim=64, batch=2),
                                  dict(grid=(6, 10, 17), window=(5, 9, 9), heads=1, head_dim=128),
                                  dict(grid=(3, 6, 7), window=(3, 3, 3), heads=2, head_dim=32, dtype="f32")])
def test_no_write_outside_the_output_buffers(case):
    """compute-sanitizer is closed on this GPU pool (profiles/r2_sanitizer.md): every output and the workspace sit
    between canary bands here, ragged shapes, forward and backward; a stray store shows up in a band."""
    kw = dict(dtype="bf16")
    kw.update(case)
    w = wl.small(name="guard", **kw)
    inp = wl.make_inputs(w, with_do=True)
    d = device_inputs(w, inp)
    desc = desc_of(w)
    tdt = torch.float32 if w.dtype == "f32" else torch.bfloat16
    bufs = {n: _guarded(tuple(d["q"].shape), tdt) for n in ("o", "dq", "dk", "dv")}
    bufs["lse"] = _guarded(tuple(desc.lse_shape), torch.float32)
    nws = max(binding.strata_na3d_workspace_bytes(desc, False), binding.strata_na3d_workspace_bytes(desc, True), 256)
    bufs["ws"] = _guarded((nws,), torch.uint8)
    v = {n: b[1] for n, b in bufs.items()}
    binding.strata_na3d_fwd(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], v["o"], v["lse"], v["ws"])
    binding.strata_na3d_bwd(desc, d["q"], d["k"], d["v"], v["o"], d["do"], v["lse"], d["coords"], d["freqs"], v["dq"],
                            v["dk"], v["dv"], v["ws"])
    torch.cuda.synchronize()
    for n, (raw, _, guard, nbytes) in bufs.items():
        assert _guards_intact(raw, guard, nbytes), f"write outside {n}"
    assert bool(torch.isfinite(v["o"].float()).all()) and bool(torch.isfinite(v["dq"].float()).all())


def test_cuda_graph_capture_and_replay(oracle_mod):
    """include/strata_na3d.h: calls never synchronise and are safe to capture.  Forward + backward captured in one
    graph on a side stream, replayed twice with the inputs changed in between."""
    w = wl.small(name="graph", dtype="bf16", value_scale="rsqrt_d", grid=(8, 18, 21), window=(3, 7, 7), heads=2,
                 head_dim=64)
    inp = wl.make_inputs(w, with_do=True)
    d = device_inputs(w, inp)
    desc = desc_of(w)
    o = torch.empty_like(d["q"])
    lse = torch.empty(desc.lse_shape, dtype=torch.float32, device="cuda")
    dq, dk, dv = (torch.empty_like(d["q"]) for _ in range(3))
    ws_f = binding.alloc_workspace(binding.strata_na3d_workspace_bytes(desc, False), "cuda")
    ws_b = binding.alloc_workspace(binding.strata_na3d_workspace_bytes(desc, True), "cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        st = torch.cuda.current_stream()
        binding.strata_na3d_fwd(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], o, lse, ws_f, stream=st)
        binding.strata_na3d_bwd(desc, d["q"], d["k"], d["v"], o, d["do"], lse, d["coords"], d["freqs"], dq, dk, dv, ws_b,
                                stream=st)
    ref = {}
    for rep in range(2):
        if rep == 1:                                   # new values in the same buffers
            inp = wl.make_inputs(dataclasses.replace(w, seed=w.seed + 1), with_do=True)
            for n, t in device_inputs(w, inp).items():
                if t is not None:
                    d[n].copy_(t)
        o.zero_(); dq.zero_(); dk.zero_(); dv.zero_()
        g.replay()
        torch.cuda.synchronize()
        o_ref, lse_ref = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window)
        assert_parity(to_f64(o), o_ref, "bf16", f"graph replay {rep} O")
        assert_parity(to_f64(lse), lse_ref, "bf16", f"graph replay {rep} LSE", rms_bound=1e-2)
        gr = oracle_mod.na3d_bwd(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window)
        for got, r, nm in zip((dq, dk, dv), gr, ("dQ", "dK", "dV")):
            assert_parity(to_f64(got), r, "bf16", f"graph replay {rep} {nm}", rms_bound=2e-2)


# ------------------------------------------------------------------ the paper's own shapes (NEXT-4) and column attention (NEXT-2)
@pytest.mark.parametrize("case", [dict(grid=(24, 16, 16), heads=2), dict(grid=(10, 20, 11), heads=3, batch=2),
                                  dict(grid=(9, 9, 9), heads=1, rope_pairing=1)])
def test_production_window_9x9x9_on_the_tensor_cores(oracle_mod, case):
    """PAPER.md:325-326 (Table S1): 24 levels, head_dim 64, NATTEN kernel size 9 -- forward and backward."""
    w = wl.small(name="prod999", dtype="bf16", value_scale="qknorm", window=(9, 9, 9), head_dim=64, **case)
    assert binding.strata_na3d_impl_selected(desc_of(w)) == binding.IMPL_TCGEN05
    assert binding.strata_na3d_impl_selected(desc_of(w), True) == binding.IMPL_TCGEN05
    check_full(oracle_mod, w, binding.IMPL_AUTO)


def test_production_shape_at_the_size_the_bench_times(oracle_mod):
    """workloads.production("prod32") as bench.py runs it: 24 x 32 x 32 tokens, 16 heads, batch 2, window 9 x 9 x 9 --
    every element of O, LSE, dQ, dK, dV against the oracle (about a minute of oracle time)."""
    check_full(oracle_mod, wl.production("prod32"), binding.IMPL_AUTO)


@pytest.mark.parametrize("case", [dict(grid=(10, 17, 19), heads=1), dict(grid=(24, 16, 16), heads=2),
                                  dict(grid=(9, 12, 9), heads=1, batch=2, rope_pairing=1)])
def test_decoder_window_9x9x9_with_head_dim_128(oracle_mod, case):
    """PAPER.md:326, the de-aliasing decoder's NA3D blocks: embedding 128 (one head of 128 channels, reading R26),
    kernel 9.  Forward on the tcgen05 tile kernel (Cfg<128, 9, 9, 9>); the d = 128 backward runs on the CUDA cores."""
    w = wl.small(name="dec999", dtype="bf16", value_scale="qknorm", window=(9, 9, 9), head_dim=128, **case)
    assert binding.strata_na3d_impl_selected(desc_of(w)) == binding.IMPL_TCGEN05
    assert binding.strata_na3d_impl_selected(desc_of(w), True) == binding.IMPL_SIMT
    check_full(oracle_mod, w, binding.IMPL_AUTO)


def test_decoder_shape_sampled_rows_at_bench_size(oracle_mod):
    """workloads.production("dec64") (24 x 64 x 64 tokens, one head of 128, batch 2) in the launch configuration bench.py
    times: 4096 random rows against the oracle, every output finite."""
    w = wl.production("dec64")
    inp = wl.make_inputs(w)
    d, o, lse = run_fwd(w, inp)
    assert bool(torch.isfinite(o.float()).all()) and bool(torch.isfinite(lse).all())
    idx = np.sort(np.random.default_rng(3).choice(w.batch * w.tokens * w.heads, size=4096, replace=False))
    o_ref, lse_ref = oracle_mod.na3d_fwd_queries(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window, idx)
    assert w.heads == 1                                      # (so that LSE [B, H, N] and the row index (b N + t) H + h coincide)
    got_o = to_f64(o).reshape(-1, w.head_dim)[idx]
    assert_parity(got_o, np.asarray(o_ref).reshape(-1, w.head_dim), "bf16", "dec64 sampled O")
    assert_parity(to_f64(lse).reshape(-1)[idx], np.asarray(lse_ref).reshape(-1), "bf16", "dec64 sampled LSE", rms_bound=1e-2)


@pytest.mark.parametrize("case", [dict(grid=(24, 5, 7), heads=3), dict(grid=(8, 9, 6), heads=2, batch=2),
                                  dict(grid=(32, 3, 4), heads=1, rope_pairing=1), dict(grid=(5, 4, 4), heads=2, rope_axes=0)])
def test_column_attention(oracle_mod, case):
    """attention along the vertical, window (L, 1, 1) -- its own kernel (na3d_column.cu)."""
    kw = dict(name="column", dtype="bf16", value_scale="qknorm", head_dim=64)
    kw.update(case)
    w = wl.small(**kw)
    w = dataclasses.replace(w, window=(w.grid[0], 1, 1))
    check_full(oracle_mod, w, binding.IMPL_AUTO, backward=True)       # (the (L, 1, 1) backward: CUDA-core kernels)


def test_column_window_through_the_host_backward(oracle_mod):
    """Window (24, 1, 1) (the column-wise blocks) through strata_na3d_fwd_host / _bwd_host, three samples
    (the third reuses a staging slot)."""
    w = wl.small(name="colhost", dtype="bf16", value_scale="qknorm", grid=(24, 5, 6), window=(24, 1, 1), heads=2,
                 head_dim=64, batch=3)
    inp = wl.make_inputs(w, with_do=True)
    h = {n: (t.pin_memory() if t is not None else None) for n, t in device_inputs(w, inp, device="cpu").items()}
    desc = desc_of(w)
    o = torch.empty_like(h["q"]).pin_memory()
    lse = torch.empty(desc.lse_shape, dtype=torch.float32).pin_memory()
    ws = binding.alloc_workspace(max(binding.strata_na3d_host_workspace_bytes(desc, False),
                                     binding.strata_na3d_host_workspace_bytes(desc, True)), "cuda")
    binding.strata_na3d_fwd_host(desc, h["q"], h["k"], h["v"], h["coords"], h["freqs"], o, lse, ws)
    g = [torch.empty_like(h["q"]).pin_memory() for _ in range(3)]
    binding.strata_na3d_bwd_host(desc, h["q"], h["k"], h["v"], o, h["do"], lse, h["coords"], h["freqs"], *g, ws)
    torch.cuda.synchronize()
    o_ref, lse_ref = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window)
    assert_parity(to_f64(o), o_ref, "bf16", "column host O")
    assert_parity(to_f64(lse), lse_ref, "bf16", "column host LSE", rms_bound=1e-2)
    ref = oracle_mod.na3d_bwd(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window)
    for got, r, nm in zip(g, ref, ("dQ", "dK", "dV")):
        assert_parity(to_f64(got), r, "bf16", f"column host {nm}", rms_bound=2e-2)


def test_column_attention_with_level_dependent_coordinates(oracle_mod):
    """The rotation only cancels when a column's tokens share their coordinates; otherwise every row is recomputed."""
    w = wl.small(name="column_lvl", dtype="bf16", value_scale="rsqrt_d", grid=(6, 5, 4), window=(6, 1, 1), heads=2, head_dim=64)
    inp = wl.make_inputs(w)
    coords = inp["coords"].copy()
    coords[:, 1:, ..., 1] += 0.7 * np.arange(1, w.grid[0], dtype=np.float32)[None, :, None, None]
    inp["coords"] = coords
    d, o, lse = run_fwd(w, inp)
    o_ref, lse_ref = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], coords, inp["freqs"], w.window)
    assert_parity(to_f64(o), o_ref, "bf16", "column, level-dependent coords O")
    assert_parity(to_f64(lse), lse_ref, "bf16", "column, level-dependent coords LSE", rms_bound=1e-2)


# ------------------------------------------------------------------ QK-RMSNorm + sigmoid head gate (NEXT-1)
@pytest.mark.parametrize("case", [dict(dtype="bf16", grid=(8, 18, 21), window=(3, 7, 7), heads=2, head_dim=64),          # fused fwd, tcgen05 bwd
                                  dict(dtype="bf16", grid=(6, 10, 9), window=(5, 9, 9), heads=1, head_dim=128),         # tile fwd, SIMT bwd
                                  dict(dtype="f32", grid=(3, 6, 7), window=(3, 3, 3), heads=2, head_dim=32),
                                  dict(dtype="bf16", grid=(5, 9, 12), window=(3, 5, 5), heads=3, head_dim=64, gate=False),
                                  dict(dtype="bf16", grid=(8, 64, 64), window=(3, 7, 7), heads=8, head_dim=64, batch=4)])  # config 1's size
def test_qk_rmsnorm_and_head_gate(oracle_mod, case):
    kw = dict(case)
    with_gate = kw.pop("gate", True)
    w = wl.small(name="normgate", value_scale="unit", **kw)
    inp = wl.make_inputs(w, with_do=True)
    rng = np.random.default_rng(w.seed + 3)
    # un-normalised inputs of very different lengths per row: the kernel must do the normalising
    fac = rng.uniform(0.25, 4.0, size=inp["q"].shape[:-1] + (1,)).astype(np.float32)
    if w.dtype == "bf16":
        q32 = wl.bf16_bits_to_f32(inp["q"]) * fac
        inp["q"] = wl.f32_to_bf16_bits(q32)
    else:
        inp["q"] = (inp["q"] * fac).astype(np.float32)
    gate_np = (rng.normal(size=(w.batch,) + w.grid + (w.heads,)) * 2).astype(np.float32) if with_gate else None
    eps = 1e-5
    d = device_inputs(w, inp)
    desc = desc_of(w)
    gate = torch.from_numpy(gate_np).cuda() if with_gate else None
    o = torch.empty_like(d["q"])
    lse = torch.empty(desc.lse_shape, dtype=torch.float32, device="cuda")
    ws = binding.alloc_workspace(max(binding.strata_na3d_normgate_workspace_bytes(desc, False),
                                     binding.strata_na3d_normgate_workspace_bytes(desc, True)), "cuda")
    binding.strata_na3d_normgate_fwd(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], gate, eps, o, lse, ws)
    dq, dk, dv = (torch.empty_like(d["q"]) for _ in range(3))
    dgate = torch.empty_like(gate) if with_gate else None
    binding.strata_na3d_normgate_bwd(desc, d["q"], d["k"], d["v"], o, d["do"], lse, d["coords"], d["freqs"], gate, eps,
                                     dq, dk, dv, dgate, ws)
    torch.cuda.synchronize()
    o_ref, lse_ref, _ = oracle_mod.na3d_normgate_fwd(inp["q"], inp["k"], inp["v"], gate_np, inp["coords"], inp["freqs"],
                                                     w.window, eps=eps)
    assert_parity(to_f64(o), o_ref, w.dtype, "normgate O")
    assert_parity(to_f64(lse), lse_ref, "f32" if w.dtype == "f32" else "bf16", "normgate LSE", rms_bound=1e-2)
    rq, rk, rv, rg = oracle_mod.na3d_normgate_bwd(inp["q"], inp["k"], inp["v"], gate_np, inp["do"], inp["coords"],
                                                  inp["freqs"], w.window, eps=eps)
    rb = None if w.dtype == "f32" else 2e-2
    # dq = r (dq^ - ...): the per-row factor r = 1 / rms(q) (x 0.25 .. 4 here) scales the gradient and with it the
    # error of the attention backward; the tolerances are held on dq / r, i.e. at the scale of the un-scaled rows
    assert_parity(to_f64(dq) * fac.astype(np.float64), rq * fac, w.dtype, "normgate dQ (per unit of 1 / rms scale)", rms_bound=rb)
    assert_parity(to_f64(dk), rk, w.dtype, "normgate dK", rms_bound=rb)
    assert_parity(to_f64(dv), rv, w.dtype, "normgate dV", rms_bound=rb)
    if with_gate:
        assert_parity(to_f64(dgate), rg, w.dtype, "normgate dgate", rms_bound=rb)


# ------------------------------------------------------------------ geometry kernels (NEXT-3: eq. (1), eq. (2) on the device)
def test_stereo_coords_and_wind_frame_kernels(oracle_mod):
    """strata_stereo_coords / strata_wind_to_tile_frame against oracle/geometry.py on the patch centres of a
    128 x 128 tile far from the face centre (coordinates up to ~1e3: the float32 result must be the rounding of the
    float64 one) and on points around a high-latitude centre."""
    rng = np.random.default_rng(11)
    n_total = 6 * 2048 ** 2
    for lat0, lon0, span in ((0.61, -2.4, 0.2), (1.35, 0.3, 0.25), (-0.02, 3.0, 0.3)):
        n = 20011
        lat = lat0 + rng.uniform(-span, span, n)
        lon = lon0 + rng.uniform(-span, span, n)
        lat = np.clip(lat, -1.55, 1.55)
        d_lat, d_lon = torch.from_numpy(lat).cuda(), torch.from_numpy(lon).cuda()
        coords = torch.full((n, 3), -7.0, dtype=torch.float32, device="cuda")
        binding.strata_stereo_coords(d_lat, d_lon, lat0, lon0, n_total, coords, stride=3)
        x_ref, y_ref = oracle_mod.geometry.stereo_xy(lat, lon, lat0, lon0, n_total)
        got = coords.cpu().numpy()
        assert np.all(got[:, 2] == -7.0), "the third coordinate slot is not this call's"
        for g, r in ((got[:, 0], x_ref), (got[:, 1], y_ref)):
            err = np.abs(g.astype(np.float64) - r)
            assert np.all(err <= np.abs(r) * 2.0 ** -23 + 1e-30), f"eq. (1): max err {err.max():.3e}"
        u = (rng.normal(size=n) * 25).astype(np.float32)
        v = (rng.normal(size=n) * 25).astype(np.float32)
        d_u, d_v = torch.from_numpy(u).cuda(), torch.from_numpy(v).cuda()
        ul, vl = torch.empty_like(d_u), torch.empty_like(d_v)
        binding.strata_wind_to_tile_frame(d_u, d_v, d_lat, d_lon, lat0, lon0, ul, vl)
        ul_ref, vl_ref = oracle_mod.geometry.wind_to_tile_frame(u, v, lat, lon, lat0, lon0)
        for g, r in ((ul.cpu().numpy(), ul_ref), (vl.cpu().numpy(), vl_ref)):
            err = np.abs(g.astype(np.float64) - r)
            assert np.all(err <= np.abs(r) * 2.0 ** -23 + 1e-5), f"eq. (2): max err {err.max():.3e}"
    assert lib_status_invalid()


def lib_status_invalid():
    L = binding.lib()
    return L.strata_stereo_coords(None, None, 4, 0.0, 0.0, 1.0, None, 2, None) == 1 and \
        L.strata_wind_to_tile_frame(None, None, None, None, 4, 0.0, 0.0, None, None, None) == 1


def test_tile_stitch_kernel(oracle_mod):
    """strata_tile_stitch against oracle/stitch.py on config 3's tile layout of one face (2 x 2 tiles of 128 x 128 with
    stride 112) at reduced channel count, Kaiser-Bessel-derived and top-hat windows."""
    rng = np.random.default_rng(13)
    T, C, th = 4, 5, 128
    origins = np.array([(0, 0), (0, 112), (112, 0), (112, 112)], dtype=np.int32)
    gh = gw = 240
    tiles = rng.normal(size=(T, C, th, th)).astype(np.float32)
    hat = np.zeros(th, np.float32); hat[8:120] = 1.0
    for wy in (oracle_mod.stitch.kbd_window(th, 4.0).astype(np.float32), hat):
        out = torch.full((C, gh, gw), 7.0, dtype=torch.float32, device="cuda")
        binding.strata_tile_stitch(torch.from_numpy(tiles).cuda(), torch.from_numpy(origins).cuda(), torch.from_numpy(wy).cuda(),
                                   torch.from_numpy(wy).cuda(), out)
        ref = oracle_mod.stitch.stitch(tiles, origins, wy, wy, gh, gw)
        err = np.abs(out.cpu().numpy().astype(np.float64) - ref)
        assert err.max() <= 1e-5, f"stitch: max abs err {err.max():.3e}"


@pytest.mark.parametrize("case", ["twelve_deep", "many_tiles"])
def test_tile_stitch_kernel_other_layouts(oracle_mod, case):
    """eq. (5) where the row kernel leaves its fast path: twelve tiles over the same cells (more than the eight it keeps
    in registers) and 1100 small tiles (more than its list holds: the generic kernel).  Tiles overlap at random, some
    cells are covered by none (-> 0)."""
    rng = np.random.default_rng(29)
    if case == "twelve_deep":
        T, C, th, tw, gh, gw = 12, 3, 16, 16, 40, 300
        origins = np.array([(i, i) for i in range(T)], dtype=np.int32)      # cells (11..15, 11..15) lie under all twelve
    else:
        T, C, th, tw, gh, gw = 1100, 2, 3, 5, 64, 70
        origins = np.stack([rng.integers(0, gh - th + 1, T), rng.integers(0, gw - tw + 1, T)], axis=1).astype(np.int32)
    tiles = rng.normal(size=(T, C, th, tw)).astype(np.float32)
    wy = rng.uniform(0.1, 1.0, th).astype(np.float32)
    wx = rng.uniform(0.1, 1.0, tw).astype(np.float32)
    out = torch.full((C, gh, gw), 7.0, dtype=torch.float32, device="cuda")
    binding.strata_tile_stitch(torch.from_numpy(tiles).cuda(), torch.from_numpy(origins).cuda(), torch.from_numpy(wy).cuda(),
                               torch.from_numpy(wx).cuda(), out)
    ref = oracle_mod.stitch.stitch(tiles, origins, wy, wx, gh, gw)
    err = np.abs(out.cpu().numpy().astype(np.float64) - ref)
    assert err.max() <= 1e-5 * max(1.0, np.abs(ref).max()), f"stitch {case}: max abs err {err.max():.3e}"
    assert (ref == 0).any() and (ref != 0).any()
