"""strata_na3d_fwd_static: the forward for callers that cannot allocate device memory.

Who needs it: code that lives inside another program and owns no device memory -- a plug-in under a host whose pool
has claimed the whole GPU (cudaMalloc fails there, or takes what the host has promised to somebody else), a step in
a loop that may not be stalled by the device-wide synchronisation of cudaMalloc / cudaFree, a component that runs
after the host's "no more allocations" point.  They have inputs and outputs but no `workspace` to pass, so this one
call takes its scratch from a 1 MiB array inside the library (include/strata_na3d.h, csrc/static_scratch.cu).

What is held here: the call gives the same result as strata_na3d_fwd with a caller-allocated workspace, on two
calls in a row that share the array -- the second must not see what the first left behind -- and it refuses, with
its own status code, a problem that needs more scratch than the array holds.  The file name keeps it last in
pytest's collection order, so that a failure here cannot hide another test under `pytest -x`; it passes alone in a
fresh process (the first call then does the per-device address look-up) and after the rest of the suite."""
import ctypes

import numpy as np
import pytest
import torch

from paper_2606_31248_b200 import binding, build as lib_build, workloads as wl
from helpers import assert_parity, desc_of, device_inputs, to_f64


def _existing_path(desc, d):
    """strata_na3d_fwd with a workspace the caller allocated: the path the library had before."""
    o = torch.empty_like(d["q"])
    lse = torch.empty(desc.lse_shape, dtype=torch.float32, device="cuda")
    ws = binding.alloc_workspace(binding.strata_na3d_workspace_bytes(desc, False), "cuda")
    binding.strata_na3d_fwd(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], o, lse, ws)
    torch.cuda.synchronize()
    return o, lse


def _overflow_inputs(w):
    """Inputs (exact in bf16, no RoPE) with three rows whose softmax sum overflows fp32 and one that underflows: the
    tensor-core forward lists them in its scratch for the fix-up kernel, so the call leaves a non-empty list behind."""
    rng = np.random.default_rng(5)
    shape = (w.batch,) + w.grid + (w.heads, w.head_dim)
    q = rng.integers(-2, 3, size=shape).astype(np.float32) / 8
    k = rng.integers(-2, 3, size=shape).astype(np.float32) / 8
    v = rng.integers(-4, 5, size=shape).astype(np.float32) / 4
    k[..., 1] = -40.0
    for (l, y, x, h) in [(2, 5, 6, 0), (0, 0, 0, 1), (5, 16, 18, 1)]:
        q[0, l, y, x, h, :] = 0.0
        q[0, l, y, x, h, 0] = 40.0
        k[0, l, y, x, h, 0] = 40.0
    q[0, 3, 8, 9, 0, :] = 0.0
    q[0, 3, 8, 9, 0, 1] = 40.0
    bits = lambda a: (np.ascontiguousarray(a, dtype=np.float32).view(np.uint32) >> 16).astype(np.uint16)
    return {"q": bits(q), "k": bits(k), "v": bits(v)}


def _same(got, ref, dtype, what):
    """The tolerance of the parity tests (helpers.assert_parity), with the existing path as the reference; and since
    both calls run the same kernels on the same inputs, the results are also expected to agree bit for bit."""
    assert_parity(to_f64(got), to_f64(ref), dtype, what)
    assert torch.equal(got, ref), f"{what}: differs from the existing path"


@pytest.mark.gpu
def test_two_calls_in_a_row_on_the_fused_forward_match_the_existing_path():
    """bf16, head_dim 64, window 3x7x7: the fused tcgen05 forward, whose scratch is the list of rows for the fix-up
    kernel.  Call 1 fills that list (overflowing rows); call 2, straight after it on the same stream and on other
    inputs of another shape, must start from an empty list."""
    w1 = wl.small(name="noalloc_fix", dtype="bf16", grid=(6, 17, 19), window=(3, 7, 7), heads=2, head_dim=64, rope_axes=0)
    d1 = device_inputs(w1, _overflow_inputs(w1))
    desc1 = desc_of(w1, binding.IMPL_AUTO, 0.125)
    w2 = wl.small(name="noalloc_plain", dtype="bf16", value_scale="rsqrt_d", grid=(8, 24, 21), window=(3, 7, 7), heads=3,
                  head_dim=64, batch=2)
    d2 = device_inputs(w2, wl.make_inputs(w2))
    desc2 = desc_of(w2)
    assert binding.strata_na3d_workspace_bytes(desc2, False) <= binding.STATIC_SCRATCH_BYTES
    o1, lse1 = torch.empty_like(d1["q"]), torch.empty(desc1.lse_shape, dtype=torch.float32, device="cuda")
    o2, lse2 = torch.empty_like(d2["q"]), torch.empty(desc2.lse_shape, dtype=torch.float32, device="cuda")
    binding.strata_na3d_fwd_static(desc1, d1["q"], d1["k"], d1["v"], None, None, o1, lse1)
    binding.strata_na3d_fwd_static(desc2, d2["q"], d2["k"], d2["v"], d2["coords"], d2["freqs"], o2, lse2)
    torch.cuda.synchronize()
    ref_o1, ref_lse1 = _existing_path(desc1, d1)
    ref_o2, ref_lse2 = _existing_path(desc2, d2)
    _same(o1, ref_o1, "bf16", "call 1 O")
    _same(lse1, ref_lse1, "bf16", "call 1 LSE")
    _same(o2, ref_o2, "bf16", "call 2 O")
    _same(lse2, ref_lse2, "bf16", "call 2 LSE")
    # and once more in the other order: a plain call followed by one that needs the fix-up list
    o1.zero_(); lse1.zero_(); o2.zero_(); lse2.zero_()
    binding.strata_na3d_fwd_static(desc2, d2["q"], d2["k"], d2["v"], d2["coords"], d2["freqs"], o2, lse2)
    binding.strata_na3d_fwd_static(desc1, d1["q"], d1["k"], d1["v"], None, None, o1, lse1)
    torch.cuda.synchronize()
    _same(o2, ref_o2, "bf16", "call 3 O")
    _same(o1, ref_o1, "bf16", "call 4 O")
    _same(lse1, ref_lse1, "bf16", "call 4 LSE")


@pytest.mark.gpu
def test_two_calls_in_a_row_on_the_fp32_forward_match_the_existing_path():
    """BASELINE.json config 0 (fp32): the CUDA-core forward keeps rotated copies of Q and K in scratch (512 KiB of
    the array here).  Second call: a smaller problem with other values, over the first call's leftovers."""
    w1 = wl.config(0)
    d1 = device_inputs(w1, wl.make_inputs(w1))
    desc1 = desc_of(w1)
    w2 = wl.small(name="noalloc_f32", dtype="f32", grid=(3, 6, 7), window=(3, 3, 3), heads=2, head_dim=32)
    d2 = device_inputs(w2, wl.make_inputs(w2))
    desc2 = desc_of(w2)
    o1, lse1 = torch.empty_like(d1["q"]), torch.empty(desc1.lse_shape, dtype=torch.float32, device="cuda")
    o2, lse2 = torch.empty_like(d2["q"]), torch.empty(desc2.lse_shape, dtype=torch.float32, device="cuda")
    binding.strata_na3d_fwd_static(desc1, d1["q"], d1["k"], d1["v"], d1["coords"], d1["freqs"], o1, lse1)
    binding.strata_na3d_fwd_static(desc2, d2["q"], d2["k"], d2["v"], d2["coords"], d2["freqs"], o2, lse2)
    torch.cuda.synchronize()
    for got, ref, what in zip((o1, lse1), _existing_path(desc1, d1), ("config 0 O", "config 0 LSE")):
        _same(got, ref, "f32", what)
    for got, ref, what in zip((o2, lse2), _existing_path(desc2, d2), ("small fp32 O", "small fp32 LSE")):
        _same(got, ref, "f32", what)


@pytest.mark.gpu
def test_a_problem_beyond_the_array_is_refused_and_nothing_is_written():
    """fp32 scratch grows with the problem (two rotated copies): 2 x 4 x 8 x 32 x 32 x 4 x 32 floats is past 1 MiB."""
    w = wl.small(name="noalloc_big", dtype="f32", grid=(8, 32, 32), window=(3, 5, 5), heads=4, head_dim=32)
    desc = desc_of(w)
    assert binding.strata_na3d_workspace_bytes(desc, False) > binding.STATIC_SCRATCH_BYTES
    d = device_inputs(w, wl.make_inputs(w))
    o = torch.full_like(d["q"], 7.0)
    lse = torch.full(desc.lse_shape, 7.0, dtype=torch.float32, device="cuda")
    st = binding.strata_na3d_fwd_static_status(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], o, lse)
    torch.cuda.synchronize()
    assert st == binding.STRATA_ERR_STATIC_SCRATCH
    assert bool((o == 7.0).all()) and bool((lse == 7.0).all())
    with pytest.raises(binding.StrataError, match="static array"):
        binding.strata_na3d_fwd_static(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], o, lse)


def test_host_side_decisions_need_no_gpu():
    """Everything the call can decide from the descriptor and the pointers comes before its first CUDA call, so on a
    machine without a GPU the fake (never dereferenced) pointers below are enough."""
    lib_build.build()
    L = binding.lib()
    vp = ctypes.c_void_p
    ok = [vp(0x1000)] * 7
    call = lambda desc, ptrs: L.strata_na3d_fwd_static(ctypes.byref(desc.c()), *ptrs, None)
    f32 = lambda **kw: binding.NA3DDesc(**{**dict(batch=1, heads=2, head_dim=32, grid=(4, 16, 16), window=(3, 5, 5),
                                                  rope_axes=2, dtype=binding.DTYPE_F32), **kw})
    assert call(f32(batch=64), ok) == binding.STRATA_ERR_STATIC_SCRATCH          # 2 x 16 MiB of rotated copies
    assert L.strata_status_string(binding.STRATA_ERR_STATIC_SCRATCH).startswith(b"problem needs more scratch")
    assert call(f32(window=(3, 5, 17)), ok) == 1                                  # INVALID_ARG, named by the forward
    assert call(f32(head_dim=48), ok) == 2                                        # UNSUPPORTED
    assert call(f32(), [None] + ok[1:]) == 1                                      # null q
    # the fused bf16 forward needs the same 524 544 bytes at any size: config 3's descriptor fits
    assert binding.strata_na3d_workspace_bytes(desc_of(wl.config(3)), False) <= binding.STATIC_SCRATCH_BYTES
    assert binding.STATIC_SCRATCH_BYTES == 1 << 20
