"""CPU-side checks of the C-ABI library: it builds, loads, exports every declared symbol, and its
argument validation (which runs before any CUDA call) returns the documented status codes."""
import ctypes
import os
import re

import pytest

from paper_2606_31248_b200 import binding, build as lib_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    lib_build.build()
    return binding.lib()


def test_exports_every_declared_symbol(L):
    header = open(os.path.join(ROOT, "include", "strata_na3d.h")).read()
    declared = set(re.findall(r"\b(strata_[a-z0-9_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name
    assert binding.strata_version() >= 100
    assert L.strata_status_string(0) == b"ok"


def _desc(**kw):
    base = dict(batch=1, heads=2, head_dim=32, grid=(4, 16, 16), window=(3, 5, 5), rope_axes=2,
                dtype=binding.DTYPE_F32)
    base.update(kw)
    return binding.NA3DDesc(**base)


def test_workspace_query_and_validation(L):
    d = _desc()
    e = 1 * 1024 * 2 * 32
    assert binding.strata_na3d_workspace_bytes(d, False) >= 2 * e * 4
    assert binding.strata_na3d_workspace_bytes(d, True) >= 4 * e * 4
    assert binding.strata_na3d_host_workspace_bytes(d, False) > binding.strata_na3d_workspace_bytes(d, False)
    assert binding.strata_na3d_impl_selected(d) == binding.IMPL_SIMT            # fp32 -> CUDA-core kernels
    for bad in (_desc(window=(3, 5, 17)), _desc(window=(0, 5, 5)), _desc(head_dim=33), _desc(batch=0),
                _desc(dtype=7), _desc(rope_pairing=2), _desc(head_dim=48), _desc(rope_axes=4)):
        assert binding.strata_na3d_workspace_bytes(bad, False) == 0
        assert binding.strata_na3d_impl_selected(bad) == -1


def test_status_codes_without_touching_the_gpu(L):
    """Validation precedes every CUDA call, so fake (aligned, never dereferenced) pointers suffice."""
    d = _desc()
    vp = ctypes.c_void_p
    ok = [vp(0x1000)] * 7
    call = lambda desc, ptrs, ws, n: L.strata_na3d_fwd(ctypes.byref(desc.c()), *ptrs, ws, n, None)
    assert call(_desc(window=(3, 5, 17)), ok, vp(0x1000), 1 << 30) == 1          # INVALID_ARG
    assert call(_desc(head_dim=48), ok, vp(0x1000), 1 << 30) == 2                # UNSUPPORTED
    assert call(d, [None] + ok[1:], vp(0x1000), 1 << 30) == 1                    # null q
    assert call(d, [vp(0x1004)] + ok[1:], vp(0x1000), 1 << 30) == 1              # misaligned q
    assert call(d, ok, None, 0) == 3                                             # WORKSPACE
    assert call(d, ok, vp(0x1000), 16) == 3
    assert call(_desc(impl=binding.IMPL_TCGEN05), ok, vp(0x1000), 1 << 30) == 2  # fp32 has no tcgen05 path
    bw = lambda desc, ptrs, ws, n: L.strata_na3d_bwd(ctypes.byref(desc.c()), *ptrs, ws, n, None)
    ok11 = [vp(0x1000)] * 11
    assert bw(d, ok11, None, 0) == 3
    assert bw(d, ok11[:9] + [None, vp(0x1000)], vp(0x1000), 1 << 30) == 1


def test_normgate_calls_validate_everything_before_enqueuing(L):
    """strata_na3d_normgate_fwd / _bwd: a null or misaligned v, lse, o, dv ... is refused on the host, before the
    normalisation kernels go on the stream (no GPU here: reaching a launch would return CUDA, not INVALID_ARG)."""
    d = _desc()
    vp = ctypes.c_void_p
    a = vp(0x1000)
    fwd = lambda q, k, v, co, fr, g, o, lse: L.strata_na3d_normgate_fwd(ctypes.byref(d.c()), q, k, v, co, fr, g, 1e-6, o, lse,
                                                                       a, 1 << 30, None)
    assert fwd(a, a, None, a, a, None, a, a) == 1                        # null v
    assert fwd(a, a, a, a, a, None, a, None) == 1                        # null lse
    assert fwd(a, a, vp(0x1004), a, a, None, a, a) == 1                  # misaligned v
    assert fwd(a, a, a, None, a, None, a, a) == 1                        # rope_axes = 2 without coords
    assert fwd(a, a, a, a, a, None, vp(0x1008), a) == 1                  # misaligned o
    bwd = lambda v, lse, dv: L.strata_na3d_normgate_bwd(ctypes.byref(d.c()), a, a, v, a, a, lse, a, a, None, 1e-6, a, a, dv,
                                                        None, a, 1 << 30, None)
    assert bwd(None, a, a) == 1 and bwd(a, None, a) == 1 and bwd(a, a, None) == 1 and bwd(a, a, vp(0x1002)) == 1


def test_backward_family_respects_the_head_limit_of_the_statistics_kernel(L):
    """The tcgen05 backward's statistics pass stages 2 x 32 x (H + 1) floats in 48 KiB of shared memory: up to 191
    heads.  Past that AUTO must resolve to the CUDA-core backward (and an explicit TCGEN05 request is UNSUPPORTED)
    instead of failing at the launch."""
    bf = lambda heads, impl=binding.IMPL_AUTO: _desc(dtype=binding.DTYPE_BF16, head_dim=64, window=(3, 7, 7),
                                                     grid=(4, 16, 16), heads=heads, impl=impl)
    assert binding.strata_na3d_impl_selected(bf(191), True) == binding.IMPL_TCGEN05
    assert binding.strata_na3d_impl_selected(bf(192), True) == binding.IMPL_SIMT
    assert binding.strata_na3d_impl_selected(bf(192, binding.IMPL_TCGEN05), True) == -1
    assert binding.strata_na3d_workspace_bytes(bf(192), True) >= 4 * 1024 * 192 * 64 * 4      # fp32 rotated copies + grads
    assert binding.strata_na3d_impl_selected(bf(192), False) == binding.IMPL_TCGEN05           # the forward has no such limit


def test_window_and_inverse_window_against_brute_force(L):
    """A3 / B3 as the kernels compute them (csrc/common.cuh) against the definition by enumeration:
    "centre the window on the query, then shift it inward until it fits" (PAPER.md:79 + reading R1),
    and the inverse neighbourhood read off that enumeration (no formula)."""
    for line in open(os.path.join(ROOT, "tests", "golden", "window_starts.txt")):      # hand-derived fixture
        if line.startswith("#") or not line.strip():
            continue
        kn, st, cnt = (list(map(int, part.split())) for part in line.split("|"))
        k, n = kn
        assert [binding.strata_na3d_window_start(i, k, n) for i in range(n)] == st
        inv = [binding.strata_na3d_inverse_window(j, k, n) for j in range(n)]
        assert [h - l + 1 for l, h in inv] == cnt
    for n in range(1, 41):
        for k in range(1, n + 1):
            starts = []
            for i in range(n):
                s = i - k // 2                      # centred ...
                while s < 0:
                    s += 1                          # ... shifted inward at the low border
                while s + k > n:
                    s -= 1                          # ... and at the high border
                starts.append(s)
                assert binding.strata_na3d_window_start(i, k, n) == s, (i, k, n)
            for j in range(n):
                attending = [i for i in range(n) if starts[i] <= j < starts[i] + k]
                assert attending == list(range(attending[0], attending[-1] + 1))   # an interval
                assert binding.strata_na3d_inverse_window(j, k, n) == (attending[0], attending[-1]), (j, k, n)
    assert binding.strata_na3d_window_start(0, 5, 4) == -1 and binding.strata_na3d_inverse_window(4, 3, 4) is None
    # hand-derived values of SURVEY.md §8(c): (k, n) = (3, 8) and (5, 8)
    assert [binding.strata_na3d_window_start(i, 3, 8) for i in range(8)] == [0, 0, 1, 2, 3, 4, 5, 5]
    assert [binding.strata_na3d_window_start(i, 5, 8) for i in range(8)] == [0, 0, 0, 1, 2, 3, 3, 3]
    counts = lambda k, n: [h - l + 1 for l, h in (binding.strata_na3d_inverse_window(j, k, n) for j in range(n))]
    assert counts(3, 8) == [2, 3, 4, 3, 3, 4, 3, 2] and counts(5, 8) == [3, 4, 5, 8, 8, 5, 4, 3]


def test_no_cpu_fallback():
    import torch
    q = torch.zeros(1, 2, 2, 2, 1, 32)
    with pytest.raises(binding.StrataError):
        binding.na3d_forward(q, q, q, None, None, (1, 1, 1))
