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


def test_no_cpu_fallback():
    import torch
    q = torch.zeros(1, 2, 2, 2, 1, 32)
    with pytest.raises(binding.StrataError):
        binding.na3d_forward(q, q, q, None, None, (1, 1, 1))
