"""Small forward + backward calls of every kernel family, for compute-sanitizer (memcheck / racecheck / synccheck):

    compute-sanitizer --tool <tool> python tests/sanitizer_smoke.py

Not collected by pytest (no test_ prefix); results are checked against the oracle so that a run under the
sanitizer is also a correctness run.  profiles/r2_sanitizer.md records the outcome."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np  # noqa: E402
import torch  # noqa: E402

import oracle  # noqa: E402
from paper_2606_31248_b200 import binding, workloads as wl  # noqa: E402
from helpers import assert_parity, desc_of, device_inputs, to_f64  # noqa: E402

CASES = [
    dict(name="plane_777", dtype="bf16", grid=(5, 11, 13), window=(3, 7, 7), heads=2, head_dim=64),          # fused fwd + tcgen05 bwd
    dict(name="plane_333_half", dtype="bf16", grid=(4, 9, 10), window=(3, 3, 3), heads=1, head_dim=64, rope_pairing=1),
    dict(name="tile_d128", dtype="bf16", grid=(5, 9, 9), window=(5, 9, 9), heads=1, head_dim=128),           # tile fwd (pre-rotated), SIMT bwd
    dict(name="simt_f32", dtype="f32", grid=(3, 6, 7), window=(3, 3, 3), heads=2, head_dim=32),
]


def main():
    for kw in CASES:
        w = wl.small(**kw)
        inp = wl.make_inputs(w, with_do=True)
        d = device_inputs(w, inp)
        desc = desc_of(w)
        o = torch.empty_like(d["q"])
        lse = torch.empty(desc.lse_shape, dtype=torch.float32, device="cuda")
        ws = binding.alloc_workspace(max(binding.strata_na3d_workspace_bytes(desc, False),
                                         binding.strata_na3d_workspace_bytes(desc, True)), "cuda")
        binding.strata_na3d_fwd(desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], o, lse, ws)
        dq, dk, dv = (torch.empty_like(d["q"]) for _ in range(3))
        binding.strata_na3d_bwd(desc, d["q"], d["k"], d["v"], o, d["do"], lse, d["coords"], d["freqs"], dq, dk, dv, ws)
        torch.cuda.synchronize()
        o_ref, lse_ref = oracle.na3d_fwd(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window,
                                         pairing=w.rope_pairing)
        assert_parity(to_f64(o), o_ref, w.dtype, f"{w.name} O")
        g = oracle.na3d_bwd(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window,
                            pairing=w.rope_pairing)
        for got, ref, nm in zip((dq, dk, dv), g, ("dQ", "dK", "dV")):
            assert_parity(to_f64(got), ref, w.dtype, f"{w.name} {nm}", rms_bound=None if w.dtype == "f32" else 2e-2)
        print(f"{w.name}: OK", flush=True)


if __name__ == "__main__":
    main()
