#!/usr/bin/env python
"""bench.py -- StereoRoPE + 3D neighbourhood attention on B200: TFLOP/s, tokens/s, % of roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]

One "step" = one pass of the hot path (strata_na3d_fwd, or strata_na3d_bwd for a backward workload)
over one batch of the seeded synthetic workload.  The default workload is BASELINE.json configs[3]
(the global-rollout batch: the largest config, the one north_star's >= 50 % roofline target is quoted
on); it fits one GPU.  Prints ONE JSON line (rank 0).  N > 1 (torchrun): the path does not shard
(replicas only) -- every rank runs the same workload, `value` is the aggregate.

`--impl reference` times the CPU float64 oracle (oracle/) on the host cores, on a bounded sample of
the same workload (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2606_31248_b200 import workloads as wl  # noqa: E402

WORKLOADS = {"cfg0": 0, "cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4,
             # not BASELINE.json configs: the paper's own attention shapes (workloads.production), as extras
             "prod16": "prod16", "prod32": "prod32", "col16": "col16", "col32": "col32", "dec64": "dec64"}


def workload_of(key: str) -> wl.Workload:
    idx = WORKLOADS[key]
    return wl.config(idx) if isinstance(idx, int) else wl.production(idx)
METRIC = "na3d_stereorope_useful_tflops"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"hbm_gbs": float(p["hbm_gbs"]), "bf16_tflops": float(p["bf16_tflops"]),
                "bf16_tflops_sustained": float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` on `workload`, from the committed ncu
    captures (profiles/*traffic.csv: workload,kernel,dram_bytes_per_launch,capture,commit), newest file first.
    Returns (bytes, "capture @ commit") or (None, None) if that kernel was never captured: the number is a
    property of the capture named beside it, not of this run."""
    import csv
    import glob
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*traffic.csv")), reverse=True):
        with open(path) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and row["kernel"] == kernel:
                    return float(row["dram_bytes_per_launch"]), f"{row.get('capture', '?')} @ {row.get('commit', '?')}"
    return None, None


def flops_of(w: wl.Workload) -> float:
    return w.useful_flops()


def run_reference(args, w: wl.Workload):
    """The oracle as it stands, on the host cores, each step a bounded sample of the workload."""
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    inp = wl.make_inputs(w, threads=os.cpu_count() or 8)
    total = w.batch * w.tokens * w.heads
    rng = np.random.default_rng(w.seed + 555)
    row_flops = (10.0 if w.backward else 4.0) * w.window_size * w.head_dim

    def step(idx):
        if w.backward:
            oracle.na3d_bwd_rows(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window, idx)
        else:
            oracle.na3d_fwd_queries(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window, idx)

    probe = rng.choice(total, size=min(total, 256 if not w.backward else 16), replace=False)
    t0 = time.perf_counter(); step(probe); dt = time.perf_counter() - t0
    budget = 60.0 / max(1, args.steps + args.warmup)          # whole run about a minute
    n = int(max(len(probe), min(total, len(probe) * min(budget, 8.0) / max(dt, 1e-6))))
    idx = rng.choice(total, size=n, replace=False)
    for _ in range(args.warmup):
        step(idx)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step(idx)
    sec = (time.perf_counter() - t0) / args.steps
    tflops = row_flops * n / sec / 1e12
    # dK/dV rows of the backward sample are brute-force (every query is asked): rate is a lower bound
    tok_s = (n / w.heads) / sec
    cores = oracle.num_threads()
    line = {"impl": "reference", "metric": METRIC, "value": tflops, "unit": "TFLOP/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "tokens_per_s": tok_s,
            "config": {"workload": w.name, "sample_rows_per_step": n, "grid": list(w.grid), "window": list(w.window),
                       "heads": w.heads, "head_dim": w.head_dim, "batch": w.batch, "backward": w.backward},
            "cpu_baseline": {"value": tflops, "unit": "TFLOP/s", "cores": cores, "kind": "oracle",
                             "sample": f"{n} random (b, token, head) rows of {w.name} per step",
                             "tokens_per_s": tok_s},
            "e2e": {"value": tflops, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def to_torch(x: np.ndarray, dtype: str):
    import torch
    if dtype == "bf16":
        return torch.from_numpy(x.view(np.int16)).view(torch.bfloat16)
    return torch.from_numpy(x)


class Session:
    """Device-resident inputs + outputs + workspace of one workload."""

    def __init__(self, w: wl.Workload, device, pinned_host: bool):
        import torch
        from paper_2606_31248_b200 import binding
        self.w, self.binding, self.torch = w, binding, torch
        inp = wl.make_inputs(w, threads=min(32, os.cpu_count() or 8), with_do=w.backward)
        names = ["q", "k", "v"] + (["do"] if w.backward else [])
        self.host = {n: to_torch(inp[n], w.dtype) for n in names}
        self.host["coords"], self.host["freqs"] = torch.from_numpy(inp["coords"]), torch.from_numpy(inp["freqs"])
        if pinned_host:
            self.host = {n: t.pin_memory() for n, t in self.host.items()}
        self.dev = {n: t.to(device, non_blocking=True) for n, t in self.host.items()}
        self.desc = binding.NA3DDesc(w.batch, w.heads, w.head_dim, w.grid, w.window, w.rope_axes, w.rope_pairing,
                                     binding.DTYPE_F32 if w.dtype == "f32" else binding.DTYPE_BF16)
        self.o = torch.empty_like(self.dev["q"])
        self.lse = torch.empty(self.desc.lse_shape, dtype=torch.float32, device=device)
        need = binding.strata_na3d_workspace_bytes(self.desc, False)
        if w.backward:
            need = max(need, binding.strata_na3d_workspace_bytes(self.desc, True))
            self.grads = [torch.empty_like(self.dev["q"]) for _ in range(3)]
        self.ws = binding.alloc_workspace(need, device)
        self.device = device
        if w.backward:          # the backward consumes the forward's O and LSE (not timed)
            self.forward()
        torch.cuda.synchronize()

    def forward(self):
        d = self.dev
        self.binding.strata_na3d_fwd(self.desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], self.o, self.lse, self.ws)

    def backward(self):
        d = self.dev
        self.binding.strata_na3d_bwd(self.desc, d["q"], d["k"], d["v"], self.o, d["do"], self.lse, d["coords"],
                                     d["freqs"], *self.grads, self.ws)

    def step(self):
        self.backward() if self.w.backward else self.forward()

    # ---- end to end through the host-buffer entry points
    def setup_e2e(self):
        torch, b = self.torch, self.binding
        self.ws_host = b.alloc_workspace(b.strata_na3d_host_workspace_bytes(self.desc, self.w.backward), self.device)
        if self.w.backward:
            self.h_o = self.o.to("cpu").pin_memory()
            self.h_lse = self.lse.to("cpu").pin_memory()
            self.h_out = [torch.empty_like(self.host["q"]).pin_memory() for _ in range(3)]
            n_in = 5 * self.host["q"].numel() * self.host["q"].element_size() + self.h_lse.numel() * 4
            n_out = 3 * self.host["q"].numel() * self.host["q"].element_size()
        else:
            self.h_o = torch.empty_like(self.host["q"]).pin_memory()
            self.h_lse = torch.empty(self.desc.lse_shape, dtype=torch.float32).pin_memory()
            n_in = 3 * self.host["q"].numel() * self.host["q"].element_size()
            n_out = self.h_o.numel() * self.h_o.element_size() + self.h_lse.numel() * 4
        n_in += self.host["coords"].numel() * 4 + self.host["freqs"].numel() * 4
        return n_in, n_out

    def step_e2e(self):
        h, b = self.host, self.binding
        if self.w.backward:
            b.strata_na3d_bwd_host(self.desc, h["q"], h["k"], h["v"], self.h_o, h["do"], self.h_lse, h["coords"],
                                   h["freqs"], *self.h_out, self.ws_host)
        else:
            b.strata_na3d_fwd_host(self.desc, h["q"], h["k"], h["v"], h["coords"], h["freqs"], self.h_o, self.h_lse,
                                   self.ws_host)


def max_over_ranks(torch, ms: float, dist, device) -> float:
    """Whole-job step time = the slowest rank's (all-reduce MAX; identity when not distributed)."""
    if dist is None:
        return ms
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate(per_rank_units: float, world: int, ms: float) -> float:
    """Replicas only: every rank processes the same units in `ms`; whole-job rate."""
    return world * per_rank_units / (ms * 1e-3)


def time_steps(torch, fn, steps, dist=None):
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s.record()
    for _ in range(steps):
        fn()
    e.record()
    torch.cuda.synchronize()
    ms = s.elapsed_time(e) / steps
    if dist is not None:
        ms = max_over_ranks(torch, ms, dist, "cuda")
        dist.barrier()
    return ms


def cpu_baseline(w: wl.Workload, sess: Session, seconds: float = 12.0):
    """The oracle, as it stands, on a bounded sample of the same workload (host cores of this box)."""
    import oracle
    inp = {n: (t.view(sess.torch.int16).numpy().view(np.uint16) if w.dtype == "bf16" and n in ("q", "k", "v", "do")
               else t.numpy()) for n, t in sess.host.items()}
    total = w.batch * w.tokens * w.heads
    rng = np.random.default_rng(w.seed + 555)
    row_flops = (10.0 if w.backward else 4.0) * w.window_size * w.head_dim

    def run(idx):
        t0 = time.perf_counter()
        if w.backward:
            oracle.na3d_bwd_rows(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window, idx)
        else:
            oracle.na3d_fwd_queries(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window, idx)
        return time.perf_counter() - t0

    n0 = min(total, 16 if w.backward else 512)
    dt = run(rng.choice(total, size=n0, replace=False))
    n = int(max(n0, min(total, n0 * seconds / max(dt, 1e-6))))
    dt = run(rng.choice(total, size=n, replace=False))
    return {"value": row_flops * n / dt / 1e12, "unit": "TFLOP/s", "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{n} random (b, token, head) rows of {w.name}, {dt:.1f} s of oracle time"
                      + (" (dK/dV rows by brute force over all queries: a lower bound)" if w.backward else ""),
            "tokens_per_s": (n / w.heads) / dt}


def measure_streaming(peaks, w: wl.Workload, steps: int = 20):
    """The elementwise kernels around the attention (NEXT rows of SURVEY.md §8(f)) as HBM streams: bytes each must
    move / time / measured copy bandwidth.  Sizes follow config 3 (24 tiles of 128 x 128 patches, stride 112, 8 levels),
    scaled so that every working set exceeds the 126 MB L2 (no flush needed); inputs are seeded torch.rand."""
    import torch
    from paper_2606_31248_b200 import binding
    dev = torch.device("cuda", torch.cuda.current_device())
    g = torch.Generator(device=dev); g.manual_seed(wl.BASE_SEED + 7)
    out = {}

    def run(name, fn, nbytes, note):
        for _ in range(3):
            fn()
        ms = time_steps(torch, fn, steps)
        gbs = nbytes / (ms * 1e-3) / 1e9
        out[name] = {"ms": ms, "bytes": int(nbytes), "achieved_gbs": gbs, "frac_of_hbm_peak": gbs / peaks["hbm_gbs"], "size": note}

    n = 4 * w.batch * w.tokens                                        # eq. (1) / eq. (2): points
    lat = (torch.rand(n, generator=g, device=dev, dtype=torch.float64) - 0.5) * 0.4 + 0.3
    lon = (torch.rand(n, generator=g, device=dev, dtype=torch.float64) - 0.5) * 0.4 + 1.0
    coords = torch.empty(n, 2, device=dev)
    run("stereo_coords", lambda: binding.strata_stereo_coords(lat, lon, 0.3, 1.0, float(wl.N_TOTAL), coords), n * 24,
        f"{n} points (4 x config 3's tokens): 16 B in, 8 B out")
    u, v = torch.rand(n, generator=g, device=dev), torch.rand(n, generator=g, device=dev)
    ul, vl = torch.empty_like(u), torch.empty_like(v)
    run("wind_to_tile_frame", lambda: binding.strata_wind_to_tile_frame(u, v, lat, lon, 0.3, 1.0, ul, vl), n * 32,
        f"{n} points: 8 + 16 B in, 8 B out")
    del lat, lon, coords, u, v, ul, vl
    T, C, th, st = 24, 128, 128, 112                                  # eq. (5): six faces of 2 x 2 tiles side by side
    origins = torch.tensor([(ty * st, f * (th + st) + tx * st) for f in range(6) for ty in range(2) for tx in range(2)],
                           dtype=torch.int32, device=dev)
    gh, gw = th + st, 6 * (th + st)
    tiles = torch.rand(T, C, th, th, generator=g, device=dev)
    win = torch.sin(torch.arange(th, device=dev, dtype=torch.float32).add(0.5).mul(3.141592653589793 / th))
    field = torch.empty(C, gh, gw, device=dev)
    run("tile_stitch", lambda: binding.strata_tile_stitch(tiles, origins, win, win, field),
        tiles.numel() * 4 + field.numel() * 4, f"{T} tiles x {C} channels x {th} x {th}, stride {st} -> [{C}, {gh}, {gw}]")
    del tiles, field
    torch.cuda.empty_cache()
    return out


def measure(w: wl.Workload, args, dist, rank, peaks, with_e2e=True, with_cpu=True, with_normgate=False):
    import torch
    from paper_2606_31248_b200 import binding
    dev = torch.device("cuda", torch.cuda.current_device())
    sess = Session(w, dev, pinned_host=with_e2e)
    for _ in range(max(3, args.warmup)):
        sess.step()
    torch.cuda.synchronize()
    launches_per_step = binding.strata_na3d_last_launch_count()
    sampler = ClockSampler(torch.cuda.current_device())
    sampler.start()
    ms = time_steps(torch, sess.step, args.steps, dist)          # the headline: nothing but the library's own launches
    clocks = sampler.stop()
    # per-kernel times come from a loop of their own (two event records per kernel would sit in the timed region)
    binding.strata_na3d_set_profiling(True)
    time_steps(torch, sess.step, args.steps, None)
    prof = binding.strata_na3d_profile_read()
    binding.strata_na3d_set_profiling(False)
    per_kernel = {}
    for name, t in prof:
        per_kernel.setdefault(name, []).append(t)
    per_kernel = {k: sum(v) / len(v) for k, v in per_kernel.items()}
    n_gpus = args.gpus
    flops, bytes_ = flops_of(w), w.compulsory_bytes()
    tflops = aggregate(flops, n_gpus, ms) / 1e12
    tok_s = aggregate(w.batch * w.tokens, n_gpus, ms)
    # roofline of the dominant kernel: all five configs are HBM-bound by SURVEY.md §8(d)
    dom = max(per_kernel, key=per_kernel.get) if per_kernel else None
    dom_ms = per_kernel.get(dom, ms)
    t_hbm = bytes_ / (peaks["hbm_gbs"] * 1e9)
    t_tc = flops / (peaks["bf16_tflops"] * 1e12)
    achieved = bytes_ / (dom_ms * 1e-3) / 1e9
    traffic, traffic_capture = measured_traffic(w.name, dom)
    roofline = {"bound": "hbm", "kernel": dom, "kernel_ms": dom_ms, "achieved": achieved, "peak": peaks["hbm_gbs"],
                "unit": "GB/s", "frac": achieved / peaks["hbm_gbs"], "traffic": traffic, "traffic_capture": traffic_capture,
                "peak_source": peaks["source"], "algorithmic_bytes": bytes_,
                "roofline_ms": max(t_hbm, t_tc) * 1e3, "step_frac_of_roofline": max(t_hbm, t_tc) * 1e3 / ms,
                "kernels_ms": per_kernel}
    out = {"ms_per_step": ms, "tflops": tflops, "tokens_per_s": tok_s, "launches_per_step": launches_per_step,
           "roofline": roofline, "clocks": clocks,
           "impl": {0: "auto", 1: "simt", 2: "tcgen05"}.get(binding.strata_na3d_impl_selected(sess.desc, w.backward))}
    if with_normgate and not w.backward:
        # PAPER.md:390 around the same forward: QK-RMSNorm + head gate.  A fused version would move the same bytes as the
        # plain forward plus 4 B of gate logit per (token, head); today three streaming kernels surround the attention.
        gate = torch.zeros((w.batch,) + tuple(w.grid) + (w.heads,), dtype=torch.float32, device=dev)
        ws_ng = binding.alloc_workspace(binding.strata_na3d_normgate_workspace_bytes(sess.desc, False), dev)
        d = sess.dev
        ng = lambda: binding.strata_na3d_normgate_fwd(sess.desc, d["q"], d["k"], d["v"], d["coords"], d["freqs"], gate, 1e-6,
                                                      sess.o, sess.lse, ws_ng)
        for _ in range(3):
            ng()
        k_ng = max(3, min(args.steps, 10))
        ms_ng = time_steps(torch, ng, k_ng, None)
        binding.strata_na3d_set_profiling(True)
        ng(); torch.cuda.synchronize()
        ng_kernels = {}
        for name, t in binding.strata_na3d_profile_read():
            ng_kernels[name] = ng_kernels.get(name, 0.0) + t
        binding.strata_na3d_set_profiling(False)
        ideal = (bytes_ + gate.numel() * 4) / (peaks["hbm_gbs"] * 1e9) * 1e3
        out["normgate_fwd"] = {"ms_per_step": ms_ng, "steps": k_ng, "vs_plain_forward": ms_ng / ms,
                               "launches_per_step": binding.strata_na3d_last_launch_count(),
                               "frac_of_roofline": ideal / ms_ng, "kernels_ms": ng_kernels}
        del gate, ws_ng
    if with_e2e:
        n_in, n_out = sess.setup_e2e()
        sess.step_e2e(); torch.cuda.synchronize()
        k = max(1, min(args.steps, args.e2e_steps))
        ms_e = time_steps(torch, sess.step_e2e, k, dist)
        out["e2e"] = {"value": n_gpus * flops / (ms_e * 1e-3) / 1e12, "unit": "TFLOP/s", "ms_per_step": ms_e, "steps": k,
                      "tokens_per_s": n_gpus * w.batch * w.tokens / (ms_e * 1e-3),
                      "h2d_bytes_per_step": int(n_in), "d2h_bytes_per_step": int(n_out),
                      "api": "strata_na3d_bwd_host" if w.backward else "strata_na3d_fwd_host"}
    if with_cpu and rank == 0 and n_gpus == 1:
        out["cpu_baseline"] = cpu_baseline(w, sess)
    del sess
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(WORKLOADS))
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--extras", default="cfg1,cfg2,cfg4,prod32,col32,dec64", help="other configs summarised in the same line ('' = none)")
    args = ap.parse_args()
    w = workload_of(args.workload)
    if args.impl == "reference":
        run_reference(args, w)
        return

    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist = dist_mod
    peaks = load_peaks()
    main_res = measure(w, args, dist, rank, peaks, with_normgate=(world == 1 and bool(args.extras)))
    others = {}
    if args.extras and world == 1:
        short = argparse.Namespace(**{**vars(args), "steps": max(3, min(args.steps, 10)), "e2e_steps": 1})
        for name in [x for x in args.extras.split(",") if x and x != args.workload]:
            r = measure(workload_of(name), short, None, rank, peaks, with_e2e=False, with_cpu=False)
            others[name] = {"ms_per_step": r["ms_per_step"], "tflops": r["tflops"], "tokens_per_s": r["tokens_per_s"],
                            "frac_of_roofline": r["roofline"]["step_frac_of_roofline"], "impl": r["impl"],
                            "kernels_ms": r["roofline"]["kernels_ms"]}
        if "normgate_fwd" in main_res:
            others["normgate_fwd_" + args.workload] = main_res["normgate_fwd"]
        others["streaming_kernels"] = measure_streaming(peaks, w, steps=max(3, min(args.steps, 20)))
    if rank == 0:
        line = {"metric": METRIC, "value": main_res["tflops"], "unit": "TFLOP/s", "n_gpus": args.gpus,
                "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": main_res["ms_per_step"],
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32" if w.dtype == "f32" else "bf16", "data": "synthetic",
                "tokens_per_s": main_res["tokens_per_s"],
                "config": {"workload": w.name, "baseline_config_index": w.index, "batch": w.batch,
                           "grid": list(w.grid), "heads": w.heads, "head_dim": w.head_dim, "window": list(w.window),
                           "backward": w.backward, "impl": main_res["impl"], "parallelism": "replicas only",
                           "l2_policy": "inputs larger than L2 (no flush)" if w.compulsory_bytes() > 2.6e8
                           else "inputs fit L2: latency-bound config, reported as is"},
                "roofline": main_res["roofline"], "clocks": main_res["clocks"],
                "e2e": main_res.get("e2e"), "gpu_launches": main_res["launches_per_step"] * args.steps,
                "cpu_baseline": main_res.get("cpu_baseline"), "other_workloads": others}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
