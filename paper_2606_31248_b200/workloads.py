"""Seeded synthetic workloads for StereoRoPE + 3D neighbourhood attention.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path: it
produces inputs and nothing else.  It holds no attention / RoPE arithmetic.  What it does
hold is the *input recipe* (DESIGN.md §4): random Q/K/V/dO, the default rotary frequency
table, and the geometry that turns a tile of a cubed-sphere face into the per-token
stereographic coordinates the kernel takes as an input (eq. (1)); the CUDA
path never computes eq. (1) itself, and `oracle/geometry.py` has its own, independent
restatement of eq. (1) that the tests hold this generator against.

The five configurations are BASELINE.json's `configs[0..4]`; SURVEY.md §8(d) gives the
recipe (seed = 31248*10 + config index, numpy `default_rng`).  The SCREAM dataset and the
trained STRATA weights are not available, so these synthetic tensors stand
in for the activations of a STRATA attention block.

Everything is generated on the host with numpy; bf16 tensors are returned as uint16 bit
patterns (numpy has no bfloat16) produced by round-to-nearest-even from float32.
"""
from __future__ import annotations

import math
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field, replace
from typing import Dict, Optional, Tuple

import numpy as np

# ----------------------------------------------------------------------------------------
# Constants of the recipe (SURVEY.md §8(c) readings 4, 5, 8, 9, 11)
# ----------------------------------------------------------------------------------------
FACE_CELLS = 2048                       # native cells per cube-face edge
PATCH = 4                               # horizontal patch size p_h (Table S1)
FACE_PATCHES = FACE_CELLS // PATCH      # 512 patch tokens per face edge
N_TOTAL = 6 * FACE_CELLS * FACE_CELLS   # reading 8: horizontal native cells on the sphere
ROPE_BASE = 100.0                       # reading 4: generator default, not from PAPER.md
BASE_SEED = 31248 * 10


@dataclass(frozen=True)
class Workload:
    """Shape and recipe of one synthetic workload (one BASELINE.json config)."""
    name: str
    index: int                           # BASELINE.json configs[] index (-1: ad hoc)
    batch: int
    heads: int
    head_dim: int
    grid: Tuple[int, int, int]           # (L, Y, X) = (levels, y, x) tokens
    window: Tuple[int, int, int]         # (k_L, k_Y, k_X)
    dtype: str                           # "f32" | "bf16"
    backward: bool = False
    value_scale: str = "unit"            # "unit": N(0,1); "rsqrt_d": N(0,1)/sqrt(d); "qknorm"
    center: str = "tile"                 # projection centre: "tile" (paper) | "face" (cfg 0)
    placement: str = "random"            # "random" tile per sample | "rollout" (cfg 3)
    rope_axes: int = 2
    rope_pairing: int = 0                # 0 interleaved (2j,2j+1), 1 half (j, j+d/2)
    seed: int = BASE_SEED

    @property
    def tokens(self) -> int:
        return self.grid[0] * self.grid[1] * self.grid[2]

    @property
    def window_size(self) -> int:
        return self.window[0] * self.window[1] * self.window[2]

    @property
    def elem_bytes(self) -> int:
        return 4 if self.dtype == "f32" else 2

    def useful_flops(self) -> float:
        """4*N*W*d per head-sample forward, 10*N*W*d backward."""
        per = (10.0 if self.backward else 4.0) * self.tokens * self.window_size * self.head_dim
        return per * self.heads * self.batch

    def compulsory_bytes(self) -> float:
        """Q,K,V read + O written (+LSE fp32 + coords); backward: 8 tensors + LSE."""
        tensor = self.batch * self.tokens * self.heads * self.head_dim * self.elem_bytes
        lse = self.batch * self.heads * self.tokens * 4
        coords = self.batch * self.tokens * self.rope_axes * 4
        if self.backward:
            return 8.0 * tensor + lse + coords
        return 4.0 * tensor + lse + coords


def config(index: int) -> Workload:
    """BASELINE.json configs[index]."""
    s = BASE_SEED + index
    if index == 0:
        return Workload("cfg0_tiny_f32", 0, 1, 2, 32, (4, 16, 16), (3, 5, 5), "f32",
                        value_scale="unit", center="face", seed=s)
    if index == 1:
        return Workload("cfg1_train_tile_fwd", 1, 4, 8, 64, (8, 64, 64), (3, 7, 7), "bf16",
                        value_scale="rsqrt_d", seed=s)
    if index == 2:
        return Workload("cfg2_wide_head_fwd", 2, 2, 16, 128, (8, 128, 128), (5, 9, 9), "bf16",
                        value_scale="rsqrt_d", seed=s)
    if index == 3:
        return Workload("cfg3_global_rollout_fwd", 3, 24, 8, 64, (8, 128, 128), (3, 7, 7),
                        "bf16", value_scale="rsqrt_d", placement="rollout", seed=s)
    if index == 4:
        return Workload("cfg4_train_tile_bwd", 4, 4, 8, 64, (8, 64, 64), (3, 7, 7), "bf16",
                        backward=True, value_scale="rsqrt_d", seed=s)
    raise ValueError(f"no BASELINE.json config {index}")


def production(which: str) -> Workload:
    """The paper's own attention shapes (PAPER.md:325-326 Table S1, 454): 24 levels, 16 heads, head_dim 1024 / 16 =
    64, NATTEN kernel size 9 (read as 9 x 9 x 9, R2), tiles of 64 x 64 or 128 x 128 cells at patch size 4;
    inputs as QK-RMSNorm leaves them.  "col*": the column-wise attention blocks that alternate with
    them: every level of one (y, x) column.  "dec64": the de-aliasing decoder's NA3D blocks (PAPER.md:326:
    embedding dimension 128, NA3D kernel size 9, at full horizontal resolution: the 64 x 64 cells of a 16 x 16-patch
    tile, 24 levels); the paper gives no head count for it -- read as ONE head of 128 channels (R26; two
    heads of 64 would be the prod shapes' kernel).  Not BASELINE.json configs: extra bench / parity shapes."""
    s = BASE_SEED + 50
    if which == "dec64":
        return Workload("dec64_fwd", -1, 2, 1, 128, (24, 64, 64), (9, 9, 9), "bf16", value_scale="qknorm", seed=s)
    shapes = {"prod16": ((24, 16, 16), (9, 9, 9)), "prod32": ((24, 32, 32), (9, 9, 9)),
              "col16": ((24, 16, 16), (24, 1, 1)), "col32": ((24, 32, 32), (24, 1, 1))}
    grid, window = shapes[which]
    return Workload(f"{which}_fwd", -1, 8 if grid[1] == 16 else 2, 16, 64, grid, window, "bf16", value_scale="qknorm", seed=s)


def small(name: str = "small", **kw) -> Workload:
    """Ad-hoc small workload for parity sweeps; keyword overrides on a 1x2x32 default."""
    base = Workload(name, -1, 1, 2, 32, (3, 6, 7), (3, 3, 3), "f32", seed=BASE_SEED + 99)
    return replace(base, **kw)


# ----------------------------------------------------------------------------------------
# bf16 helpers (bit-level; RNE) -- data movement only
# ----------------------------------------------------------------------------------------
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bfloat16 bit pattern (uint16), round-to-nearest-even."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rounding = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + rounding) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """bfloat16 bit pattern (uint16) -> float32 (exact)."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def as_f64(x: np.ndarray, dtype: str) -> np.ndarray:
    """Exact float64 view of a generated tensor (bf16 bits or float32)."""
    if dtype == "bf16":
        return bf16_bits_to_f32(x).astype(np.float64)
    return np.asarray(x, dtype=np.float64)


# ----------------------------------------------------------------------------------------
# Geometry: equiangular cubed sphere -> (lat, lon) -> tile-centred stereographic, eq. (1)
# ----------------------------------------------------------------------------------------
def l_scale(n_total: int = N_TOTAL) -> float:
    """l_scale = sqrt(4*pi/N_total)."""
    return math.sqrt(4.0 * math.pi / n_total)


def patch_angle(p):
    """Equiangular face coordinate of the centre of patch index p (may be fractional).

    Cell i has centre (i + 1/2)*(pi/2)/2048 - pi/4 (reading 11); patch p covers cells
    4p..4p+3, so its centre sits at cell coordinate 4p + 2 (reading 9)."""
    return (PATCH * np.asarray(p, dtype=np.float64) + PATCH / 2.0) * (math.pi / 2.0) / FACE_CELLS - math.pi / 4.0


def face_point_to_latlon(face: int, alpha, beta):
    """(alpha, beta) on cube face `face` -> (lat, lon) in radians (reading 11).

    Face 0 is centred at (lat, lon) = (0, 0) with point ~ (1, tan a, tan b); faces 1..3
    follow eastwards in 90 degree steps; 4 = north polar face, 5 = south polar face."""
    ta, tb = np.tan(alpha), np.tan(beta)
    one = np.ones_like(ta)
    if face < 4:
        x0, y0, z0 = one, ta, tb
        ang = face * (math.pi / 2.0)
        ca, sa = math.cos(ang), math.sin(ang)
        X, Y, Z = ca * x0 - sa * y0, sa * x0 + ca * y0, z0
    elif face == 4:
        X, Y, Z = -tb, ta, one
    elif face == 5:
        X, Y, Z = tb, ta, -one
    else:
        raise ValueError("face must be 0..5")
    r = np.sqrt(X * X + Y * Y + Z * Z)
    return np.arcsin(Z / r), np.arctan2(Y, X)


def stereographic_xy(lat, lon, lat0: float, lon0: float, n_total: int = N_TOTAL):
    """Tile-centred stereographic coordinates, eq. (1), in float64."""
    dlon = lon - lon0
    cos_c = math.sin(lat0) * np.sin(lat) + math.cos(lat0) * np.cos(lat) * np.cos(dlon)
    if np.any(1.0 + cos_c <= 0.5):       # reading 17: far from the antipode by construction
        raise ValueError("token too far from projection centre")
    k = 2.0 / (1.0 + cos_c)
    ls = l_scale(n_total)
    x = (k / ls) * np.cos(lat) * np.sin(dlon)
    y = (k / ls) * (math.cos(lat0) * np.sin(lat) - math.sin(lat0) * np.cos(lat) * np.cos(dlon))
    return x, y


def tile_coords(face: int, py0: int, px0: int, ny: int, nx: int, center: str = "tile"):
    """Stereographic (x, y) of the ny x nx patch tokens of a tile; returns [ny, nx, 2] f64."""
    alpha = patch_angle(px0 + np.arange(nx))          # x index runs along alpha
    beta = patch_angle(py0 + np.arange(ny))           # y index runs along beta
    A, Bt = np.meshgrid(alpha, beta, indexing="xy")   # [ny, nx]
    lat, lon = face_point_to_latlon(face, A, Bt)
    if center == "tile":
        a0 = patch_angle(px0 + (nx - 1) / 2.0)
        b0 = patch_angle(py0 + (ny - 1) / 2.0)
        lat0, lon0 = face_point_to_latlon(face, np.float64(a0), np.float64(b0))
    elif center == "face":
        lat0, lon0 = face_point_to_latlon(face, np.float64(0.0), np.float64(0.0))
    else:
        raise ValueError("center must be 'tile' or 'face'")
    x, y = stereographic_xy(lat, lon, float(lat0), float(lon0))
    return np.stack([x, y], axis=-1)


def tile_placements(w: Workload):
    """(face, py0, px0) per batch element, seeded (SURVEY.md §8(d) coords column)."""
    rng = np.random.default_rng([w.seed, 7])
    _, ny, nx = w.grid
    out = []
    if w.placement == "rollout":
        # 4 tiles per face x 6 faces: a 2x2 block with stride (tile - 16) patches (overlap 16)
        stride_y, stride_x = ny - 16, nx - 16
        for face in range(6):
            oy = int(rng.integers(0, FACE_PATCHES - (ny + stride_y) + 1))
            ox = int(rng.integers(0, FACE_PATCHES - (nx + stride_x) + 1))
            for ty in range(2):
                for tx in range(2):
                    out.append((face, oy + ty * stride_y, ox + tx * stride_x))
        out = out[: w.batch] if w.batch <= len(out) else out + out[: w.batch - len(out)]
    else:
        for _ in range(w.batch):
            face = int(rng.integers(0, 6)) if w.center == "tile" else 0
            out.append((face, int(rng.integers(0, FACE_PATCHES - ny + 1)),
                        int(rng.integers(0, FACE_PATCHES - nx + 1))))
    return out


def make_coords(w: Workload) -> np.ndarray:
    """coords [B, L, Y, X, A] float32; (x, y) shared by all levels; axis 2 (A=3) = level."""
    L, ny, nx = w.grid
    A = w.rope_axes
    out = np.zeros((w.batch, L, ny, nx, max(A, 1)), dtype=np.float32)
    if A == 0:
        return out[..., :0]
    for b, (face, py0, px0) in enumerate(tile_placements(w)):
        xy = tile_coords(face, py0, px0, ny, nx, w.center)
        out[b, :, :, :, 0:2] = xy[None].astype(np.float32)
        if A >= 3:
            out[b, :, :, :, 2] = np.arange(L, dtype=np.float32)[:, None, None]
    return out


def make_freqs(head_dim: int, rope_axes: int = 2, base: float = ROPE_BASE) -> np.ndarray:
    """Default axial frequency table F[A, d/2] float32 (readings 4, 5).

    The d/2 rotary pairs are split evenly between the axes; pair t of an axis block of size
    m gets theta_t = base**(-t/m); a pair rotates with exactly one axis."""
    half = head_dim // 2
    F = np.zeros((max(rope_axes, 1), half), dtype=np.float64)
    if rope_axes == 0:
        return F[:0].astype(np.float32)
    per = half // rope_axes
    for a in range(rope_axes):
        lo = a * per
        hi = half if a == rope_axes - 1 else lo + per
        m = hi - lo
        F[a, lo:hi] = base ** (-np.arange(m, dtype=np.float64) / m)
    return F.astype(np.float32)


# ----------------------------------------------------------------------------------------
# Random tensors
# ----------------------------------------------------------------------------------------
_TENSOR_ID = {"q": 1, "k": 2, "v": 3, "do": 4}


def _fill_one(args):
    w, name, b = args
    shape = w.grid + (w.heads, w.head_dim)
    rng = np.random.default_rng([w.seed, _TENSOR_ID[name], b])
    x = rng.standard_normal(shape, dtype=np.float32)
    if name != "do":
        if w.value_scale == "rsqrt_d":
            x *= np.float32(1.0 / math.sqrt(w.head_dim))
        elif w.value_scale == "qknorm" and name in ("q", "k"):
            # what QK-RMSNorm hands the kernel: rows of RMS 1, logits up to sqrt(d)
            x /= np.sqrt(np.mean(x.astype(np.float64) ** 2, axis=-1, keepdims=True)).astype(np.float32)
    return f32_to_bf16_bits(x) if w.dtype == "bf16" else x


def make_tensor(w: Workload, name: str, threads: int = 8) -> np.ndarray:
    """One of q, k, v, do as [B, L, Y, X, H, d]; float32 or bf16 bits (uint16)."""
    jobs = [(w, name, b) for b in range(w.batch)]
    if w.batch == 1 or threads <= 1:
        parts = [_fill_one(j) for j in jobs]
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            parts = list(ex.map(_fill_one, jobs))
    return np.stack(parts, axis=0)


def make_inputs(w: Workload, threads: int = 8, with_do: Optional[bool] = None) -> Dict[str, np.ndarray]:
    """All inputs of a workload: q, k, v (+ do), coords [B,L,Y,X,A] f32, freqs [A,d/2] f32."""
    out = {n: make_tensor(w, n, threads) for n in ("q", "k", "v")}
    if with_do if with_do is not None else w.backward:
        out["do"] = make_tensor(w, "do", threads)
    out["coords"] = make_coords(w)
    out["freqs"] = make_freqs(w.head_dim, w.rope_axes)
    return out
