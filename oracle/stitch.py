"""ORACLE (test infrastructure only): tile stitching, PAPER.md:470-478 (App. F.1, eq. (5)).

"Each tile's output is weighted by a 2D Kaiser-Bessel-derived window, which tapers smoothly to zero at the edges; the
final value at each grid cell is the weighted average of all overlapping tile outputs", S = D^-1 P^T W with
D = P^T W 1.  Reading (R25): for tiles that lie inside one cube face the padding operator P copies cells
(one non-zero per row), so P^T scatters a tile back to its place; the 4-nearest-neighbour rows of P across face edges are
not modelled.  The window is separable, w2d = wy (x) wx, and an INPUT (the paper gives neither length nor shape
parameter): `kbd_window` builds the Kaiser-Bessel-derived window from its textbook definition.
"""
from __future__ import annotations

import numpy as np


def kbd_window(n: int, alpha: float = 4.0) -> np.ndarray:
    """Kaiser-Bessel-derived window of even length n: w[j] = sqrt(sum_{i<=j} k[i] / sum_{i<=n/2} k[i]) for j < n/2,
    mirrored, with the Kaiser window k[i] = I0(pi alpha sqrt(1 - (2 i / (n/2) - 1)^2)), i = 0 .. n/2."""
    assert n % 2 == 0 and n >= 2
    h = n // 2
    i = np.arange(h + 1, dtype=np.float64)
    k = np.i0(np.pi * alpha * np.sqrt(np.maximum(0.0, 1.0 - (2.0 * i / h - 1.0) ** 2)))
    c = np.cumsum(k)
    w = np.sqrt(c[:h] / c[h])
    return np.concatenate([w, w[::-1]])


def stitch(tiles, origins, wy, wx, gh: int, gw: int) -> np.ndarray:
    """tiles [T, C, th, tw], origins [T, 2] = (y0, x0) of each tile in the [C, gh, gw] field -> the weighted average
    of the overlapping tiles, cell by cell (0 where no tile has weight)."""
    tiles = np.asarray(tiles, dtype=np.float64)
    T, C, th, tw = tiles.shape
    w2 = np.outer(np.asarray(wy, dtype=np.float64), np.asarray(wx, dtype=np.float64))
    num = np.zeros((C, gh, gw))
    den = np.zeros((gh, gw))
    for t in range(T):
        y0, x0 = int(origins[t][0]), int(origins[t][1])
        num[:, y0:y0 + th, x0:x0 + tw] += w2[None] * tiles[t]          # P^T (W y)
        den[y0:y0 + th, x0:x0 + tw] += w2                                # D = P^T W 1
    out = np.zeros_like(num)
    np.divide(num, den[None], out=out, where=den[None] > 0)
    return out
