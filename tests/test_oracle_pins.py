"""Pins for the CPU float64 oracle (oracle/na3d_oracle.c): what the paper and the mathematics fix.

None of these re-types the oracle's loops: each compares it with an independent formulation
(dense masked attention in numpy / torch float64 autograd, complex-multiply RoPE, banded 1D
attention), a closed form, an invariant, or a brute-force enumeration on a tiny grid.
"""
import itertools
import math
import os

import numpy as np
import pytest
import torch

from paper_2606_31248_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ independent helpers
def slide_then_clamp(i, k, n):
    """NATTEN-style window in words: centre the window on i, then shift it inward until it fits."""
    lo = i - k // 2
    hi = lo + k
    while lo < 0:
        lo += 1
        hi += 1
    while hi > n:
        lo -= 1
        hi -= 1
    return list(range(lo, hi))


def neighbour_mask(grid, window):
    """Dense boolean [N, N] mask from the enumeration above (independent of the oracle)."""
    L, Y, X = grid
    N = L * Y * X
    M = np.zeros((N, N), dtype=bool)
    for l, y, x in itertools.product(range(L), range(Y), range(X)):
        i = (l * Y + y) * X + x
        for a in slide_then_clamp(l, window[0], L):
            for b in slide_then_clamp(y, window[1], Y):
                for c in slide_then_clamp(x, window[2], X):
                    M[i, (a * Y + b) * X + c] = True
    return M


def rope_complex(x, coords, freqs, pairing=0):
    """RoPE as a complex multiplication (a + ib) e^{i phi}; x [B,L,Y,X,H,D] float64."""
    D = x.shape[-1]
    phi = np.einsum("blyxa,aj->blyxj", coords.astype(np.float64), freqs.astype(np.float64))
    rot = np.exp(1j * phi)[..., None, :]                       # [B,L,Y,X,1,D/2]
    out = np.empty_like(x)
    if pairing == 0:
        z = (x[..., 0::2] + 1j * x[..., 1::2]) * rot
        out[..., 0::2], out[..., 1::2] = z.real, z.imag
    else:
        z = (x[..., : D // 2] + 1j * x[..., D // 2:]) * rot
        out[..., : D // 2], out[..., D // 2:] = z.real, z.imag
    return out


def dense_masked_attention(q, k, v, mask, scale):
    """Textbook softmax(Q K^T scale + mask) V per (b, h); q,k,v [B,N,H,D] float64."""
    s = np.einsum("bihd,bjhd->bhij", q, k) * scale
    s = np.where(mask[None, None], s, -np.inf)
    m = s.max(-1, keepdims=True)
    e = np.exp(s - m)
    z = e.sum(-1, keepdims=True)
    o = np.einsum("bhij,bjhd->bihd", e / z, v)
    return o, (m + np.log(z))[..., 0]                           # o [B,N,H,D], lse [B,H,N]


def rand_problem(seed, B=1, H=2, D=8, grid=(3, 4, 5), A=2, coord_scale=3.0):
    rng = np.random.default_rng(seed)
    shp = (B,) + grid + (H, D)
    q, k, v, do = (rng.standard_normal(shp) for _ in range(4))
    coords = (rng.standard_normal((B,) + grid + (A,)) * coord_scale).astype(np.float32)
    freqs = rng.uniform(0.05, 1.0, size=(A, D // 2)).astype(np.float32)
    return q, k, v, do, coords, freqs


def flat(x):
    B, L, Y, X, H, D = x.shape
    return x.reshape(B, L * Y * X, H, D)


def reference_fwd(q, k, v, coords, freqs, grid, window, scale=None, pairing=0):
    D = q.shape[-1]
    scale = scale or 1.0 / math.sqrt(D)
    qr, kr = rope_complex(q, coords, freqs, pairing), rope_complex(k, coords, freqs, pairing)
    o, lse = dense_masked_attention(flat(qr), flat(kr), flat(v), neighbour_mask(grid, window), scale)
    return o.reshape(q.shape), lse.reshape(lse.shape[:2] + grid)


# ------------------------------------------------------------------ A3 neighbourhood
def _golden_windows():
    rows = []
    for line in open(os.path.join(GOLD, "window_starts.txt")):
        if line.startswith("#") or not line.strip():
            continue
        kn, starts, counts = [p.split() for p in line.split("|")]
        rows.append((int(kn[0]), int(kn[1]), list(map(int, starts)), list(map(int, counts))))
    return rows


@pytest.mark.parametrize("k,n,starts,counts", _golden_windows())
def test_window_start_hand_values(oracle_mod, k, n, starts, counts):
    got = [oracle_mod.window_start(i, k, n) for i in range(n)]
    assert got == starts
    per_key = [sum(1 for i in range(n) if got[i] <= j < got[i] + k) for j in range(n)]
    assert per_key == counts


@pytest.mark.parametrize("k,n", [(1, 1), (1, 5), (3, 3), (3, 8), (5, 8), (7, 64), (9, 128), (4, 6), (2, 7), (6, 6)])
def test_window_start_vs_enumeration(oracle_mod, k, n):
    for i in range(n):
        w = slide_then_clamp(i, k, n)
        assert oracle_mod.window_start(i, k, n) == w[0]
        assert len(w) == k and w[0] >= 0 and w[-1] < n
        if k // 2 <= i < n - (k - 1 - k // 2):                # interior: window is centred
            assert w[0] == i - k // 2


def test_uniform_attention_reads_window_out(oracle_mod):
    """K = 0 gives uniform weights; V = one-hot(token) makes O_i the window indicator / W."""
    grid, window = (3, 4, 5), (3, 3, 5)
    N, W = 60, 45
    B, H, D = 1, 1, N
    q = np.random.default_rng(0).standard_normal((B,) + grid + (H, D))
    k = np.zeros_like(q)
    v = np.eye(N).reshape((B,) + grid + (H, D))
    coords = np.zeros((B,) + grid + (2,), np.float32)
    freqs = np.ones((2, D // 2), np.float32)
    o, lse = oracle_mod.na3d_fwd(q, k, v, coords, freqs, window)
    M = neighbour_mask(grid, window)
    assert np.array_equal(M.sum(1), np.full(N, W)) and M.sum() == N * W
    np.testing.assert_allclose(o.reshape(N, N), M / W, atol=1e-15)
    np.testing.assert_allclose(lse, math.log(W), atol=1e-14)


# ------------------------------------------------------------------ A4-A6 softmax / LSE / PV
@pytest.mark.parametrize("pairing", [0, 1])
def test_whole_grid_window_is_dense_attention(oracle_mod, pairing):
    grid = (2, 3, 4)
    q, k, v, _, coords, freqs = rand_problem(1, B=2, H=3, D=8, grid=grid)
    o, lse = oracle_mod.na3d_fwd(q, k, v, coords, freqs, grid, pairing=pairing)
    qr, kr = rope_complex(q, coords, freqs, pairing), rope_complex(k, coords, freqs, pairing)
    full = np.ones((24, 24), dtype=bool)
    o_ref, lse_ref = dense_masked_attention(flat(qr), flat(kr), flat(v), full, 1 / math.sqrt(8))
    np.testing.assert_allclose(o, o_ref.reshape(o.shape), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(lse, lse_ref.reshape(lse.shape), rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("grid,window", [((3, 4, 5), (3, 3, 3)), ((4, 6, 7), (3, 5, 5)), ((2, 5, 6), (2, 4, 3)),
                                         ((5, 3, 9), (5, 1, 7))])
def test_windowed_equals_dense_masked(oracle_mod, grid, window):
    q, k, v, _, coords, freqs = rand_problem(2, B=1, H=2, D=6, grid=grid)
    o, lse = oracle_mod.na3d_fwd(q, k, v, coords, freqs, window, scale=0.37)
    o_ref, lse_ref = reference_fwd(q, k, v, coords, freqs, grid, window, scale=0.37)
    np.testing.assert_allclose(o, o_ref, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(lse, lse_ref, rtol=1e-12, atol=1e-13)


def test_k1_window_closed_form(oracle_mod):
    """k = 1: O = V exactly, LSE_i = scale * q_i . k_i whatever the coordinates (rotations cancel)."""
    grid = (2, 3, 4)
    q, k, v, _, coords, freqs = rand_problem(3, B=1, H=2, D=8, grid=grid, coord_scale=50.0)
    o, lse = oracle_mod.na3d_fwd(q, k, v, coords, freqs, (1, 1, 1))
    np.testing.assert_allclose(o, v, rtol=0, atol=1e-15)
    want = np.einsum("blyxhd,blyxhd->bhlyx", q, k) / math.sqrt(8)
    np.testing.assert_allclose(lse, want, rtol=1e-12, atol=1e-12)


def test_dimensional_reductions(oracle_mod):
    """L = 1 is 2D NA; L = Y = 1 is 1D sliding-window attention (independent banded matrix)."""
    n, kk, D = 11, 5, 4
    rng = np.random.default_rng(4)
    q, k, v = (rng.standard_normal((1, 1, 1, n, 1, D)) for _ in range(3))
    coords = np.zeros((1, 1, 1, n, 2), np.float32)
    freqs = np.zeros((2, D // 2), np.float32)
    o, _ = oracle_mod.na3d_fwd(q, k, v, coords, freqs, (1, 1, kk))
    S = q[0, 0, 0, :, 0] @ k[0, 0, 0, :, 0].T / math.sqrt(D)
    band = np.full((n, n), -np.inf)
    for i in range(n):
        lo = min(max(i - kk // 2, 0), n - kk)
        band[i, lo:lo + kk] = 0.0
    P = np.exp(S + band - (S + band).max(1, keepdims=True))
    P /= P.sum(1, keepdims=True)
    np.testing.assert_allclose(o[0, 0, 0, :, 0], P @ v[0, 0, 0, :, 0], rtol=1e-12, atol=1e-13)
    # 2D: a (1, ky, kx) window on an (L, Y, X) grid treats every level as its own 2D problem
    grid = (3, 5, 6)
    q, k, v, _, coords, freqs = rand_problem(5, grid=grid, D=4)
    o3, l3 = oracle_mod.na3d_fwd(q, k, v, coords, freqs, (1, 3, 3))
    for lev in range(3):
        o2, l2 = oracle_mod.na3d_fwd(q[:, lev:lev + 1], k[:, lev:lev + 1], v[:, lev:lev + 1],
                                     coords[:, lev:lev + 1], freqs, (1, 3, 3))
        np.testing.assert_allclose(o3[:, lev:lev + 1], o2, rtol=1e-13, atol=1e-14)
        np.testing.assert_allclose(l3[:, :, lev:lev + 1], l2, rtol=1e-13, atol=1e-14)


# ------------------------------------------------------------------ A1-A2 StereoRoPE
def test_rope_norm_and_zero_angle(oracle_mod):
    q, _, _, _, coords, freqs = rand_problem(6, B=2, H=2, D=16, grid=(2, 3, 3), coord_scale=200.0)
    for pairing in (0, 1):
        r = oracle_mod.rope_rotate(q, coords, freqs, pairing)
        np.testing.assert_allclose(np.linalg.norm(r, axis=-1), np.linalg.norm(q, axis=-1), rtol=1e-14)
        np.testing.assert_allclose(r, rope_complex(q, coords, freqs, pairing), rtol=1e-12, atol=1e-13)
        back = oracle_mod.rope_rotate(r, coords, freqs, pairing, sign=-1.0)   # R(-phi) R(phi) = I
        np.testing.assert_allclose(back, q, rtol=1e-12, atol=1e-13)
    z = oracle_mod.rope_rotate(q, np.zeros_like(coords), freqs)
    assert np.array_equal(z, q)
    z = oracle_mod.rope_rotate(q, coords, np.zeros_like(freqs))
    assert np.array_equal(z, q)


def test_rope_integer_coords_is_axial_2d_rope(oracle_mod):
    """the coordinates replace row/column indices of axial 2D RoPE.  With integer
    (column, row) coordinates and the axial table, pair t of the first half rotates by col*theta_t
    and of the second half by row*theta_t -- ordinary axial RoPE, written with explicit 2x2 blocks."""
    B, L, Y, X, H, D = 1, 2, 4, 5, 1, 8
    rng = np.random.default_rng(7)
    x = rng.standard_normal((B, L, Y, X, H, D))
    coords = np.zeros((B, L, Y, X, 2), np.float32)
    coords[..., 0] = np.arange(X)[None, None, None, :]
    coords[..., 1] = np.arange(Y)[None, None, :, None]
    freqs = wl.make_freqs(D, 2)
    got = oracle_mod.rope_rotate(x, coords, freqs)
    theta = 100.0 ** (-np.arange(D // 4) / (D // 4))
    want = np.empty_like(x)
    for yy in range(Y):
        for xx in range(X):
            for j in range(D // 2):
                ang = (xx if j < D // 4 else yy) * float(np.float32(theta[j % (D // 4)]))
                R = np.array([[math.cos(ang), -math.sin(ang)], [math.sin(ang), math.cos(ang)]])
                want[:, :, yy, xx, :, 2 * j:2 * j + 2] = x[:, :, yy, xx, :, 2 * j:2 * j + 2] @ R.T
    np.testing.assert_allclose(got, want, rtol=1e-12, atol=1e-13)


def test_coordinate_shift_invariance(oracle_mod):
    """phi is linear in coords, so a constant shift rotates q and k alike: O and LSE unchanged."""
    grid, window = (3, 4, 5), (3, 3, 3)
    q, k, v, do, coords, freqs = rand_problem(8, grid=grid, D=8)
    # coords that stay exactly representable in float32 after the shift: quarter-integers
    coords = (np.round(coords.astype(np.float64) * 4) / 4).astype(np.float32)
    shifted = (coords.astype(np.float64) + np.array([3.0, -7.0])).astype(np.float32)
    o1, l1 = oracle_mod.na3d_fwd(q, k, v, coords, freqs, window)
    o2, l2 = oracle_mod.na3d_fwd(q, k, v, shifted, freqs, window)
    np.testing.assert_allclose(o1, o2, rtol=0, atol=1e-12)
    np.testing.assert_allclose(l1, l2, rtol=0, atol=1e-12)
    g1 = oracle_mod.na3d_bwd(q, k, v, do, coords, freqs, window)
    g2 = oracle_mod.na3d_bwd(q, k, v, do, shifted, freqs, window)
    # dv is invariant; dq, dk rotate with the shift, their norms per pair do not change
    np.testing.assert_allclose(g1[2], g2[2], rtol=0, atol=1e-12)
    np.testing.assert_allclose(np.linalg.norm(g1[0], axis=-1), np.linalg.norm(g2[0], axis=-1), atol=1e-12)


def test_three_axis_rope_variant(oracle_mod):
    grid, window = (3, 3, 4), (3, 3, 3)
    q, k, v, _, coords, freqs = rand_problem(9, grid=grid, D=12, A=3)
    o, lse = oracle_mod.na3d_fwd(q, k, v, coords, freqs, window)
    o_ref, lse_ref = reference_fwd(q, k, v, coords, freqs, grid, window)
    np.testing.assert_allclose(o, o_ref, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(lse, lse_ref, rtol=1e-12, atol=1e-13)


def test_no_rope_variant(oracle_mod):
    grid, window = (2, 3, 4), (1, 3, 3)
    q, k, v, _, coords, freqs = rand_problem(10, grid=grid, D=4)
    none_c = np.zeros((1,) + grid + (0,), np.float32)
    o, lse = oracle_mod.na3d_fwd(q, k, v, none_c, np.zeros((0, 2), np.float32), window)
    o_ref, lse_ref = reference_fwd(q, k, v, np.zeros_like(coords), freqs, grid, window)
    np.testing.assert_allclose(o, o_ref, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(lse, lse_ref, rtol=1e-12, atol=1e-13)


# ------------------------------------------------------------------ eq. (1) geometry
def test_eq1_golden_and_closed_forms(oracle_mod):
    gold = dict(l.split() for l in open(os.path.join(GOLD, "eq1_equator.txt")) if not l.startswith("#"))
    n_total = 6 * 2048 * 2048
    x, y = oracle_mod.geometry.stereo_xy(0.0, 4 * (math.pi / 2) / 2048, 0.0, 0.0, n_total)
    assert abs(float(x) - float(gold["x"])) < 1e-12 and abs(float(y)) < 1e-15
    rng = np.random.default_rng(11)
    lat0, lon0 = 0.6, -2.0
    lat = lat0 + rng.uniform(-0.3, 0.3, 200)
    lon = lon0 + rng.uniform(-0.3, 0.3, 200)
    x, y = oracle_mod.geometry.stereo_xy(lat, lon, lat0, lon0, n_total)
    ell = math.sqrt(4 * math.pi / n_total)
    hav = np.sin((lat - lat0) / 2) ** 2 + np.cos(lat0) * np.cos(lat) * np.sin((lon - lon0) / 2) ** 2
    c = 2 * np.arcsin(np.sqrt(hav))                         # haversine: independent route to c
    np.testing.assert_allclose(ell * np.hypot(x, y), 2 * np.tan(c / 2), rtol=1e-11)
    x0, y0 = oracle_mod.geometry.stereo_xy(lat0, lon0, lat0, lon0, n_total)
    assert abs(x0) < 1e-9 and abs(y0) < 1e-9                # centre maps to the origin
    xn, yn = oracle_mod.geometry.stereo_xy(lat0 + 0.1, lon0, lat0, lon0, n_total)
    assert abs(xn) < 1e-9 and yn > 0                        # due north: x = 0, y > 0
    # conformal: Jacobian wrt local metric (d lat, cos(lat) d lon) is scalar * rotation
    h = 1e-6
    for la, lo in [(0.7, -1.9), (0.45, -2.2)]:
        fx = lambda a, b: np.array(oracle_mod.geometry.stereo_xy(a, b, lat0, lon0, n_total), dtype=np.float64)
        d_north = (fx(la + h, lo) - fx(la - h, lo)) / (2 * h)
        d_east = (fx(la, lo + h) - fx(la, lo - h)) / (2 * h * math.cos(la))
        assert abs(np.dot(d_north, d_east)) < 1e-5 * np.dot(d_north, d_north)
        assert abs(np.linalg.norm(d_north) - np.linalg.norm(d_east)) < 1e-6 * np.linalg.norm(d_north)


# ------------------------------------------------------------------ backward
def _torch_grads(q, k, v, do, coords, freqs, grid, window, scale, pairing=0):
    """Second route: torch float64 autograd through the dense masked formulation."""
    tq, tk, tv = (torch.tensor(t, dtype=torch.float64, requires_grad=True) for t in (q, k, v))
    phi = torch.einsum("blyxa,aj->blyxj", torch.tensor(coords, dtype=torch.float64),
                       torch.tensor(freqs, dtype=torch.float64))
    cs, sn = torch.cos(phi)[..., None, :], torch.sin(phi)[..., None, :]

    def rot(x):
        D = x.shape[-1]
        a, b = (x[..., 0::2], x[..., 1::2]) if pairing == 0 else (x[..., :D // 2], x[..., D // 2:])
        ra, rb = a * cs - b * sn, a * sn + b * cs
        if pairing == 0:
            return torch.stack([ra, rb], dim=-1).reshape(x.shape)
        return torch.cat([ra, rb], dim=-1)

    B, L, Y, X, H, D = q.shape
    qf, kf, vf = (t.reshape(B, L * Y * X, H, D) for t in (rot(tq), rot(tk), tv))
    s = torch.einsum("bihd,bjhd->bhij", qf, kf) * scale
    mask = torch.tensor(neighbour_mask(grid, window))
    s = s.masked_fill(~mask[None, None], float("-inf"))
    o = torch.einsum("bhij,bjhd->bihd", torch.softmax(s, dim=-1), vf).reshape(q.shape)
    o.backward(torch.tensor(do, dtype=torch.float64))
    return tq.grad.numpy(), tk.grad.numpy(), tv.grad.numpy()


@pytest.mark.parametrize("grid,window,pairing", [((3, 4, 5), (3, 3, 3), 0), ((2, 5, 4), (1, 5, 3), 1),
                                                 ((4, 3, 3), (3, 3, 3), 0), ((2, 2, 6), (2, 2, 4), 0)])
def test_backward_vs_torch_autograd(oracle_mod, grid, window, pairing):
    q, k, v, do, coords, freqs = rand_problem(12, B=2, H=2, D=8, grid=grid)
    dq, dk, dv = oracle_mod.na3d_bwd(q, k, v, do, coords, freqs, window, scale=0.4, pairing=pairing)
    rq, rk, rv = _torch_grads(q, k, v, do, coords, freqs, grid, window, 0.4, pairing)
    np.testing.assert_allclose(dq, rq, rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(dk, rk, rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(dv, rv, rtol=1e-10, atol=1e-12)


def test_backward_vs_finite_differences(oracle_mod):
    grid, window = (3, 4, 5), (3, 3, 3)
    q, k, v, do, coords, freqs = rand_problem(13, B=1, H=1, D=4, grid=grid)
    dq, dk, dv = oracle_mod.na3d_bwd(q, k, v, do, coords, freqs, window)

    def loss(qq, kk, vv):
        o, _ = oracle_mod.na3d_fwd(qq, kk, vv, coords, freqs, window)
        return float((o * do).sum())

    rng = np.random.default_rng(14)
    h = 1e-5
    for which, grad in (("q", dq), ("k", dk), ("v", dv)):
        for _ in range(12):
            pos = tuple(int(rng.integers(0, s)) for s in q.shape)
            args = {"q": q.copy(), "k": k.copy(), "v": v.copy()}
            args[which][pos] += h
            up = loss(args["q"], args["k"], args["v"])
            args[which][pos] -= 2 * h
            dn = loss(args["q"], args["k"], args["v"])
            fd = (up - dn) / (2 * h)
            assert abs(fd - grad[pos]) <= 1e-7 * max(1.0, abs(fd)), (which, pos, fd, grad[pos])


def test_dv_with_unit_do_is_column_sum_of_p(oracle_mod):
    grid, window = (2, 4, 4), (1, 3, 3)
    q, k, v, _, coords, freqs = rand_problem(15, B=1, H=1, D=4, grid=grid)
    do = np.ones_like(q)
    _, _, dv = oracle_mod.na3d_bwd(q, k, v, do, coords, freqs, window)
    qr, kr = rope_complex(q, coords, freqs), rope_complex(k, coords, freqs)
    s = np.einsum("id,jd->ij", flat(qr)[0, :, 0], flat(kr)[0, :, 0]) / 2.0
    s = np.where(neighbour_mask(grid, window), s, -np.inf)
    P = np.exp(s - s.max(1, keepdims=True))
    P /= P.sum(1, keepdims=True)
    np.testing.assert_allclose(flat(dv)[0, :, 0, :], np.repeat(P.sum(0)[:, None], 4, 1), rtol=1e-12)


# ------------------------------------------------------------------ sampled entry points, dtypes
def test_row_sampled_entry_points_match_full(oracle_mod):
    w = wl.small(grid=(4, 6, 7), window=(3, 5, 3), heads=2, head_dim=8, batch=2)
    inp = wl.make_inputs(w, with_do=True)
    o, lse = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window)
    dq, dk, dv = oracle_mod.na3d_bwd(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window)
    total = w.batch * w.tokens * w.heads
    idx = np.random.default_rng(16).choice(total, size=40, replace=False)
    o_s, lse_s = oracle_mod.na3d_fwd_queries(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window, idx)
    np.testing.assert_allclose(o_s, o.reshape(total, -1)[idx], rtol=1e-13, atol=1e-14)
    lse_flat = np.transpose(lse.reshape(w.batch, w.heads, w.tokens), (0, 2, 1)).reshape(total)
    np.testing.assert_allclose(lse_s, lse_flat[idx], rtol=1e-13, atol=1e-14)
    g = oracle_mod.na3d_bwd_rows(inp["q"], inp["k"], inp["v"], inp["do"], inp["coords"], inp["freqs"], w.window, idx)
    for got, full in zip(g, (dq, dk, dv)):
        np.testing.assert_allclose(got, full.reshape(total, -1)[idx], rtol=1e-11, atol=1e-13)


def test_bf16_and_f32_inputs_are_read_exactly(oracle_mod):
    w = wl.small(grid=(2, 4, 4), window=(1, 3, 3), heads=1, head_dim=8, dtype="bf16")
    inp = wl.make_inputs(w)
    as64 = {n: wl.as_f64(inp[n], "bf16") for n in ("q", "k", "v")}
    o16, l16 = oracle_mod.na3d_fwd(inp["q"], inp["k"], inp["v"], inp["coords"], inp["freqs"], w.window)
    o64, l64 = oracle_mod.na3d_fwd(as64["q"], as64["k"], as64["v"], inp["coords"], inp["freqs"], w.window)
    assert np.array_equal(o16, o64) and np.array_equal(l16, l64)
    as32 = {n: as64[n].astype(np.float32) for n in as64}
    o32, _ = oracle_mod.na3d_fwd(as32["q"], as32["k"], as32["v"], inp["coords"], inp["freqs"], w.window)
    assert np.array_equal(o32, o64)


# ------------------------------------------------------------------ eq. (2): winds in the tile-centre frame
def test_eq2_wind_rotation_closed_forms_and_special_cases(oracle_mod):
    """PAPER.md:101-108.  The oracle builds 3D vectors and projects; the pins are (i) the component form obtained by
    multiplying out the dot products by hand, e . e0 = cos dl, n . e0 = -sin p sin dl, e . n0 = sin p0 sin dl,
    n . n0 = sin p sin p0 cos dl + cos p cos p0 (r0 is orthogonal to e0 and n0, so the radial part drops out);
    (ii) textbook special cases; (iii) what the projection removes is exactly the radial component."""
    g = oracle_mod.geometry
    rng = np.random.default_rng(5)
    lat0, lon0 = 0.37, -1.21
    lat = lat0 + rng.uniform(-0.3, 0.3, 200)
    lon = lon0 + rng.uniform(-0.3, 0.3, 200)
    u, v = rng.normal(size=200) * 20, rng.normal(size=200) * 20
    ul, vl = g.wind_to_tile_frame(u, v, lat, lon, lat0, lon0)
    dl = lon - lon0
    ul_c = u * np.cos(dl) - v * np.sin(lat) * np.sin(dl)
    vl_c = u * np.sin(lat0) * np.sin(dl) + v * (np.sin(lat) * np.sin(lat0) * np.cos(dl) + np.cos(lat) * np.cos(lat0))
    assert np.max(np.abs(ul - ul_c)) < 1e-12 and np.max(np.abs(vl - vl_c)) < 1e-12
    # at the tile centre nothing changes
    a, b = g.wind_to_tile_frame(3.0, -4.0, lat0, lon0, lat0, lon0)
    assert abs(a - 3.0) < 1e-14 and abs(b + 4.0) < 1e-14
    # same meridian: East is East; the North component is foreshortened by the cosine of the latitude difference
    a, b = g.wind_to_tile_frame(3.0, -4.0, lat0 + 0.2, lon0, lat0, lon0)
    assert abs(a - 3.0) < 1e-14 and abs(b + 4.0 * math.cos(0.2)) < 1e-14
    # centre on the equator, point on the equator: North is North, East foreshortened
    a, b = g.wind_to_tile_frame(3.0, -4.0, 0.0, 0.5, 0.0, 0.3)
    assert abs(a - 3.0 * math.cos(0.2)) < 1e-14 and abs(b + 4.0) < 1e-14
    # |v_perp|^2 = |v|^2 - (v . r0)^2: the projection removes the radial leakage and nothing else
    r0 = np.array([math.cos(lat0) * math.cos(lon0), math.cos(lat0) * math.sin(lon0), math.sin(lat0)])
    e = np.stack([-np.sin(lon), np.cos(lon), np.zeros_like(lon)], -1)
    n = np.stack([-np.sin(lat) * np.cos(lon), -np.sin(lat) * np.sin(lon), np.cos(lat)], -1)
    vec = u[:, None] * e + v[:, None] * n
    rad = vec @ r0
    assert np.max(np.abs(ul ** 2 + vl ** 2 - (u ** 2 + v ** 2 - rad ** 2))) < 1e-9


# ------------------------------------------------------------------ QK-RMSNorm + sigmoid head gate
def _ng_inputs(rng, grid=(3, 4, 5), H=2, D=8, A=2):
    B = 1
    shape = (B,) + grid + (H, D)
    q, k, v = (rng.normal(size=shape) for _ in range(3))
    gate = rng.normal(size=(B,) + grid + (H,))
    coords = rng.normal(size=(B,) + grid + (A,)).astype(np.float32) * 3
    freqs = rng.uniform(0.1, 1.0, size=(A, D // 2)).astype(np.float32)
    return q, k, v, gate, coords, freqs


def test_normgate_forward_properties(oracle_mod):
    rng = np.random.default_rng(21)
    q, k, v, gate, coords, freqs = _ng_inputs(rng)
    window = (3, 3, 3)
    o, lse, a = oracle_mod.na3d_normgate_fwd(q, k, v, gate, coords, freqs, window, eps=0.0)
    # (i) what reaches the attention has RMS 1 per (token, head) vector: same result from explicitly normalised inputs
    qn = q / np.sqrt(np.mean(q ** 2, -1, keepdims=True))
    kn = k / np.sqrt(np.mean(k ** 2, -1, keepdims=True))
    assert np.allclose(np.sqrt(np.mean(qn ** 2, -1)), 1.0, atol=1e-14)
    a2, lse2 = oracle_mod.na3d_fwd(qn, kn, v, coords, freqs, window)
    assert np.max(np.abs(a - a2)) < 1e-13 and np.max(np.abs(lse - lse2)) < 1e-13
    # (ii) RMSNorm without a learnable scale forgets the length of q and k (eps = 0): positive per-row factors change nothing
    fq = rng.uniform(0.2, 5.0, size=q.shape[:-1] + (1,))
    fk = rng.uniform(0.2, 5.0, size=k.shape[:-1] + (1,))
    o3, lse3, _ = oracle_mod.na3d_normgate_fwd(q * fq, k * fk, v, gate, coords, freqs, window, eps=0.0)
    assert np.max(np.abs(o - o3)) < 1e-12 and np.max(np.abs(lse - lse3)) < 1e-12
    # (iii) |logit| <= scale * d after the normalisation (what it is for: "bounding the logit magnitude")
    assert np.max(np.abs(lse)) <= (1.0 / math.sqrt(8)) * 8 + math.log(27) + 1e-9
    # (iv) the gate: one factor per (token, head), sigmoid(0) = 1/2, sigmoid(+40) = 1, no gate = a
    assert np.max(np.abs(o - a / (1.0 + np.exp(-gate))[..., None])) < 1e-14
    o0, _, _ = oracle_mod.na3d_normgate_fwd(q, k, v, np.zeros_like(gate), coords, freqs, window, eps=0.0)
    assert np.max(np.abs(o0 - 0.5 * a)) < 1e-14
    o1, _, _ = oracle_mod.na3d_normgate_fwd(q, k, v, np.full_like(gate, 40.0), coords, freqs, window, eps=0.0)
    on, _, _ = oracle_mod.na3d_normgate_fwd(q, k, v, None, coords, freqs, window, eps=0.0)
    assert np.max(np.abs(o1 - a)) < 1e-12 and np.max(np.abs(on - a)) == 0.0
    # (v) eps: the denominator is sqrt(mean x^2 + eps) -- a single vector by hand
    x = np.array([[[[[[3.0, 4.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0]]]]]])
    from oracle import normgate
    assert np.allclose(normgate.rmsnorm(x, 0.875)[0, 0, 0, 0, 0, :2], np.array([3.0, 4.0]) / 2.0, atol=1e-15)   # mean = 25/8, + 7/8 = 4


def test_normgate_backward_vs_finite_differences(oracle_mod):
    rng = np.random.default_rng(22)
    q, k, v, gate, coords, freqs = _ng_inputs(rng, grid=(3, 3, 4), H=1, D=4)
    window = (3, 3, 3)
    eps = 1e-3
    d_o = rng.normal(size=q.shape)
    dq, dk, dv, dg = oracle_mod.na3d_normgate_bwd(q, k, v, gate, d_o, coords, freqs, window, eps=eps)

    def loss(q_, k_, v_, g_):
        o, _, _ = oracle_mod.na3d_normgate_fwd(q_, k_, v_, g_, coords, freqs, window, eps=eps)
        return float(np.sum(o * d_o))

    h = 1e-6
    for name, x, g in (("q", q, dq), ("k", k, dk), ("v", v, dv), ("gate", gate, dg)):
        flat = x.reshape(-1)
        for idx in rng.choice(flat.size, size=12, replace=False):
            old = flat[idx]
            flat[idx] = old + h
            lp = loss(q, k, v, gate)
            flat[idx] = old - h
            lm = loss(q, k, v, gate)
            flat[idx] = old
            fd = (lp - lm) / (2 * h)
            assert abs(fd - g.reshape(-1)[idx]) <= 1e-6 * max(1.0, abs(fd)), (name, idx, fd, g.reshape(-1)[idx])
    # with eps = 0 the output does not depend on |q|: the gradient is orthogonal to q, row by row
    dq0, dk0, _, _ = oracle_mod.na3d_normgate_bwd(q, k, v, gate, d_o, coords, freqs, window, eps=0.0)
    assert np.max(np.abs(np.sum(dq0 * q, -1))) < 1e-12 and np.max(np.abs(np.sum(dk0 * k, -1))) < 1e-12


# ------------------------------------------------------------------ tile stitching, eq. (5)
def test_stitch_and_kbd_window(oracle_mod):
    st = oracle_mod.stitch
    w = st.kbd_window(32, 4.0)
    # the defining property of a Kaiser-Bessel-DERIVED window (Princen-Bradley): w[j]^2 + w[j + n/2]^2 = 1; symmetric;
    # rising over the first half; "tapers smoothly to zero at the edges"
    assert np.max(np.abs(w[:16] ** 2 + w[16:] ** 2 - 1.0)) < 1e-14
    assert np.array_equal(w, w[::-1]) and np.all(np.diff(w[:16]) > 0) and w[0] < 0.01 and abs(w[15] - 1.0) < 1e-2
    # hand value, n = 2: k = (I0(0), I0(0)) -> w = sqrt(1/2)
    assert np.allclose(st.kbd_window(2, 4.0), [math.sqrt(0.5)] * 2, atol=1e-15)
    rng = np.random.default_rng(3)
    th = tw = 16
    origins = [(0, 0), (0, 12), (12, 0), (12, 12)]                     # stride 12: tiles share a border of 4 cells
    gh = gw = 28
    field = rng.normal(size=(3, gh, gw))
    tiles = np.stack([field[:, y:y + th, x:x + tw] for y, x in origins])
    wk = st.kbd_window(16, 4.0)
    # (i) tiles cut from one field stitch back to it, whatever the (positive) window: S P = identity
    assert np.max(np.abs(st.stitch(tiles, origins, wk, wk, gh, gw) - field)) < 1e-13
    # (ii) "a 2D top-hat filter that is 1 in the interior and 0 in the halo ... reduces to simply a crop"
    noisy = tiles + rng.normal(size=tiles.shape)                        # tile outputs that disagree in the overlaps
    hat = np.zeros(16); hat[2:14] = 1.0                                 # halo of 2 on each side: interiors tile the field
    got = st.stitch(noisy, origins, hat, hat, gh, gw)
    for t, (y, x) in enumerate(origins):
        assert np.array_equal(got[:, y + 2:y + 14, x + 2:x + 14], noisy[t][:, 2:14, 2:14])
    assert np.all(got[:, :2, :] == 0.0)                                 # nobody's interior: weight 0, value 0
    # (iii) a weighted AVERAGE: between the min and max of the contributing tiles, cell by cell; by hand in one cell
    got = st.stitch(noisy, origins, wk, wk, gh, gw)
    y, x = 5, 13                                                        # covered by tiles 0 (5, 13) and 1 (5, 1)
    w0, w1 = wk[5] * wk[13], wk[5] * wk[1]
    assert abs(got[1, y, x] - (w0 * noisy[0, 1, 5, 13] + w1 * noisy[1, 1, 5, 1]) / (w0 + w1)) < 1e-14
