"""Host-side input generator: determinism, bf16 bit helpers, geometry recipe vs the oracle's eq. (1)."""
import math

import numpy as np
import torch

from paper_2606_31248_b200 import workloads as wl


def test_bf16_roundtrip_matches_torch():
    x = np.random.default_rng(0).standard_normal(4096).astype(np.float32) * 3
    x[:4] = [0.0, -0.0, 1.0 + 2 ** -8, 1.0 + 3 * 2 ** -8]          # ties -> even
    bits = wl.f32_to_bf16_bits(x)
    want = torch.from_numpy(x).to(torch.bfloat16)
    assert np.array_equal(bits.view(np.int16), want.view(torch.int16).numpy())
    assert np.array_equal(wl.bf16_bits_to_f32(bits), want.float().numpy())


def test_configs_match_baseline_json():
    import json, os
    base = json.load(open(os.path.join(os.path.dirname(__file__), "..", "BASELINE.json")))
    assert len(base["configs"]) == 5
    c = [wl.config(i) for i in range(5)]
    assert (c[0].grid, c[0].window, c[0].heads, c[0].head_dim, c[0].dtype, c[0].batch) == ((4, 16, 16), (3, 5, 5), 2, 32, "f32", 1)
    assert (c[1].grid, c[1].window, c[1].heads, c[1].head_dim, c[1].batch) == ((8, 64, 64), (3, 7, 7), 8, 64, 4)
    assert (c[2].grid, c[2].window, c[2].heads, c[2].head_dim, c[2].batch) == ((8, 128, 128), (5, 9, 9), 16, 128, 2)
    assert (c[3].grid, c[3].window, c[3].heads, c[3].head_dim, c[3].batch) == ((8, 128, 128), (3, 7, 7), 8, 64, 24)
    assert c[4].backward and c[4].grid == c[1].grid and c[4].batch == 4
    # useful FLOP and compulsory bytes
    assert abs(c[1].useful_flops() / 39.46e9 - 1) < 1e-3 and abs(c[1].compulsory_bytes() / 542.1e6 - 1) < 2e-3
    assert abs(c[2].useful_flops() / 869.7e9 - 1) < 1e-3 and abs(c[3].useful_flops() / 947.0e9 - 1) < 1e-3
    assert abs(c[3].compulsory_bytes() / 13.01e9 - 1) < 2e-3 and abs(c[4].useful_flops() / 98.65e9 - 1) < 1e-3


def test_inputs_are_seeded_and_shaped():
    w = wl.small(grid=(2, 4, 5), heads=2, head_dim=8, batch=2, dtype="bf16", value_scale="rsqrt_d")
    a, b = wl.make_inputs(w, with_do=True), wl.make_inputs(w, with_do=True)
    for n in a:
        assert np.array_equal(a[n], b[n])
    assert a["q"].shape == (2, 2, 4, 5, 2, 8) and a["q"].dtype == np.uint16
    assert a["coords"].shape == (2, 2, 4, 5, 2) and a["freqs"].shape == (2, 4)
    assert not np.array_equal(a["q"], a["k"])
    std = wl.as_f64(a["q"], "bf16").std()
    assert 0.2 < std * math.sqrt(8) < 2.0
    assert np.array_equal(a["coords"][:, 0], a["coords"][:, 1])      # levels share (x, y)


def test_generator_geometry_against_oracle_eq1(oracle_mod):
    for face in range(6):
        py0, px0, ny, nx = 37, 401, 6, 9
        xy = wl.tile_coords(face, py0, px0, ny, nx, "tile")
        alpha = wl.patch_angle(px0 + np.arange(nx))
        beta = wl.patch_angle(py0 + np.arange(ny))
        A, Bt = np.meshgrid(alpha, beta, indexing="xy")
        lat, lon = wl.face_point_to_latlon(face, A, Bt)
        lat0, lon0 = wl.face_point_to_latlon(face, np.float64(wl.patch_angle(px0 + (nx - 1) / 2)),
                                             np.float64(wl.patch_angle(py0 + (ny - 1) / 2)))
        x, y = oracle_mod.geometry.stereo_xy(lat, lon, float(lat0), float(lon0), wl.N_TOTAL)
        np.testing.assert_allclose(xy[..., 0], x, rtol=1e-12, atol=1e-9)
        np.testing.assert_allclose(xy[..., 1], y, rtol=1e-12, atol=1e-9)
        # neighbouring patch tokens are about 4 native cells apart (reading 8)
        step = np.hypot(*(xy[0, 1] - xy[0, 0]))
        assert 3.0 < step < 6.5


def test_face_centre_spacing_and_rollout_placement():
    # one patch east of a face centre: 4.34 coordinate units (tests/golden/eq1_equator.txt)
    xy = wl.tile_coords(0, 255, 255, 2, 2, "tile")
    assert abs(np.hypot(*(xy[0, 1] - xy[0, 0])) - 4.3416) < 2e-3
    w = wl.config(3)
    pl = wl.tile_placements(w)
    assert len(pl) == 24 and sorted({p[0] for p in pl}) == list(range(6))
    for f in range(6):
        t = [p for p in pl if p[0] == f]
        assert len(t) == 4
        assert t[1][2] - t[0][2] == 112 and t[2][1] - t[0][1] == 112          # stride 112 -> overlap 16
        assert all(0 <= p[1] and p[1] + 128 <= 512 and 0 <= p[2] and p[2] + 128 <= 512 for p in t)


def test_default_frequency_table():
    F = wl.make_freqs(64, 2)
    assert F.shape == (2, 32)
    assert np.all(F[0, 16:] == 0) and np.all(F[1, :16] == 0)                # one axis per pair
    np.testing.assert_allclose(F[0, :16], 100.0 ** (-np.arange(16) / 16), rtol=1e-6)
    np.testing.assert_allclose(F[1, 16:], F[0, :16])
