"""ORACLE (test infrastructure only): eq. (1), restated on its own in float64.

Independent of `paper_2606_31248_b200.workloads` (which holds the input generator's copy of the
recipe); tests/test_workloads.py holds one against the other, and tests/test_oracle_pins.py pins
this one to closed forms (2 tan(c/2) radius via the haversine route, conformality, centre at 0).
"""
from __future__ import annotations

import numpy as np


def stereo_xy(lat, lon, lat0, lon0, n_total):
    """Eq. (1): cos c = sin p0 sin p + cos p0 cos p cos(l - l0); k = 2/(1 + cos c);
    x = (k/l_scale) cos p sin(l - l0); y = (k/l_scale)(cos p0 sin p - sin p0 cos p cos(l - l0));
    l_scale = sqrt(4 pi / N_total)."""
    lat = np.asarray(lat, dtype=np.float64)
    lon = np.asarray(lon, dtype=np.float64)
    ell = np.sqrt(4.0 * np.pi / float(n_total))
    cosc = np.sin(lat0) * np.sin(lat) + np.cos(lat0) * np.cos(lat) * np.cos(lon - lon0)
    kk = 2.0 / (1.0 + cosc)
    x = kk / ell * np.cos(lat) * np.sin(lon - lon0)
    y = kk / ell * (np.cos(lat0) * np.sin(lat) - np.sin(lat0) * np.cos(lat) * np.cos(lon - lon0))
    return x, y


def wind_to_tile_frame(u, v, lat, lon, lat0, lon0):
    """PAPER.md:101-108 eq. (2), step by step in float64: the 3D wind vector v = U e + V n with the local unit vectors
    (e, n) at (lat, lon); its part in the tangent plane at the tile centre, v_perp = v - (v . r0) r0; the components
    U_loc = v_perp . e0, V_loc = v_perp . n0 in the tile centre's East-North frame (e0, n0), r0 the radial unit
    vector there.  Returns (U_loc, V_loc).  Geocentric Cartesian axes: x through (lat, lon) = (0, 0), z the pole."""
    u = np.asarray(u, dtype=np.float64)
    v = np.asarray(v, dtype=np.float64)
    lat = np.asarray(lat, dtype=np.float64)
    lon = np.asarray(lon, dtype=np.float64)

    def frame(p, l):
        e = np.stack([-np.sin(l), np.cos(l), np.zeros_like(l)], axis=-1)
        n = np.stack([-np.sin(p) * np.cos(l), -np.sin(p) * np.sin(l), np.cos(p)], axis=-1)
        r = np.stack([np.cos(p) * np.cos(l), np.cos(p) * np.sin(l), np.sin(p)], axis=-1)
        return e, n, r

    e, n, _ = frame(lat, lon)
    e0, n0, r0 = frame(np.float64(lat0), np.float64(lon0))
    vec = u[..., None] * e + v[..., None] * n
    vperp = vec - np.sum(vec * r0, axis=-1, keepdims=True) * r0
    return np.sum(vperp * e0, axis=-1), np.sum(vperp * n0, axis=-1)
