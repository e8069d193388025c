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
