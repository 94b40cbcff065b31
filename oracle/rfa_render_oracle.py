"""fp64 restatement of the headless heat-zone view (row f4; Figs. 11-12) -- TEST INFRASTRUCTURE.

The paper draws the ablation zone as the 42.5 C isotherm in its VR / fluoroscopy views but gives no rendering
arithmetic; the definition is this repository's (include/rfa.h: rfa_render_zone, R-30) and is restated
here step by step in numpy, fp64:

  image plane through the volume centre c, e1 = normalise(up x dir), e2 = dir x e1 (dir normalised);
  pixel (px,py): u = (px-(W-1)/2) pixel_mm, v = (py-(H-1)/2) pixel_mm;
  samples p(m) = c + u e1 + v e2 + (-R + m step_mm) dir,  m = 0 .. floor(2R/step_mm),  R = half the volume diagonal;
  a sample counts if it lies inside the box of voxel centres; there T is interpolated trilinearly;
  tmax = max over the samples (t_blood if none), depth = m*step_mm of the first sample with T >= iso, else -1.

Returns, besides the two images, ``margin`` = min over the ray's samples of |T - iso| (the pixels whose first-hit
decision can legitimately differ in fp32 are those with a small margin).
Only tests/ may import this module; it shares nothing with the CUDA library.  Pins: tests/test_render_oracle.py.
"""
from __future__ import annotations

import numpy as np


def render_zone(T, spacing_mm, direction, up, width, height, pixel_mm, step_mm, iso_c, t_blood=37.0):
    T = np.asarray(T, dtype=np.float64)
    nz, ny, nx = T.shape
    h = np.array([float(s) for s in spacing_mm])
    n = np.array([nx, ny, nz], dtype=np.float64)
    w = np.array([float(np.float32(x)) for x in direction])
    upv = np.array([float(np.float32(x)) for x in up])
    w = w / np.sqrt(np.dot(w, w))
    e1 = np.cross(upv, w)
    e1 = e1 / np.sqrt(np.dot(e1, e1))
    e2 = np.cross(w, e1)
    c = 0.5 * n * h
    R = 0.5 * np.sqrt(np.sum((n * h) ** 2))
    pixel, step = float(np.float32(pixel_mm)), float(np.float32(step_mm))
    ns = int(np.floor(2.0 * R / step)) + 1
    px, py = np.meshgrid(np.arange(width), np.arange(height))                 # (H, W)
    u = (px - 0.5 * (width - 1)) * pixel
    v = (py - 0.5 * (height - 1)) * pixel
    o = c[None, None, :] + u[..., None] * e1 + v[..., None] * e2 - R * w      # (H, W, 3) ray starts
    tmax = np.full((height, width), -np.inf)
    depth = np.full((height, width), -1.0)
    margin = np.full((height, width), np.inf)
    iso = float(np.float32(iso_c))
    for m in range(ns):
        p = o + (m * step) * w
        q = p / h - 0.5                                                        # voxel coordinates (x, y, z)
        inside = np.all((q >= 0.0) & (q <= n - 1.0), axis=-1)
        if not inside.any():
            continue
        qi = q[inside]
        lo = np.minimum(np.floor(qi), np.maximum(n - 2.0, 0.0)).astype(np.int64)
        a = qi - lo
        hi = np.minimum(lo + 1, (n - 1).astype(np.int64))
        val = np.zeros(len(qi))
        for kz, wz in ((lo[:, 2], 1.0 - a[:, 2]), (hi[:, 2], a[:, 2])):
            for jy, wy in ((lo[:, 1], 1.0 - a[:, 1]), (hi[:, 1], a[:, 1])):
                for ix, wx in ((lo[:, 0], 1.0 - a[:, 0]), (hi[:, 0], a[:, 0])):
                    val += wz * wy * wx * T[kz, jy, ix]
        tm = tmax[inside]
        tmax[inside] = np.maximum(tm, val)
        mg = margin[inside]
        margin[inside] = np.minimum(mg, np.abs(val - iso))
        d = depth[inside]
        hit = (d < 0) & (val >= iso)
        d[hit] = m * step
        depth[inside] = d
    tmax[~np.isfinite(tmax)] = float(t_blood)
    return tmax, depth, margin
