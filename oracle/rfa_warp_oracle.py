"""fp64 oracle of the breathing-motion warp, Eq. 14 -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

    T(x_t) = T_ref(x_t + u^-1(x_t, t))

The temperature shown at position x_t of the moving anatomy is the reference-frame temperature looked up
through the (inverse) motion field of the current breathing phase.  On the voxel grid (SURVEY.md 8(f) row f3,
DESIGN.md R-29): the sample position of voxel v is its centre plus scale * u[v] (u in millimetres, divided by the
voxel spacing), clamped to the box of voxel centres, and T_ref is interpolated trilinearly -- the plain
definition of trilinear interpolation: the eight surrounding voxel centres weighted by the products of
(1 - a) and a along each axis, a = fractional position.

Only tests/ may import this module.  It shares nothing with the CUDA library.  Pins: tests/test_warp_oracle.py
(identity, integer shifts, exactness on linear fields, bounds, scipy.ndimage.map_coordinates, scalar brute force).
"""
from __future__ import annotations

import numpy as np


def warp_temperature(T, disp_mm, scale, spacing_mm, index=None) -> np.ndarray:
    """T: (nz, ny, nx) deg C; disp_mm: (3, nz, ny, nx) = (u_x, u_y, u_z) in mm; returns the warped image, or,
    with ``index`` (flat voxel indices), only those voxels."""
    T = np.asarray(T, dtype=np.float64)
    nz, ny, nx = T.shape
    d = np.asarray(disp_mm)
    if index is None:
        k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
        ux, uy, uz = (d[c].astype(np.float64) for c in range(3))
    else:
        idx = np.asarray(index, dtype=np.int64)
        i, j, k = idx % nx, (idx // nx) % ny, idx // (nx * ny)
        ux, uy, uz = (d[c].reshape(-1)[idx].astype(np.float64) for c in range(3))
    s = float(scale)
    # sample position in voxel units, clamped to the box of voxel centres
    px = np.clip(i + s * ux / float(spacing_mm[0]), 0.0, nx - 1.0)
    py = np.clip(j + s * uy / float(spacing_mm[1]), 0.0, ny - 1.0)
    pz = np.clip(k + s * uz / float(spacing_mm[2]), 0.0, nz - 1.0)
    i0, j0, k0 = np.floor(px).astype(np.int64), np.floor(py).astype(np.int64), np.floor(pz).astype(np.int64)
    ax, ay, az = px - i0, py - j0, pz - k0
    i1, j1, k1 = np.minimum(i0 + 1, nx - 1), np.minimum(j0 + 1, ny - 1), np.minimum(k0 + 1, nz - 1)
    out = np.zeros(px.shape, dtype=np.float64)
    for kk, wz in ((k0, 1.0 - az), (k1, az)):
        for jj, wy in ((j0, 1.0 - ay), (j1, ay)):
            for ii, wx in ((i0, 1.0 - ax), (i1, ax)):
                out += wz * wy * wx * T[kk, jj, ii]
    return out
