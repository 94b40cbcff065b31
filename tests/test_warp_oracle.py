"""Pins of the fp64 warp oracle (row f3, Eq. 14): identity, integer shifts, exactness on linear
fields, bounds, the library routine it reduces to (scipy map_coordinates, order 1, mode nearest) and a scalar
brute force written from the textbook cell formula."""
import numpy as np
import pytest

from oracle import rfa_warp_oracle as WO
from paper_1907_05709_b200 import workloads as W

SP = (0.7, 0.9, 1.3)


def _field(shape, seed=0):
    return 37.0 + 50.0 * np.random.default_rng(seed).random(shape)


def test_zero_displacement_is_identity():
    T = _field((5, 6, 7))
    assert np.array_equal(WO.warp_temperature(T, np.zeros((3, 5, 6, 7), np.float32), 1.0, SP), T)
    assert np.array_equal(WO.warp_temperature(T, np.ones((3, 5, 6, 7), np.float32), 0.0, SP), T)


def test_integer_shift_moves_the_image_and_replicates_the_edge():
    T = _field((6, 7, 9))
    d = np.empty((3, 6, 7, 9), np.float32)
    d[0], d[1], d[2] = 2 * SP[0], -1 * SP[1], 3 * SP[2]
    out = WO.warp_temperature(T, d, 1.0, SP)
    k, j, i = np.meshgrid(np.arange(6), np.arange(7), np.arange(9), indexing="ij")
    exp = T[np.clip(k + 3, 0, 5), np.clip(j - 1, 0, 6), np.clip(i + 2, 0, 8)]
    assert np.max(np.abs(out - exp)) < 1e-5            # fp32 spacing products: positions within 1e-6 voxel
    d[0], d[1], d[2] = 2.0, -1.0, 3.0                  # exact in voxel units with unit spacing
    assert np.array_equal(WO.warp_temperature(T, d, 1.0, (1.0, 1.0, 1.0)), exp)


def test_linear_field_is_reproduced_exactly():
    nz, ny, nx = 8, 9, 10
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    T = 1.5 * i - 0.7 * j + 2.25 * k + 40.0
    d = W.breathing_field((nx, ny, nz), amp_mm=(1.0, 1.5, 2.0))
    out = WO.warp_temperature(T, d, 0.8, SP)
    px = np.clip(i + 0.8 * d[0].astype(np.float64) / SP[0], 0, nx - 1)
    py = np.clip(j + 0.8 * d[1].astype(np.float64) / SP[1], 0, ny - 1)
    pz = np.clip(k + 0.8 * d[2].astype(np.float64) / SP[2], 0, nz - 1)
    assert np.max(np.abs(out - (1.5 * px - 0.7 * py + 2.25 * pz + 40.0))) < 1e-12


def test_bounds_and_constants():
    T = _field((7, 8, 9), 3)
    d = (np.random.default_rng(4).random((3, 7, 8, 9)).astype(np.float32) - 0.5) * 20.0
    out = WO.warp_temperature(T, d, 1.0, SP)
    assert out.min() >= T.min() - 1e-12 and out.max() <= T.max() + 1e-12
    assert np.max(np.abs(WO.warp_temperature(np.full((7, 8, 9), 41.5), d, 1.0, SP) - 41.5)) < 1e-13


def test_equals_scipy_map_coordinates_order1_nearest():
    from scipy.ndimage import map_coordinates
    T = _field((9, 8, 11), 5)
    d = (np.random.default_rng(6).random((3, 9, 8, 11)).astype(np.float32) - 0.5) * 6.0
    out = WO.warp_temperature(T, d, 1.3, SP)
    k, j, i = np.meshgrid(np.arange(9), np.arange(8), np.arange(11), indexing="ij")
    coords = np.array([k + 1.3 * d[2].astype(np.float64) / SP[2], j + 1.3 * d[1].astype(np.float64) / SP[1],
                       i + 1.3 * d[0].astype(np.float64) / SP[0]])
    ref = map_coordinates(T, coords, order=1, mode="nearest")
    assert np.max(np.abs(out - ref)) < 1e-10


def test_scalar_brute_force():
    nz, ny, nx = 4, 5, 6
    T = _field((nz, ny, nx), 7)
    d = (np.random.default_rng(8).random((3, nz, ny, nx)).astype(np.float32) - 0.5) * 5.0
    out = WO.warp_temperature(T, d, 1.0, SP)
    idx = np.array([0, 17, 59, 119])
    assert np.array_equal(WO.warp_temperature(T, d, 1.0, SP, index=idx), out.ravel()[idx])
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                p = [min(max(c + float(d[a, k, j, i]) / SP[a], 0.0), n - 1.0) for a, c, n in ((0, i, nx), (1, j, ny), (2, k, nz))]
                lo = [int(np.floor(x)) for x in p]
                acc = 0.0
                for dz in (0, 1):
                    for dy in (0, 1):
                        for dx in (0, 1):
                            w = 1.0
                            for a, dd in ((0, dx), (1, dy), (2, dz)):
                                f = p[a] - lo[a]
                                w *= f if dd else 1.0 - f
                            acc += w * T[min(lo[2] + dz, nz - 1), min(lo[1] + dy, ny - 1), min(lo[0] + dx, nx - 1)]
                assert abs(acc - out[k, j, i]) < 1e-12
