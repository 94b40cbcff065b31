"""Pins of the fp64 view oracle (row f4): along a grid axis with samples on voxel centres it reduces to numpy's max /
argmax along that axis; for a radial field the images have closed forms (closest approach, chord entry) and do not
depend on the viewing direction."""
import numpy as np

from oracle import rfa_render_oracle as RO


def test_axis_aligned_view_reduces_to_numpy_max_and_argmax():
    rng = np.random.default_rng(2)
    nz, ny, nx = 12, 6, 4                                   # extents 4, 6, 12 mm: diagonal 14, R = 7 exactly
    T = 37.0 + 30.0 * rng.random((nz, ny, nx))
    h = (1.0, 1.0, 1.0)
    # look along +z; up = +y -> e1 = y x z = +x, e2 = z x x = +y; pixels on the voxel centres of the xy plane;
    # rays start at z = c_z - R = -1, so the samples -1 + m/2 hit every voxel centre k + 1/2 (m = 2k + 3)
    tmax, depth, _ = RO.render_zone(T, h, (0, 0, 1), (0, 1, 0), nx, ny, 1.0, 0.5, 55.0)
    assert np.max(np.abs(tmax - T.max(axis=0))) < 1e-12     # in between the centres the interpolant stays below the max
    first = np.argmax(T >= 55.0, axis=0).astype(np.float64)
    has = (T >= 55.0).any(axis=0)
    assert np.array_equal(has, depth >= 0)
    # voxel centre k is at depth k + 1.5 mm; the interpolant may cross the isotherm up to two half-steps earlier
    z_first = first + 1.5
    assert np.all(depth[has] <= z_first[has] + 1e-12) and np.all(depth[has] >= z_first[has] - 0.5 - 1e-12)
    # a column that is hot from the first voxel on is hit exactly at that voxel's centre or the sample before it
    T2 = T.copy()
    T2[:, 2, 1] = 70.0
    _, d2, _ = RO.render_zone(T2, h, (0, 0, 1), (0, 1, 0), nx, ny, 1.0, 0.5, 55.0)
    assert d2[2, 1] == 1.5                                  # sample m = 3 (z = 0.5, centre of voxel 0): first inside sample


def _radial(n, h, f):
    k, j, i = np.meshgrid(*(np.arange(n),) * 3, indexing="ij")
    c = 0.5 * n * h
    r = np.sqrt(((i + 0.5) * h - c) ** 2 + ((j + 0.5) * h - c) ** 2 + ((k + 0.5) * h - c) ** 2)
    return f(r)


def test_radial_field_closed_forms_and_direction_independence():
    n, h = 64, 0.5
    f = lambda r: 37.0 + 53.0 * np.exp(-(r / 6.0) ** 2)      # smooth hot ball, 90 C at the centre
    T = _radial(n, h, f)
    W = 33
    views = [((0, 0, 1), (0, 1, 0)), ((1, 0, 0), (0, 0, 1)), ((1, 2, 3), (0, 1, 0)), ((-2, 1, 0.5), (0, 0, 1))]
    imgs = [RO.render_zone(T, (h, h, h), d, up, W, W, 0.5, 0.125, 42.5) for d, up in views]
    px = (np.arange(W) - 0.5 * (W - 1)) * 0.5
    b = np.sqrt(px[None, :] ** 2 + px[:, None] ** 2)         # impact parameter of the pixel's ray
    # tmax = f(closest approach) up to the trilinear interpolation error: 3 axes * h^2/8 * |f''|max = 3 * 0.25/8 * 2.94 = 0.28
    for tmax, depth, _ in imgs:
        assert np.max(np.abs(tmax - f(b))) < 0.3
    # isotherm radius r0: f(r0) = 42.5; the ray enters the ball at -sqrt(r0^2 - b^2) from the centre plane
    r0 = 6.0 * np.sqrt(np.log(53.0 / 5.5))
    R = 0.5 * np.sqrt(3.0) * n * h
    inside = b < r0 - 0.3
    for tmax, depth, _ in imgs:
        assert np.all(depth[inside] >= 0) and np.all(depth[b > r0 + 0.3] < 0)
        entry = R - np.sqrt(r0 ** 2 - b[inside] ** 2)
        assert np.max(np.abs(depth[inside] - entry)) < 0.125 + 0.15    # one step + interpolation error
    # the image of a radial field does not depend on the direction
    for tmax, depth, _ in imgs[1:]:
        assert np.max(np.abs(tmax - imgs[0][0])) < 0.3


def test_empty_rays_and_margin():
    T = np.full((4, 4, 4), 40.0)
    tmax, depth, margin = RO.render_zone(T, (1, 1, 1), (0, 0, 1), (0, 1, 0), 12, 12, 1.0, 0.5, 42.5)
    assert tmax[0, 0] == 37.0 and depth[0, 0] == -1.0 and np.isinf(margin[0, 0])      # the ray misses the volume
    assert abs(tmax[6, 6] - 40.0) < 1e-12 and depth[6, 6] == -1.0 and abs(margin[6, 6] - 2.5) < 1e-12


def test_linear_field_oblique_view_is_exact():
    """Trilinear interpolation reproduces a linear field exactly, so for T = T0 + g . x the images of an OBLIQUE view have
    closed forms to rounding: along a ray T is linear in the sample index m, tmax is its value at the last (or first)
    sample inside the box of voxel centres, and the first sample with T >= iso solves one linear inequality.  The inside
    range of m is computed here by testing every sample against the box (no slab formula shared with anything).
    Catches swapped axes, wrong spacing, transposed weights and an off-by-half in the voxel-centre convention."""
    nx, ny, nz = 14, 11, 9
    h = np.array([0.7, 0.9, 1.3])
    g = np.array([1.9, -0.8, 1.1])                          # deg C per mm
    T0 = 40.0
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    T = T0 + g[0] * (i + 0.5) * h[0] + g[1] * (j + 0.5) * h[1] + g[2] * (k + 0.5) * h[2]
    direction, up = np.array([1.0, 2.0, 3.0]), np.array([0.0, 1.0, 0.0])
    W_, H_, pixel, step, iso = 9, 7, 0.75, 0.25, 52.0        # exactly representable in fp32 (the API takes floats)
    tmax, depth, _ = RO.render_zone(T, tuple(h), tuple(direction), tuple(up), W_, H_, pixel, step, iso)
    w = direction / np.linalg.norm(direction)
    e1 = np.cross(up, w)
    e1 /= np.linalg.norm(e1)
    e2 = np.cross(w, e1)
    n = np.array([nx, ny, nz], dtype=np.float64)
    c, R = 0.5 * n * h, 0.5 * np.sqrt(np.sum((n * h) ** 2))
    ns = int(np.floor(2.0 * R / step)) + 1
    m = np.arange(ns)
    seen_inside = 0
    for py in range(H_):
        for px in range(W_):
            o = c + (px - 0.5 * (W_ - 1)) * pixel * e1 + (py - 0.5 * (H_ - 1)) * pixel * e2 - R * w
            p = o[None, :] + (m * step)[:, None] * w[None, :]          # sample positions in mm
            q = p / h - 0.5
            inside = np.all((q >= 0.0) & (q <= n - 1.0), axis=1)
            if not inside.any():
                assert tmax[py, px] == 37.0 and depth[py, px] == -1.0
                continue
            seen_inside += 1
            Tm = T0 + p[inside] @ g                                  # the field itself at the samples that count
            assert abs(tmax[py, px] - Tm.max()) < 1e-9
            hit = np.nonzero(Tm >= iso)[0]
            if hit.size:
                assert depth[py, px] == m[inside][hit[0]] * step
            else:
                assert depth[py, px] == -1.0
    assert seen_inside > 20
