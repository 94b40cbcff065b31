"""Seeded synthetic inputs for the RFA bioheat hot path (BASELINE.json configs C1..C5).

This module is *data only*: label volumes, tissue-constant tables, needle voxel masks and
initial fields.  It holds none of the method's arithmetic (no stencil, no Euler update, no
necrosis test), so both the fp64 oracle (``oracle/``) and the CUDA library may take their inputs
from it without sharing any computation.

The phantoms stand in for the paper's segmented CT "virtual body models" (PAPER.md:45, :139 --
256^2 x 234 voxels at 1.552^2 x 2 mm, and the 0.5 mm evaluation grid of PAPER.md:145), which are
not available.  The recipe is SURVEY.md section 8(d); DESIGN.md section 4 restates it.

Conventions: volumes are numpy arrays of shape (nz, ny, nx), x fastest (idx = i + nx*(j + ny*k));
voxel (i, j, k) has its centre at ((i+0.5)*dx, (j+0.5)*dy, (k+0.5)*dz) millimetres.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# ----------------------------------------------------------------------------------------------
# Tissue table.  One row per label id:  k [W/(m K)], rho [kg/m^3], cp [J/(kg K)],
# wb_cb [W/(m^3 K)] (= w_b*c_b of PAPER.md:102 Eq. 9), q_m [W/m^3], t_init [deg C], flags.
# ----------------------------------------------------------------------------------------------
TISSUE_DTYPE = np.dtype(
    [("k", "<f4"), ("rho", "<f4"), ("cp", "<f4"), ("wb_cb", "<f4"), ("q_m", "<f4"),
     ("t_init", "<f4"), ("flags", "<u4")],
    align=False,
)
TISSUE_HELD = 1  # never updated, stays at t_init (vessel, exterior) -- PAPER.md:122-125, Alg. 1 :306

SRC_OFF, SRC_DIRICHLET, SRC_POWER = 0, 1, 2

# Blood constants used to turn a perfusion rate omega_b [1/s] into wb_cb:
RHO_BLOOD = 1050.0   # kg/m^3 (the paper names a blood density at PAPER.md:104 but gives no value)
C_BLOOD = 3617.0     # J/(kg K)
T_BLOOD = 37.0       # deg C

FAT, LIVER, TUMOUR, VESSEL, SPLEEN, KIDNEY, EXTERIOR = range(7)


def _row(k, rho, cp, omega_b, q_m=0.0, t_init=T_BLOOD, flags=0):
    return (k, rho, cp, omega_b * RHO_BLOOD * C_BLOOD, q_m, t_init, flags)


def tissue_table() -> np.ndarray:
    """The 7-label table used by C1..C5 (BASELINE.json configs; spleen/kidney: SURVEY.md G-25)."""
    rows = [
        _row(0.21, 911.0, 2348.0, 0.0005),                 # 0 fat
        _row(0.512, 1060.0, 3600.0, 6.4e-3),               # 1 liver
        _row(0.512, 1060.0, 3600.0, 0.01),                 # 2 tumour (liver params, w_b = 0.01)
        _row(0.512, 1060.0, 3600.0, 0.0, flags=TISSUE_HELD),   # 3 vessel: fixed 37 C heat sink
        _row(0.53, 1050.0, 3700.0, 0.02),                  # 4 spleen (stand-in, G-25)
        _row(0.53, 1050.0, 3700.0, 0.07),                  # 5 kidney (w_b = 0.07)
        _row(0.21, 911.0, 2348.0, 0.0, flags=TISSUE_HELD),     # 6 exterior: held at 37 C
    ]
    return np.array(rows, dtype=TISSUE_DTYPE)


def paper_liver_table() -> np.ndarray:
    """Single-label table with the constants printed at PAPER.md:104 (incl. Q_m = 10714 W/m^3)."""
    return np.array([(0.52, 1079.0, 3540.0, 16.687 * 3617.0, 10714.0, T_BLOOD, 0)], dtype=TISSUE_DTYPE)


def make_table(rows) -> np.ndarray:
    """rows: iterable of (k, rho, cp, wb_cb, q_m, t_init, flags)."""
    return np.array([tuple(r) for r in rows], dtype=TISSUE_DTYPE)


# ----------------------------------------------------------------------------------------------
@dataclass
class Needle:
    mask: np.ndarray            # uint8 (nz, ny, nx), nonzero = electrode voxel
    mode: int                   # SRC_DIRICHLET / SRC_POWER
    value: float                # deg C or W/m^3
    tip_mm: tuple = (0.0, 0.0, 0.0)
    axis: tuple = (0.0, 0.0, 1.0)


@dataclass
class Workload:
    name: str
    dims: tuple                 # (nx, ny, nz)
    spacing_mm: tuple           # (dx, dy, dz)
    labels: np.ndarray          # uint8 (nz, ny, nx)
    table: np.ndarray           # TISSUE_DTYPE rows
    dt: float
    steps: int
    needles: list = field(default_factory=list)    # one Needle per scenario
    t_blood: float = T_BLOOD
    t0: np.ndarray | None = None                   # optional explicit initial field (deg C), float64
    meta: dict = field(default_factory=dict)

    @property
    def batch(self) -> int:
        return max(1, len(self.needles))

    @property
    def n_voxels(self) -> int:
        return int(self.dims[0]) * int(self.dims[1]) * int(self.dims[2])


def _rng(c: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(190705709 + 1000 * c))


def _axes_mm(dims, spacing):
    nx, ny, nz = dims
    x = (np.arange(nx, dtype=np.float64) + 0.5) * spacing[0]
    y = (np.arange(ny, dtype=np.float64) + 0.5) * spacing[1]
    z = (np.arange(nz, dtype=np.float64) + 0.5) * spacing[2]
    return x, y, z


def _unit(v):
    v = np.asarray(v, dtype=np.float64)
    return v / np.linalg.norm(v)


def _uniform_sphere(rng) -> np.ndarray:
    return _unit(rng.normal(size=3))


def _bbox(dims, spacing, lo_mm, hi_mm):
    """Index slices (z, y, x) covering the axis-aligned box [lo_mm, hi_mm] (clipped to the grid)."""
    sl = []
    for a in (2, 1, 0):
        n = dims[a]
        i0 = int(np.floor(lo_mm[a] / spacing[a] - 0.5))
        i1 = int(np.ceil(hi_mm[a] / spacing[a] - 0.5)) + 1
        sl.append(slice(max(0, i0), min(n, max(i1, 0))))
    return tuple(sl)


def _segment_sub(dims, spacing, p0_mm, p1_mm, radius_mm):
    """(slices, bool sub-volume) of voxels whose centre lies within ``radius_mm`` of segment p0-p1,
    evaluated in fp64 inside the capsule's bounding box only; None if the box misses the grid."""
    p0 = np.asarray(p0_mm, dtype=np.float64)
    p1 = np.asarray(p1_mm, dtype=np.float64)
    lo = np.minimum(p0, p1) - radius_mm
    hi = np.maximum(p0, p1) + radius_mm
    sz, sy, sx = _bbox(dims, spacing, lo, hi)
    if sz.start >= sz.stop or sy.start >= sy.stop or sx.start >= sx.stop:
        return None
    x, y, z = _axes_mm(dims, spacing)
    X = x[sx][None, None, :]
    Y = y[sy][None, :, None]
    Z = z[sz][:, None, None]
    d = p1 - p0
    dd = float(d @ d)
    if dd == 0.0:
        dist2 = (X - p0[0]) ** 2 + (Y - p0[1]) ** 2 + (Z - p0[2]) ** 2
    else:
        t = ((X - p0[0]) * d[0] + (Y - p0[1]) * d[1] + (Z - p0[2]) * d[2]) / dd
        t = np.clip(t, 0.0, 1.0)
        dist2 = (X - (p0[0] + t * d[0])) ** 2 + (Y - (p0[1] + t * d[1])) ** 2 + (Z - (p0[2] + t * d[2])) ** 2
    return (sz, sy, sx), dist2 <= radius_mm * radius_mm


def segment_mask(dims, spacing, p0_mm, p1_mm, radius_mm, out=None, value=1) -> np.ndarray:
    """Voxels whose centre lies within ``radius_mm`` of the segment p0-p1 (a capsule).
    Returns/updates a uint8 (nz, ny, nx) volume."""
    nx, ny, nz = dims
    if out is None:
        out = np.zeros((nz, ny, nx), dtype=np.uint8)
    r = _segment_sub(dims, spacing, p0_mm, p1_mm, radius_mm)
    if r is not None:
        sl, m = r
        out[sl][m] = value
    return out


def ellipsoid_mask(dims, spacing, centre_mm, semi_mm) -> tuple:
    """Returns (slices, bool sub-volume) of voxels whose centre lies inside the ellipsoid."""
    c = np.asarray(centre_mm, dtype=np.float64)
    s = np.asarray(semi_mm, dtype=np.float64)
    sz, sy, sx = _bbox(dims, spacing, c - s, c + s)
    x, y, z = _axes_mm(dims, spacing)
    X = ((x[sx] - c[0]) / s[0])[None, None, :]
    Y = ((y[sy] - c[1]) / s[1])[None, :, None]
    Z = ((z[sz] - c[2]) / s[2])[:, None, None]
    return (sz, sy, sx), (X * X + Y * Y + Z * Z) <= 1.0


def _paint_ellipsoid(labels, dims, spacing, centre_mm, semi_mm, value, only_where=None):
    sl, m = ellipsoid_mask(dims, spacing, centre_mm, semi_mm)
    sub = labels[sl]
    if only_where is not None:
        m = m & np.isin(sub, only_where)
    sub[m] = value


def _paint_cylinder(labels, dims, spacing, p0, p1, r, value, only_where=None):
    res = _segment_sub(dims, spacing, p0, p1, r)
    if res is None:
        return
    sl, m = res
    sub = labels[sl]
    if only_where is not None:
        m = m & np.isin(sub, only_where)
    sub[m] = value


# ----------------------------------------------------------------------------------------------
# C1: homogeneous liver cube (BASELINE.json configs[0])
# ----------------------------------------------------------------------------------------------
def c1_cube(n: int = 64, steps: int = 100) -> Workload:
    dims = (n, n, n)
    labels = np.full((n, n, n), LIVER, dtype=np.uint8)
    mask = np.zeros((n, n, n), dtype=np.uint8)
    c = n // 2
    mask[c, c, c] = 1
    tip = tuple((c + 0.5) * 1.0 for _ in range(3))
    return Workload("C1", dims, (1.0, 1.0, 1.0), labels, tissue_table(), 0.1, steps,
                    [Needle(mask, SRC_DIRICHLET, 90.0, tip, (0.0, 0.0, 1.0))])


def c1_green(n: int = 64, h_mm: float = 1.0, dt: float = 0.1, steps: int = 1000,
             energy: float = 1.0e4) -> Workload:
    """C1-G: perfusion = 0, no needle, T0 = 37 + energy*delta at the centre voxel (Eq. 2 check)."""
    dims = (n, n, n)
    labels = np.zeros((n, n, n), dtype=np.uint8)
    table = make_table([(0.512, 1060.0, 3600.0, 0.0, 0.0, T_BLOOD, 0)])
    t0 = np.full((n, n, n), T_BLOOD, dtype=np.float64)
    c = n // 2
    t0[c, c, c] += energy
    return Workload("C1-G", dims, (h_mm,) * 3, labels, table, dt, steps, [], t0=t0,
                    meta={"centre": (c, c, c), "energy": energy})


# ----------------------------------------------------------------------------------------------
# C2 / C3: block phantoms in a 128 mm cube (BASELINE.json configs[1], [2])
# ----------------------------------------------------------------------------------------------
def fig6_probes(dims, spacing, centre_voxel, dists_mm=(2.5, 5.0)) -> np.ndarray:
    """Flat voxel indices of the symmetric probe sets of PAPER.md:147 / Fig. 6: for each distance the six
    points at +-d along x, y, z from the tip voxel (rounded to voxel centres).  Shape (len(dists), 6)."""
    nx, ny, nz = dims
    ci, cj, ck = centre_voxel
    out = []
    for d in dists_mm:
        row = []
        for a in range(3):
            for sgn in (-1, 1):
                o = [0, 0, 0]
                o[a] = sgn * int(round(d / spacing[a]))
                i, j, k = ci + o[0], cj + o[1], ck + o[2]
                assert 0 <= i < nx and 0 <= j < ny and 0 <= k < nz, "probe outside the grid"
                row.append(i + nx * (j + ny * k))
        out.append(row)
    return np.array(out, dtype=np.int64)


def paper_probe_case(tip_c: float = 90.0, n: int = 64, steps: int = 1200) -> Workload:
    """The paper's evaluation set-up: 0.5 mm grid, liver constants of :104 (with
    Q_m), a 2.5 mm hemispherical tip (5 x 5 x 3 voxels) held at 90 or 60 C, dt = 0.1 s, 120 s."""
    h = 0.5
    labels = np.zeros((n, n, n), np.uint8)
    c = n // 2
    mask = np.zeros((n, n, n), np.uint8)
    for dz in range(0, 3):
        for dy in range(-2, 3):
            for dx in range(-2, 3):
                if (dx * dx + dy * dy + dz * dz) * h * h <= 1.25 * 1.25 + 1e-9:
                    mask[c + dz, c + dy, c + dx] = 1
    nd = Needle(mask=mask, mode=SRC_DIRICHLET, value=float(tip_c),
                tip_mm=((c + 0.5) * h, (c + 0.5) * h, (c + 0.5) * h), axis=(0.0, 0.0, 1.0))
    return Workload(name=f"paper_probe_{int(tip_c)}", dims=(n, n, n), spacing_mm=(h, h, h), labels=labels,
                    table=paper_liver_table(), dt=0.1, steps=steps, needles=[nd],
                    meta={"centre_voxel": (c, c, c)})


def _block_phantom(c: int, n: int, h: float, n_tumours: int, n_vessels: int):
    rng = _rng(c)
    dims = (n, n, n)
    spacing = (h, h, h)
    labels = np.full((n, n, n), FAT, dtype=np.uint8)
    # liver box [16,112)^2 x [24,104) mm
    lo = np.array([16.0, 16.0, 24.0])
    hi = np.array([112.0, 112.0, 104.0])
    sz, sy, sx = _bbox(dims, spacing, lo + 0.5 * h, hi - 0.5 * h)
    labels[sz, sy, sx] = LIVER
    third = (hi - lo) / 3.0
    tumours = []
    for _ in range(n_tumours):
        r = rng.uniform(8.0, 15.0)
        ctr = lo + third + rng.uniform(0.0, 1.0, size=3) * third
        tumours.append((ctr, r))
    vessels = []
    for _ in range(n_vessels):
        r = rng.uniform(2.0, 4.0)
        p = lo + rng.uniform(0.0, 1.0, size=3) * (hi - lo)
        d = _uniform_sphere(rng)
        vessels.append((p - 200.0 * d, p + 200.0 * d, r))
    for ctr, r in tumours:
        _paint_ellipsoid(labels, dims, spacing, ctr, (r, r, r), TUMOUR, only_where=[LIVER])
    for p0, p1, r in vessels:                                   # clipped to the liver box
        _paint_cylinder(labels, dims, spacing, p0, p1, r, VESSEL, only_where=[LIVER, TUMOUR])
    return rng, dims, spacing, labels, tumours, vessels


def c2_phantom(steps: int = 6000) -> Workload:
    rng, dims, spacing, labels, tumours, vessels = _block_phantom(2, 128, 1.0, 1, 3)
    ctr, r = tumours[0]
    axis = _uniform_sphere(rng)
    p0, p1 = ctr - 10.0 * axis, ctr + 10.0 * axis               # 20 mm electrode centred on tumour
    mask = segment_mask(dims, spacing, p0, p1, 1.0)
    return Workload("C2", dims, spacing, labels, tissue_table(), 0.1, steps,
                    [Needle(mask, SRC_DIRICHLET, 90.0, tuple(p1), tuple(axis))],
                    meta={"tumours": tumours, "vessels": vessels})


def umbrella_mask(dims, spacing, hub_mm, axis, n_tines=9, tine_len=15.0, R=10.0, shaft_len=10.0,
                  r_e=0.75) -> np.ndarray:
    """Multi-tine umbrella electrode: a shaft behind the hub plus ``n_tines`` circular arcs
    hub + R sin(s/R) a + R (1 - cos(s/R)) e_r(phi_i), s in [0, tine_len]."""
    a = _unit(axis)
    ref = np.array([1.0, 0.0, 0.0]) if abs(a[0]) < 0.9 else np.array([0.0, 1.0, 0.0])
    e1 = _unit(np.cross(a, ref))
    e2 = np.cross(a, e1)
    hub = np.asarray(hub_mm, dtype=np.float64)
    out = segment_mask(dims, spacing, hub - shaft_len * a, hub, r_e)
    nseg = 30
    for i in range(n_tines):
        phi = 2.0 * np.pi * i / n_tines
        er = np.cos(phi) * e1 + np.sin(phi) * e2
        s = np.linspace(0.0, tine_len, nseg + 1)
        pts = hub[None, :] + (R * np.sin(s / R))[:, None] * a[None, :] + (R * (1 - np.cos(s / R)))[:, None] * er[None, :]
        for q0, q1 in zip(pts[:-1], pts[1:]):
            segment_mask(dims, spacing, q0, q1, r_e, out=out)
    return out


def c3_phantom(steps: int = 24000, n: int = 256) -> Workload:
    h = 128.0 / n
    rng, dims, spacing, labels, tumours, vessels = _block_phantom(3, n, h, 2, 6)
    ctr, _ = tumours[0]
    axis = _uniform_sphere(rng)
    mask = umbrella_mask(dims, spacing, ctr, axis, r_e=1.5 * h)   # G-26: 0.75 mm at 0.5 mm voxels
    return Workload("C3", dims, spacing, labels, tissue_table(), 0.025, steps,
                    [Needle(mask, SRC_POWER, 5.0e7, tuple(ctr), tuple(axis))],
                    meta={"tumours": tumours, "vessels": vessels})


# ----------------------------------------------------------------------------------------------
# C4: CT-sized body model 512 x 512 x 256 at 0.7 x 0.7 x 1.0 mm (BASELINE.json configs[3])
# ----------------------------------------------------------------------------------------------
def c4_body(steps: int = 12000, dims=(512, 512, 256), spacing=(0.7, 0.7, 1.0)) -> Workload:
    rng = _rng(4)
    nx, ny, nz = dims
    ext = np.array([nx * spacing[0], ny * spacing[1], nz * spacing[2]])
    g = 0.5 * ext
    sc = ext / np.array([358.4, 358.4, 256.0])     # lets tests build a geometrically similar mini body
    labels = np.full((nz, ny, nx), EXTERIOR, dtype=np.uint8)
    _paint_ellipsoid(labels, dims, spacing, g, np.array([165.0, 115.0, 125.0]) * sc, FAT)
    liver_semi = np.array([70.0, 55.0, 60.0]) * rng.uniform(0.9, 1.1, size=3) * sc
    liver_c = g + np.array([-60.0, -10.0, 10.0]) * sc
    _paint_ellipsoid(labels, dims, spacing, liver_c, liver_semi, LIVER, only_where=[FAT])
    _paint_ellipsoid(labels, dims, spacing, g + np.array([95.0, 20.0, 15.0]) * sc,
                     np.array([30.0, 25.0, 45.0]) * sc, SPLEEN, only_where=[FAT])
    for sgn in (-1.0, 1.0):
        _paint_ellipsoid(labels, dims, spacing, g + np.array([sgn * 55.0, 45.0, -40.0]) * sc,
                         np.array([22.0, 18.0, 40.0]) * sc, KIDNEY, only_where=[FAT])
    # tumours: spheres fully inside the liver
    smin = float(sc.min())
    tumours = []
    while len(tumours) < 3:
        r = rng.uniform(8.0, 15.0) * smin
        u = rng.uniform(-1.0, 1.0, size=3)
        if u @ u > 1.0:
            continue
        ctr = liver_c + u * (liver_semi - r - 2.0 * smin) * 0.9
        if all(np.linalg.norm(ctr - c2) > r + r2 + 2.0 * smin for c2, r2 in tumours):
            tumours.append((ctr, r))
    for ctr, r in tumours:
        _paint_ellipsoid(labels, dims, spacing, ctr, (r, r, r), TUMOUR, only_where=[LIVER])
    # vessel tree: 40 cylinders grown from the hilum, clipped to the liver (and tumours)
    hilum = liver_c + np.array([0.35, 0.0, -0.2]) * liver_semi
    segs = []
    frontier = [(hilum, _unit(liver_c - hilum + 1e-9), 6.0 * smin)]
    while len(segs) < 40 and frontier:
        p, d, r = frontier.pop(0)
        length = rng.uniform(20.0, 50.0) * smin
        q = p + length * d
        segs.append((p, q, r))
        for _ in range(2):
            ang = np.deg2rad(rng.uniform(25.0, 50.0))
            perp = _unit(np.cross(d, _uniform_sphere(rng)))
            nd = _unit(np.cos(ang) * d + np.sin(ang) * perp)
            frontier.append((q, nd, max(r * 0.75, 0.8 * min(spacing))))
    for p, q, r in segs:
        _paint_cylinder(labels, dims, spacing, p, q, r, VESSEL, only_where=[LIVER, TUMOUR])
    ctr, r = tumours[0]
    axis = _uniform_sphere(rng)
    half = 15.0 * smin
    p0, p1 = ctr - half * axis, ctr + half * axis
    mask = segment_mask(dims, spacing, p0, p1, max(1.0 * smin, 0.75 * max(spacing[0], spacing[1])))
    return Workload("C4", tuple(dims), tuple(spacing), labels, tissue_table(), 0.05, steps,
                    [Needle(mask, SRC_DIRICHLET, 90.0, tuple(p1), tuple(axis))],
                    meta={"tumours": tumours, "n_vessel_segments": len(segs)})


# ----------------------------------------------------------------------------------------------
# C5: planning sweep, 64 scenarios on the C2 label volume (BASELINE.json configs[4], G-24)
# ----------------------------------------------------------------------------------------------
def c5_sweep(batch: int = 64, steps: int = 3000) -> Workload:
    base = c2_phantom()
    rng = _rng(5)
    ctr, r_t = base.meta["tumours"][0]
    needles = []
    for _ in range(batch):
        while True:
            u = rng.uniform(-1.0, 1.0, size=3)
            if u @ u <= 1.0:
                break
        tip = ctr + max(r_t - 2.0, 0.0) * u
        axis = _uniform_sphere(rng)
        mask = segment_mask(base.dims, base.spacing_mm, tip - 20.0 * axis, tip, 1.0)
        needles.append(Needle(mask, SRC_DIRICHLET, 90.0, tuple(tip), tuple(axis)))
    return Workload("C5", base.dims, base.spacing_mm, base.labels, base.table, 0.1, steps, needles,
                    meta=dict(base.meta))


# ----------------------------------------------------------------------------------------------
# Small ragged cases for parity tests: sizes that span several tiles and leave ragged tails.
# ----------------------------------------------------------------------------------------------
def ragged_phantom(dims=(45, 38, 29), spacing=(0.7, 0.9, 1.3), seed: int = 7, dt: float = 0.05,
                   steps: int = 40, mode: int = SRC_DIRICHLET, value: float = 90.0,
                   batch: int = 1, q_m: float = 0.0) -> Workload:
    """Random blobs of all seven labels on a non-cubic anisotropic grid, with a needle per scenario."""
    rng = np.random.Generator(np.random.PCG64(190705709 + seed))
    nx, ny, nz = dims
    ext = np.array([nx * spacing[0], ny * spacing[1], nz * spacing[2]])
    labels = np.full((nz, ny, nx), FAT, dtype=np.uint8)
    for lab in (LIVER, SPLEEN, KIDNEY, TUMOUR, EXTERIOR):
        for _ in range(2):
            c = rng.uniform(0.0, 1.0, size=3) * ext
            s = rng.uniform(0.12, 0.4, size=3) * ext
            _paint_ellipsoid(labels, dims, spacing, c, s, lab)
    for _ in range(3):
        p = rng.uniform(0.0, 1.0, size=3) * ext
        d = _uniform_sphere(rng)
        _paint_cylinder(labels, dims, spacing, p - 300 * d, p + 300 * d, rng.uniform(1.0, 2.5), VESSEL)
    table = tissue_table()
    if q_m:
        table["q_m"][[LIVER, TUMOUR]] = q_m
    needles = []
    for _ in range(batch):
        c = (0.25 + 0.5 * rng.uniform(0.0, 1.0, size=3)) * ext
        a = _uniform_sphere(rng)
        L = 0.25 * float(ext.min())
        mask = segment_mask(dims, spacing, c - L * a, c + L * a, 1.1 * max(spacing))
        needles.append(Needle(mask, mode, value, tuple(c + L * a), tuple(a)))
    return Workload(f"ragged{dims}", tuple(dims), tuple(spacing), labels, table, dt, steps, needles)


def breathing_field(dims, amp_mm=(2.0, 4.0, 12.0)) -> np.ndarray:
    """Synthetic smooth displacement field (3, nz, ny, nx) in mm standing in for the paper's 4D-CT motion fields
    (not available): mostly cranio-caudal (z), strongest mid-volume, vanishing at the z ends, varying
    smoothly across x and y.  Scaled by the breathing amplitude of the phase by the caller."""
    nx, ny, nz = dims
    sz = np.sin(np.pi * (np.arange(nz, dtype=np.float32) + 0.5) / nz)[:, None, None]
    cy = (0.6 + 0.4 * np.cos(2.0 * np.pi * (np.arange(ny, dtype=np.float32) + 0.5) / ny))[None, :, None]
    sx = (0.8 + 0.2 * np.sin(2.0 * np.pi * (np.arange(nx, dtype=np.float32) + 0.5) / nx))[None, None, :]
    base = (sz * cy * sx).astype(np.float32)
    out = np.empty((3, nz, ny, nx), np.float32)
    out[0] = amp_mm[0] * base * np.cos(np.pi * (np.arange(ny, dtype=np.float32) + 0.5) / ny)[None, :, None]
    out[1] = -amp_mm[1] * base
    out[2] = amp_mm[2] * base
    return out


def with_smooth_field(w: Workload, amp_c: float = 8.0, periods=(64.0, 48.0, 32.0)) -> Workload:
    """Gives workload w a smooth non-uniform initial temperature 37 + amp cos cos cos (deg C; periods in voxels
    along x, y, z), so that every voxel of the volume changes from the first step on (held labels keep what is
    written): the field-wide full-size parity cases, where a uniform 37 C far field would hide tile seams."""
    nx, ny, nz = w.dims
    cx = np.cos(2.0 * np.pi * (np.arange(nx) + 0.5) / periods[0])
    cy = np.cos(2.0 * np.pi * (np.arange(ny) + 0.5) / periods[1])
    cz = np.cos(2.0 * np.pi * (np.arange(nz) + 0.5) / periods[2])
    w.t0 = 37.0 + amp_c * cz[:, None, None] * cy[None, :, None] * cx[None, None, :]
    return w


def c4_face_case(steps: int = 400) -> Workload:
    """C4 body model with a smooth non-uniform initial temperature (37 + 8 cos cos cos, deg C), so that heat
    crosses every tissue interface from the first step: the full-size case of the conservative conduction
    term (row f1).  Needle as in C4."""
    w = with_smooth_field(c4_body(steps=steps))
    w.name = "C4F"
    return w


BENCH_CONFIGS = {"C1": c1_cube, "C2": c2_phantom, "C3": c3_phantom, "C4": c4_body, "C5": c5_sweep,
                 "C4F": c4_face_case}
