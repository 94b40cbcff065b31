"""Pins for the fp64 oracle (oracle/rfa_oracle.c) against what the paper and the mathematics fix.

None of these tests re-types the oracle's update formula as the expected value: the expectations are
closed forms (DCT spectrum of the replicate-boundary second difference, geometric decay, erfc,
Green's function, linear / exponential steady states), conservation laws, theorems (monotonicity,
maximum principle, symmetry) and a brute-force dense-matrix formulation assembled from the PDE's
flux picture rather than from the voxel loop.  A plausible mistake (dropped term, wrong sign, swapped
dx/dy, transposed index, mm/m slip, wrong held handling) fails at least one of them.

Citations are to /root/reference/PAPER.md lines.
"""
import math

import numpy as np
import pytest
import scipy.fft
import scipy.special

from paper_1907_05709_b200 import workloads as W

RHO_CP_LIVER = 1060.0 * 3600.0
ALPHA_LIVER = float(np.float32(0.512)) / RHO_CP_LIVER          # m^2/s (the ABI's tissue table is fp32)


def one_label(k=0.512, rho=1060.0, cp=3600.0, wb_cb=0.0, q_m=0.0, t_init=37.0, flags=0):
    return W.make_table([(k, rho, cp, wb_cb, q_m, t_init, flags)])


# ----------------------------------------------------------------------------------------------
# 1. Exact discrete closed form (homogeneous, replicate boundaries => DCT-II eigenmodes)
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims,spacing", [((6, 5, 4), (0.7, 0.9, 1.3)), ((9, 4, 7), (1.3, 0.6, 0.8))])
def test_dct_closed_form_anisotropic(oracle, dims, spacing):
    """T^n = T_inf + IDCT[lambda^n DCT(T^0 - T_inf)],  lambda_abc = 1 - p - 4 sum_a c_a sin^2(pi a/2n_a),
    T_inf = T_a + Q_m/beta.  Non-cubic anisotropic grid: catches any x/y/z or dx/dy/dz mix-up,
    a wrong perfusion sign, a missing Q_m and the mm->m conversion."""
    nx, ny, nz = dims
    k, rho, cp, beta, qm, ta, dt = 0.52, 1079.0, 3540.0, 16.687 * 3617.0, 10714.0, 37.0, 0.02
    table = one_label(k, rho, cp, beta, qm)
    k, rho, cp, beta, qm = (float(table[f][0]) for f in ("k", "rho", "cp", "wb_cb", "q_m"))  # fp32 table
    rng = np.random.default_rng(1)
    T0 = 37.0 + 30.0 * rng.random((nz, ny, nx))
    sim = oracle.OracleSim(dims, spacing, np.zeros((nz, ny, nx), np.uint8), table, ta, dt)
    sim.set_temperature(T0)
    n = 200
    sim.step(n)
    D = dt / (rho * cp)
    c = [D * k / (s * 1e-3) ** 2 for s in spacing]
    p = D * beta
    lam = 1.0 - p
    lam = lam - 4.0 * c[0] * np.sin(np.pi * np.arange(nx) / (2 * nx))[None, None, :] ** 2
    lam = lam - 4.0 * c[1] * np.sin(np.pi * np.arange(ny) / (2 * ny))[None, :, None] ** 2
    lam = lam - 4.0 * c[2] * np.sin(np.pi * np.arange(nz) / (2 * nz))[:, None, None] ** 2
    t_inf = ta + qm / beta
    spec = scipy.fft.dctn(T0 - t_inf, type=2, norm="ortho")
    expect = t_inf + scipy.fft.idctn(spec * lam ** n, type=2, norm="ortho")
    assert np.max(np.abs(sim.T - expect)) < 1e-10


def test_uniform_relaxation_zero_mode(oracle):
    """Uniform field: theta^n = (1-p)^n theta^0 about T_inf = T_a + Q_m/beta = 37.1775 C for the paper's
    liver constants."""
    table = W.paper_liver_table()
    dims = (5, 4, 3)
    sim = oracle.OracleSim(dims, (1.0, 1.0, 1.0), np.zeros((3, 4, 5), np.uint8), table, 37.0, 0.1)
    sim.set_temperature(np.full((3, 4, 5), 50.0))
    sim.step(500)
    beta = float(table["wb_cb"][0])                                # the ABI table is fp32
    p = 0.1 * beta / (1079.0 * 3540.0)
    t_inf = 37.0 + 10714.0 / beta
    assert abs(t_inf - 37.1775) < 1e-4
    expect = t_inf + (1 - p) ** 500 * (50.0 - t_inf)
    assert np.max(np.abs(sim.T - expect)) < 1e-11


# ----------------------------------------------------------------------------------------------
# 2. Brute force: dense one-step matrix assembled from face fluxes, powered
# ----------------------------------------------------------------------------------------------
def _dense_operator(dims, spacing, lab, table, held, power, q_power, ta, dt):
    """A, b with T^{n+1} = A T^n + b, assembled face by face: every interior face (u,v) along axis a
    contributes K_u/(h_a^2) (T_v - T_u) to voxel u's conduction sum (centre-voxel K);
    outer faces carry no flux.  Independent of the oracle's neighbour-clamping loop."""
    nx, ny, nz = dims
    N = nx * ny * nz
    A = np.zeros((N, N))
    b = np.zeros(N)
    h = [s * 1e-3 for s in spacing]
    idx = lambda i, j, k: i + nx * (j + ny * k)
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                u = idx(i, j, k)
                if held[k, j, i]:
                    A[u, u] = 1.0
                    continue
                row = table[lab[k, j, i]]
                D = dt / (float(row["rho"]) * float(row["cp"]))
                A[u, u] += 1.0
                for (di, dj, dk, a) in ((1, 0, 0, 0), (-1, 0, 0, 0), (0, 1, 0, 1), (0, -1, 0, 1), (0, 0, 1, 2), (0, 0, -1, 2)):
                    ii, jj, kk = i + di, j + dj, k + dk
                    if 0 <= ii < nx and 0 <= jj < ny and 0 <= kk < nz:
                        g = D * float(row["k"]) / (h[a] * h[a])
                        A[u, idx(ii, jj, kk)] += g
                        A[u, u] -= g
                A[u, u] -= D * float(row["wb_cb"])
                b[u] += D * (float(row["wb_cb"]) * ta + float(row["q_m"]) + (q_power if power[k, j, i] else 0.0))
    return A, b


@pytest.mark.parametrize("dims,spacing,mode", [((4, 4, 4), (1.0, 1.0, 1.0), W.SRC_DIRICHLET),
                                               ((6, 5, 4), (0.7, 0.9, 1.3), W.SRC_DIRICHLET),
                                               ((6, 5, 4), (0.7, 0.9, 1.3), W.SRC_POWER)])
def test_bruteforce_dense_matrix(oracle, dims, spacing, mode):
    nx, ny, nz = dims
    rng = np.random.default_rng(3)
    table = W.tissue_table()
    table["q_m"][1] = 10714.0                                   # exercise Q_m as well
    lab = rng.integers(0, 7, size=(nz, ny, nx)).astype(np.uint8)
    mask = np.zeros((nz, ny, nx), np.uint8)
    mask[1, 2, 1] = 1
    mask[2, 2, 2] = 1
    lab[2, 2, 2] = W.VESSEL                                     # needle voxel inside a vessel (R-15 / R-17)
    dt, ta = 0.05, 37.0
    value = 90.0 if mode == W.SRC_DIRICHLET else 5.0e7
    sim = oracle.OracleSim(dims, spacing, lab, table, ta, dt)
    sim.set_needle(mask, mode, value)
    T0 = sim.T.copy()
    label_held = (table["flags"][lab] & 1) != 0
    if mode == W.SRC_DIRICHLET:
        held = label_held | (mask != 0)                          # needle overrides the label
        power = np.zeros_like(mask)
        assert T0[2, 2, 2] == 90.0 and T0[1, 2, 1] == 90.0
    else:
        held = label_held                                        # a held label under a POWER mask stays held
        power = mask
        assert T0[2, 2, 2] == 37.0
    A, b = _dense_operator(dims, spacing, lab, table, held, power, value if mode == W.SRC_POWER else 0.0, ta, dt)
    n = 300
    sim.step(n)
    t = T0.ravel().copy()
    for _ in range(n):
        t = A @ t + b
    assert np.max(np.abs(sim.T.ravel() - t)) < 1e-9
    # held voxels are bit-identical before/after (Alg. 1 :313)
    assert np.array_equal(sim.T[held], T0[held])


# ----------------------------------------------------------------------------------------------
# 3. Conservation
# ----------------------------------------------------------------------------------------------
def test_energy_conservation_homogeneous(oracle):
    """Zero-flux boundaries, no perfusion, no sources: sum(T) is conserved (north_star energy check)."""
    dims = (12, 9, 7)
    rng = np.random.default_rng(5)
    T0 = 37.0 + 40.0 * rng.random((7, 9, 12))
    sim = oracle.OracleSim(dims, (0.8, 1.1, 0.9), np.zeros((7, 9, 12), np.uint8), one_label(), 37.0, 0.1)
    sim.set_temperature(T0)
    sim.step(500)
    assert abs(sim.T.sum() - T0.sum()) / T0.sum() < 1e-13
    assert sim.T.std() < T0.std()                               # it did diffuse


def test_weighted_energy_mixed_tissues(oracle):
    """With the centre-voxel K of Eq. 12 (R-3) and mixed tissues the conserved
    quantity is sum_v (rho c_p / K)_v T_v, not sum rho c_p T."""
    dims = (10, 8, 6)
    rng = np.random.default_rng(6)
    table = W.make_table([(0.21, 911.0, 2348.0, 0, 0, 37.0, 0), (0.512, 1060.0, 3600.0, 0, 0, 37.0, 0),
                          (0.53, 1050.0, 3700.0, 0, 0, 37.0, 0)])
    lab = rng.integers(0, 3, size=(6, 8, 10)).astype(np.uint8)
    T0 = 37.0 + 40.0 * rng.random((6, 8, 10))
    sim = oracle.OracleSim(dims, (1.0, 0.7, 1.2), lab, table, 37.0, 0.05)
    sim.set_temperature(T0)
    wgt = (table["rho"].astype(np.float64) * table["cp"] / table["k"])[lab]
    sim.step(500)
    e0, e1 = (wgt * T0).sum(), (wgt * sim.T).sum()
    assert abs(e1 - e0) / e0 < 1e-13
    plain0, plain1 = ((table["rho"].astype(np.float64) * table["cp"])[lab] * T0).sum(), ((table["rho"].astype(np.float64) * table["cp"])[lab] * sim.T).sum()
    assert abs(plain1 - plain0) / plain0 > 1e-9                 # the plain sum is NOT conserved


def test_power_source_energy_balance(oracle):
    """Constant power Q in m voxels, no perfusion, nothing held: sum(T) rises by exactly
    n*m*dt*Q/(rho c_p) (R-17; first law)."""
    dims = (9, 8, 7)
    mask = np.zeros((7, 8, 9), np.uint8)
    mask[3, 3:6, 4] = 1
    sim = oracle.OracleSim(dims, (1.0, 1.0, 1.0), np.zeros((7, 8, 9), np.uint8), one_label(), 37.0, 0.1)
    sim.set_needle(mask, W.SRC_POWER, 5.0e7)
    s0 = sim.T.sum()
    sim.step(50)
    expect = 50 * 3 * 0.1 * 5.0e7 / RHO_CP_LIVER
    assert abs((sim.T.sum() - s0) - expect) / expect < 1e-11


# ----------------------------------------------------------------------------------------------
# 4. Stability (CFL)
# ----------------------------------------------------------------------------------------------
def test_stability_bound_highest_mode(oracle):
    """The fastest mode of the replicate-boundary Laplacian is the DCT mode (n-1,n-1,n-1) with factor
    lambda = 1 - p - 4 sum_a c_a sin^2(pi (n_a-1)/(2 n_a)).  5 % above the dt where lambda = -1 it grows,
    5 % below it decays (north_star: 'the CFL stability bound')."""
    n = 8
    dims = (n, n, n)
    h = 1.0e-3
    beta = float(np.float32(24306.24))
    s2 = math.sin(math.pi * (n - 1) / (2 * n)) ** 2
    # lambda(dt) = 1 - dt*(beta/(rho cp) + 12 alpha s2 / h^2) = -1
    dt_crit = 2.0 / (beta / RHO_CP_LIVER + 12.0 * ALPHA_LIVER * s2 / h ** 2)
    ax = np.cos(np.pi * (np.arange(n) + 0.5) * (n - 1) / n)
    mode = ax[:, None, None] * ax[None, :, None] * ax[None, None, :]
    for f, grows in ((1.05, True), (0.95, False)):
        sim = oracle.OracleSim(dims, (1.0, 1.0, 1.0), np.zeros((n, n, n), np.uint8),
                               one_label(wb_cb=beta), 37.0, f * dt_crit)
        sim.set_temperature(37.0 + mode)
        a0 = np.abs(sim.T - 37.0).max()
        sim.step(60)
        a1 = np.abs(sim.T - 37.0).max()
        lam = 1.0 - f * dt_crit * (beta / RHO_CP_LIVER + 12.0 * ALPHA_LIVER * s2 / h ** 2)
        assert (a1 > 2 * a0) == grows
        assert a1 / a0 == pytest.approx(abs(lam) ** 60, rel=1e-6)
        # the monotone bound of DESIGN.md R-18, dt (2 alpha sum 1/h^2 + beta/(rho cp)) <= 1, sits just
        # below the von Neumann one, dt (2 alpha s2 sum 1/h^2 + beta/(2 rho cp)) <= 1: on this grid
        # it separates the growing from the decaying run
        assert (sim.stability_number() > 1.0) == grows


def test_stability_number_of_configs(oracle):
    """All BASELINE configs sit far below the monotone bound; the paper's own setting (0.5 mm, 0.1 s,
    PAPER.md:145) gives about 0.33."""
    w = W.c1_cube()
    sim = oracle.OracleSim(w.dims, w.spacing_mm, w.labels, w.table, 37.0, w.dt)
    assert 0.05 < sim.stability_number() < 0.1
    sim = oracle.OracleSim((4, 4, 4), (0.5, 0.5, 0.5), np.zeros((4, 4, 4), np.uint8), W.paper_liver_table(), 37.0, 0.1)
    assert 0.30 < sim.stability_number() < 0.36


# ----------------------------------------------------------------------------------------------
# 5. Monotone heating, maximum principle, symmetry
# ----------------------------------------------------------------------------------------------
def test_monotone_heating_and_max_principle(oracle):
    w = W.ragged_phantom(dims=(24, 20, 16), steps=0)
    sim = oracle.OracleSim(w.dims, w.spacing_mm, w.labels, w.table, 37.0, w.dt)
    nd = w.needles[0]
    sim.set_needle(nd.mask, nd.mode, nd.value)
    assert sim.stability_number() <= 1.0
    prev_T, prev_n = sim.T.copy(), int(sim.necro.sum())
    for _ in range(40):
        sim.step(5)
        assert np.all(sim.T >= prev_T)                          # every voxel non-decreasing
        assert int(sim.necro.sum()) >= prev_n                    # necrotic volume non-decreasing
        assert sim.T.min() >= 37.0 and sim.T.max() <= 90.0       # max principle (Q_m = Q = 0)
        prev_T, prev_n = sim.T.copy(), int(sim.necro.sum())
    m = nd.mask != 0
    assert np.all(sim.necro[m] == 1)                            # necro contains the 90 C mask
    assert np.array_equal(sim.necro != 0, (sim.T >= 60.0))       # sticky == instantaneous when monotone


def test_symmetry_48fold(oracle):
    """Single-voxel tip in a homogeneous isotropic odd cube: invariant under axis permutations and flips
    (the zone 'converges to a spherical shape')."""
    n = 15
    lab = np.ones((n, n, n), np.uint8)
    mask = np.zeros((n, n, n), np.uint8)
    mask[7, 7, 7] = 1
    sim = oracle.OracleSim((n, n, n), (1.0, 1.0, 1.0), lab, W.tissue_table(), 37.0, 0.1)
    sim.set_needle(mask, W.SRC_DIRICHLET, 90.0)
    sim.step(300)
    T = sim.T
    for perm in ((0, 1, 2), (1, 0, 2), (2, 1, 0), (0, 2, 1), (1, 2, 0), (2, 0, 1)):
        P = np.transpose(T, perm)
        for fz in (1, -1):
            for fy in (1, -1):
                for fx in (1, -1):
                    assert np.max(np.abs(P[::fz, ::fy, ::fx] - T)) < 1e-12
    assert T[7, 7, 8] > T[7, 8, 8] > T[8, 8, 8] > 37.0


def test_vessel_cools_the_zone(oracle):
    """A held 37 C vessel next to the tip makes the zone aspherical (Fig. 11b,c)."""
    n = 21
    lab = np.ones((n, n, n), np.uint8)
    lab[:, :, 13:15] = W.VESSEL
    mask = np.zeros((n, n, n), np.uint8)
    mask[10, 10, 10] = 1
    sim = oracle.OracleSim((n, n, n), (1.0, 1.0, 1.0), lab, W.tissue_table(), 37.0, 0.1)
    sim.set_needle(mask, W.SRC_DIRICHLET, 90.0)
    sim.step(600)
    assert sim.T[10, 10, 12] < sim.T[10, 10, 8] - 0.5           # vessel side is cooler
    assert np.all(sim.T[:, :, 13:15] == 37.0)


# ----------------------------------------------------------------------------------------------
# 6. Continuum solutions: Green's function (Eq. 2), erfc plane source (Eq. 4), steady states
# ----------------------------------------------------------------------------------------------
def _green_error(oracle, n, h_mm, dt, t_end):
    w = W.c1_green(n=n, h_mm=h_mm, dt=dt, steps=int(round(t_end / dt)), energy=1.0e4)
    sim = oracle.run_workload(w)
    c = n // 2
    x = (np.arange(n) - c) * h_mm * 1e-3
    r2 = x[:, None, None] ** 2 + x[None, :, None] ** 2 + x[None, None, :] ** 2
    vol = (h_mm * 1e-3) ** 3
    # Eq. 2 in its 3-D product form, for a heat content of energy*vol in one voxel
    exact = 1.0e4 * vol * (4 * np.pi * ALPHA_LIVER * t_end) ** -1.5 * np.exp(-r2 / (4 * ALPHA_LIVER * t_end))
    num = sim.T - 37.0
    return np.max(np.abs(num - exact)) / exact.max(), num.sum() * vol / (1.0e4 * vol)


def test_greens_function_refinement(oracle):
    """Error against Eq. 2 shrinks ~4x per halving of h (dt ~ h^2), 32 mm box, t = 25 s."""
    e = []
    for n, h, dt in ((16, 2.0, 0.4), (32, 1.0, 0.1), (64, 0.5, 0.025)):
        err, mass = _green_error(oracle, n, h, dt, 25.0)
        assert abs(mass - 1.0) < 1e-12                           # heat content conserved
        e.append(err)
    assert e[0] > e[1] > e[2]
    assert 3.0 < e[1] / e[2] < 5.0
    assert e[2] < 0.02


def _plane_source(oracle, nx, h_mm, dt, t_end, beta=0.0):
    lab = np.zeros((1, 1, nx), np.uint8)
    mask = np.zeros((1, 1, nx), np.uint8)
    mask[0, 0, 0] = 1
    sim = oracle.OracleSim((nx, 1, 1), (h_mm, 1.0, 1.0), lab, one_label(wb_cb=beta), 37.0, dt)
    sim.set_needle(mask, W.SRC_DIRICHLET, 90.0)
    sim.step(int(round(t_end / dt)))
    return sim.T[0, 0, :]


def test_erfc_plane_source(oracle):
    """Held plane at 90 C, no perfusion: theta = theta_0 erfc(x / (2 sqrt(alpha t))) -- the integral of
    Eq. 4 with h(s) = T_0 (R-21) -- with second-order convergence."""
    errs = []
    for nx, h, dt in ((100, 1.0, 0.1), (200, 0.5, 0.025)):
        T = _plane_source(oracle, nx, h, dt, 100.0)
        x = np.arange(nx) * h * 1e-3
        exact = 37.0 + 53.0 * scipy.special.erfc(x / (2 * math.sqrt(ALPHA_LIVER * 100.0)))
        errs.append(np.max(np.abs(T - exact)))
    assert errs[0] < 0.06 and errs[1] < 0.015                   # out of a 53 C amplitude
    assert 3.0 < errs[0] / errs[1] < 5.0


def test_steady_state_line_and_exponential(oracle):
    """Between two held planes the steady state without perfusion 'is a line' (Fig. 2b);
    with perfusion the discrete steady state is A r^i + B r^-i with c (r + 1/r - 2) = p."""
    nx = 21
    lab = np.zeros((1, 1, nx), np.uint8)
    lab[0, 0, -1] = 1
    for beta in (0.0, float(np.float32(60357.0))):
        table = W.make_table([(0.512, 1060.0, 3600.0, beta, 0.0, 37.0, 0),
                              (0.512, 1060.0, 3600.0, 0.0, 0.0, 37.0, 1)])
        mask = np.zeros((1, 1, nx), np.uint8)
        mask[0, 0, 0] = 1
        sim = oracle.OracleSim((nx, 1, 1), (1.0, 1.0, 1.0), lab, table, 37.0, 1.0)
        sim.set_needle(mask, W.SRC_DIRICHLET, 90.0)
        assert sim.stability_number() <= 1.0
        sim.step(40000)
        i = np.arange(nx)
        if beta == 0.0:
            expect = 90.0 - 53.0 * i / (nx - 1)
        else:
            c = 1.0 * ALPHA_LIVER / 1e-6
            p = 1.0 * beta / RHO_CP_LIVER
            s = 2.0 + p / c
            r = (s + math.sqrt(s * s - 4.0)) / 2.0
            # theta_0 = 53, theta_{nx-1} = 0
            Bc = 53.0 / (1.0 - r ** (-2.0 * (nx - 1)))
            Ac = 53.0 - Bc
            expect = 37.0 + Ac * r ** i + Bc * r ** (-i.astype(float))
        assert np.max(np.abs(sim.T[0, 0, :] - expect)) < 1e-9


# ----------------------------------------------------------------------------------------------
# 7. Needle semantics and necrosis (R-11..R-16)
# ----------------------------------------------------------------------------------------------
def test_needle_override_release_and_sticky_necrosis(oracle):
    n = 9
    lab = np.ones((n, n, n), np.uint8)
    lab[4, 4, 5] = W.VESSEL
    sim = oracle.OracleSim((n, n, n), (1.0, 1.0, 1.0), lab, W.tissue_table(), 37.0, 0.1)
    m1 = np.zeros((n, n, n), np.uint8)
    m1[4, 4, 4] = 1
    m1[4, 4, 5] = 1                       # inside the vessel: needle overrides (R-15)
    sim.set_needle(m1, W.SRC_DIRICHLET, 90.0)
    assert sim.T[4, 4, 5] == 90.0 and sim.necro[4, 4, 4] == 1
    sim.step(200)
    hot = sim.T[4, 4, 3]
    assert hot > 50.0 and sim.T[4, 4, 5] == 90.0
    nec = sim.necro.copy()
    m2 = np.zeros((n, n, n), np.uint8)
    m2[1, 1, 1] = 1
    sim.set_needle(m2, W.SRC_DIRICHLET, 59.9995)          # move the needle (R-16); below threshold
    assert sim.T[4, 4, 4] == 90.0                         # released voxel keeps its temperature ...
    sim.step(1)
    assert sim.T[4, 4, 4] < 90.0                          # ... and is ordinary tissue again
    assert sim.T[4, 4, 5] == 90.0                         # the vessel voxel is held again (at its value)
    assert sim.necro[1, 1, 1] == 0                        # 59.9995 < 60: not necrotic (>= 60, R-11)
    sim.step(2000)
    assert sim.T[4, 4, 3] < hot                           # cooled down
    assert np.all(sim.necro[nec != 0] == 1)               # necrosis is sticky (R-12)
    sim.set_needle(None, W.SRC_OFF, 0.0)
    assert sim.held.sum() == 1                            # only the vessel voxel


def test_threshold_is_inclusive(oracle):
    lab = np.zeros((2, 2, 2), np.uint8)
    sim = oracle.OracleSim((2, 2, 2), (1.0, 1.0, 1.0), lab, one_label(t_init=60.0), 37.0, 0.1)
    assert sim.necro.sum() == 8                           # T >= 60 on the initial state (R-11, R-14)
    sim = oracle.OracleSim((2, 2, 2), (1.0, 1.0, 1.0), lab, one_label(t_init=59.999), 37.0, 0.1)
    assert sim.necro.sum() == 0


# ----------------------------------------------------------------------------------------------
# 8. The stored golden files were written by this oracle from these inputs
# ----------------------------------------------------------------------------------------------
def test_golden_c2_is_reproducible_prefix(oracle):
    """Re-runs the first quarter (1500 steps) of C2 and compares with tests/golden/C2_golden.npz."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "C2_golden.npz")
    g = np.load(path)
    w = W.c2_phantom()
    sim = oracle.run_workload(w, steps=int(g["checkpoints"][0]))
    got = sim.T.ravel()[g["sample_idx"]]
    assert np.array_equal(got, g["sample_T"][0])


# ----------------------------------------------------------------------------------------------
# Probe time series (SURVEY.md 8(f) f2; PAPER.md:147 Fig. 6 probe sets, :159 / Fig. 14 monotone convergence)
# ----------------------------------------------------------------------------------------------
def _probe_series(oracle, tip_c, steps=600, every=10):
    w = W.paper_probe_case(tip_c, steps=steps)
    pr = W.fig6_probes(w.dims, w.spacing_mm, w.meta["centre_voxel"])
    sim = oracle.OracleSim(w.dims, w.spacing_mm, w.labels, w.table, w.t_blood, w.dt)
    nd = w.needles[0]
    sim.set_needle(nd.mask, nd.mode, nd.value)
    return sim.step_record(steps, every, pr.ravel()), pr


def test_probe_series_monotone_symmetric_affine(oracle):
    s90, pr = _probe_series(oracle, 90.0)
    s60, _ = _probe_series(oracle, 60.0)
    s75, _ = _probe_series(oracle, 75.0)
    assert s90.shape == (60, 12)
    # the paper's claim (Fig. 14): monotone convergence at the probes, from step 0 (R-18)
    assert np.all(np.diff(s90, axis=0) >= -1e-12) and np.all(np.diff(s60, axis=0) >= -1e-12)
    # Fig. 6: the +-x and +-y probes of one distance are equivalent by the symmetry of the hemispherical tip
    # (x <-> y exactly; +x vs -x up to the wall reflection, the tip voxel is not the centre of an even box)
    for base in (0, 6):
        assert np.max(np.abs(s90[:, base + 0] - s90[:, base + 2])) < 1e-11
        assert np.max(np.abs(s90[:, base + 1] - s90[:, base + 3])) < 1e-11
        assert np.max(np.abs(s90[:, base + 0] - s90[:, base + 1])) < 1e-8
    # the 2.5 mm set is hotter than the 5 mm set; the tip side (+z, inside/above the dome) is the hottest
    assert np.all(s90[-1, :4] > s90[-1, 6:10]) and s90[-1, 5] > s90[-1, 0] > s90[-1, 4]
    # the update is affine in the held tip value: T(75) = (T(90) + T(60)) / 2 at every probe and time
    assert np.max(np.abs(s75 - 0.5 * (s90 + s60))) < 1e-11
    # bounded by the tip temperature and by the far-field equilibrium T_a + Q_m / (w_b c_b) from below
    assert s90.max() < 90.0 and s90.min() >= 37.0


@pytest.mark.parametrize("every", [1, 4])
def test_probe_series_row_m_is_the_field_after_m_plus_1_times_every_steps(oracle, every):
    """Pin of OracleSim.step_record's row <-> step mapping on the paper's probe set-up (Fig. 6 :250,
    Fig. 14 :282): row m must equal the field of a FRESH simulation advanced (m+1)*every times by plain step(1) calls and
    read at the probe voxels.  A record taken before the step, a row shifted by one record, or `every` applied once too
    often or too seldom all change some row: the probes heat strictly monotonically, so consecutive fields differ."""
    w = W.paper_probe_case(90.0, n=32, steps=24)
    pr = W.fig6_probes(w.dims, w.spacing_mm, w.meta["centre_voxel"]).ravel()
    nd = w.needles[0]

    def fresh():
        sim = oracle.OracleSim(w.dims, w.spacing_mm, w.labels, w.table, w.t_blood, w.dt)
        sim.set_needle(nd.mask, nd.mode, nd.value)
        return sim

    rec = fresh().step_record(w.steps, every, pr)
    assert rec.shape == (w.steps // every, pr.size)
    nx, ny, nz = w.dims
    ref = fresh()
    fields = []                                   # fields[t] = probe values after t+1 single steps, read by (k, j, i)
    for _ in range(w.steps):
        ref.step(1)
        fields.append(np.array([ref.T[p // (nx * ny), (p // nx) % ny, p % nx] for p in pr]))
    for m in range(rec.shape[0]):
        assert np.array_equal(rec[m], fields[(m + 1) * every - 1]), f"row {m} is not the field after {(m + 1) * every} steps"
    # the pin has teeth: neighbouring candidates (one step / one record earlier or later) are different fields
    assert not np.array_equal(fields[every - 1], fields[every]) and not np.array_equal(fields[0], np.full(pr.size, 37.0))
    if every > 1:
        assert not np.array_equal(rec[0], fields[0])
    # the simulation that recorded has advanced n steps in total
    sim = fresh()
    sim.step_record(w.steps, every, pr)
    assert sim.steps_done == w.steps and np.array_equal(sim.T, ref.T)


def test_necrotic_volume_counts_tissue_voxels_in_cubic_millimetres(oracle):
    """Pin of OracleSim.necrotic_volume_mm3 (necrosis at T >= 60 C: PAPER.md:37; reported volume without needle and
    held-label voxels: DESIGN.md R-13) on a hand-built anisotropic grid, 0.7 x 0.9 x 1.3 mm, where every count is known
    by construction: no step is taken, the mask comes from the initial image alone."""
    dims, spacing = (6, 5, 4), (0.7, 0.9, 1.3)
    vox = 0.7 * 0.9 * 1.3                                             # mm^3, typed here from the spacing
    table = W.make_table([
        (0.52, 1079.0, 3540.0, 0.0, 0.0, 37.0, 0),                   # 0 tissue, cold
        (0.52, 1079.0, 3540.0, 0.0, 0.0, 61.0, 0),                   # 1 tissue that starts above the threshold
        (0.512, 1060.0, 3600.0, 0.0, 0.0, 75.0, W.TISSUE_HELD),       # 2 HELD label that is hot (not tissue damage)
        (0.52, 1079.0, 3540.0, 0.0, 0.0, 59.999, 0),                 # 3 tissue just below the threshold
        (0.52, 1079.0, 3540.0, 0.0, 0.0, 60.0, 0),                   # 4 tissue exactly at it: inclusive
    ])
    lab = np.zeros((4, 5, 6), np.uint8)                               # (nz, ny, nx)
    lab[0, 0, 0:5] = 1                                                # 5 hot tissue voxels
    lab[1, 1:4, 2] = 2                                                # 3 hot held-label voxels
    lab[2, 4, 0:2] = 3                                                # 2 voxels at 59.999: not necrotic
    lab[3, 2, 1:5] = 4                                                # 4 voxels at exactly 60.0: necrotic
    sim = oracle.OracleSim(dims, spacing, lab, table, 37.0, 0.05)
    assert int(sim.necro.sum()) == 5 + 3 + 4
    assert sim.necrotic_volume_mm3() == pytest.approx((5 + 4) * vox, rel=1e-12)
    assert sim.necrotic_volume_mm3(exclude_held=False) == pytest.approx((5 + 3 + 4) * vox, rel=1e-12)
    # a Dirichlet needle at 90 C over 7 voxels: 2 of them were hot tissue already, 1 is a held-label voxel, 4 were cold
    mask = np.zeros_like(lab)
    mask[0, 0, 3:5] = 1
    mask[1, 1, 2] = 1
    mask[2, 0:4, 5] = 1
    sim.set_needle(mask, W.SRC_DIRICHLET, 90.0)
    assert int(sim.necro.sum()) == 12 + 4
    assert sim.necrotic_volume_mm3() == pytest.approx((3 + 4) * vox, rel=1e-12)              # tissue only: 5 - 2 + 4
    assert sim.necrotic_volume_mm3(exclude_held=False) == pytest.approx(16 * vox, rel=1e-12)
    # a POWER needle heats but holds nothing, yet its voxels are electrode, not tissue (R-13): a hot tissue voxel under
    # the mask leaves the reported volume; the 4 voxels the Dirichlet needle burnt stay in the sticky mask and count again
    mask2 = np.zeros_like(lab)
    mask2[3, 2, 1] = 1
    sim.set_needle(mask2, W.SRC_POWER, 1.0e6)
    assert sim.necrotic_volume_mm3(exclude_held=False) == pytest.approx(16 * vox, rel=1e-12)
    assert sim.necrotic_volume_mm3() == pytest.approx((5 + 3 + 4) * vox, rel=1e-12)          # 5 hot + (4 - 1) at 60 + 4 burnt


# ----------------------------------------------------------------------------------------------
# Row f1: conservative heterogeneous conduction div(K grad T) of Eq. 9, harmonic-mean
# face conductivities (R-28).  Pins of rfa_oracle_step_cons.
# ----------------------------------------------------------------------------------------------
_MIX = [(0.21, 911.0, 2348.0, 0, 0, 37.0, 0), (0.512, 1060.0, 3600.0, 0, 0, 37.0, 0),
        (0.53, 1050.0, 3700.0, 0, 0, 37.0, 0)]


def test_cons_energy_is_conserved_with_mixed_tissues(oracle):
    """The defining property of the conservative form (north_star: "energy conservation with zero-flux
    boundaries and no sources"): sum_v rho c_p T_v is constant for ANY mix of tissues, which the
    centre-K form of Eq. 12 does not give (test_weighted_energy_mixed_tissues)."""
    dims = (10, 8, 6)
    rng = np.random.default_rng(16)
    table = W.make_table(_MIX)
    lab = rng.integers(0, 3, size=(6, 8, 10)).astype(np.uint8)
    T0 = 37.0 + 40.0 * rng.random((6, 8, 10))
    sim = oracle.OracleSim(dims, (1.0, 0.7, 1.2), lab, table, 37.0, 0.05, conservative=True)
    sim.set_temperature(T0)
    rc = (table["rho"].astype(np.float64) * table["cp"])[lab]
    sim.step(500)
    e0, e1 = (rc * T0).sum(), (rc * sim.T).sum()
    assert abs(e1 - e0) / e0 < 1e-13
    assert np.ptp(sim.T) < np.ptp(T0)                       # and it diffuses
    wgt = rc / table["k"].astype(np.float64)[lab]
    assert abs((wgt * sim.T).sum() - (wgt * T0).sum()) / (wgt * T0).sum() > 1e-9   # the Eq. 12 invariant is not


def test_cons_equals_eq12_when_homogeneous(oracle):
    """One tissue (K constant): div(K grad T) = K lap T, so both forms must agree (Eq. 9 -> Eq. 10)."""
    w = W.ragged_phantom(dims=(14, 11, 9), spacing=(0.7, 0.9, 1.3), steps=60, dt=0.05)
    lab = np.where(w.labels == W.VESSEL, W.VESSEL, W.LIVER).astype(np.uint8)     # liver + held vessel, same K
    a = oracle.OracleSim(w.dims, w.spacing_mm, lab, w.table, 37.0, w.dt)
    b = oracle.OracleSim(w.dims, w.spacing_mm, lab, w.table, 37.0, w.dt, conservative=True)
    for s in (a, b):
        s.set_needle(w.needles[0].mask, W.SRC_DIRICHLET, 90.0)
        s.step(60)
    assert np.max(np.abs(a.T - b.T)) < 1e-11 and a.T.max() == 90.0


def test_cons_two_layer_slab_is_series_resistors(oracle):
    """1-D fat | liver slab between two held faces: the steady heat flux is (T_L - T_R) / sum(R) with
    the thermal resistances h/K of the half-cells in series (textbook), and the temperature drops by
    q R along the way.  The harmonic-mean face conductivity is exactly the two half-cells in series."""
    n, m = 24, 10                                           # m fat voxels, then liver
    table = W.make_table([(0.21, 911.0, 2348.0, 0, 0, 37.0, 0), (0.512, 1060.0, 3600.0, 0, 0, 37.0, 0),
                          (0.21, 911.0, 2348.0, 0, 0, 80.0, W.TISSUE_HELD),
                          (0.512, 1060.0, 3600.0, 0, 0, 37.0, W.TISSUE_HELD)])
    lab = np.array([2] + [0] * (m - 1) + [1] * (n - m - 1) + [3], np.uint8).reshape(1, 1, n)
    sim = oracle.OracleSim((n, 1, 1), (1.0, 1.0, 1.0), lab, table, 37.0, 1.0, conservative=True)
    assert sim.stability_number() <= 1.0
    sim.step(120000)
    h = 1.0e-3
    k_fat, k_liv = float(table["k"][0]), float(table["k"][1])   # the fp32 table values both sides are given
    kv = np.array([k_fat] * m + [k_liv] * (n - m))
    R = np.concatenate([[0.0], np.cumsum(0.5 * h / kv[:-1] + 0.5 * h / kv[1:])])   # centre-to-centre
    q = (80.0 - 37.0) / R[-1]
    assert np.max(np.abs(sim.T.ravel() - (80.0 - q * R))) < 1e-9
    # the kink: slopes on the two sides are in the ratio K_liver / K_fat
    T = sim.T.ravel()
    assert abs((T[3] - T[4]) / (T[n - 5] - T[n - 4]) - k_liv / k_fat) < 1e-8


def test_cons_operator_is_symmetric_stochastic_nonnegative(oracle):
    """The one-step map A (columns = images of unit fields) of the conservative form: flux antisymmetry
    makes diag(rho c_p)(A - I) symmetric, no-flux walls make every row sum to 1, and under the monotone
    bound all entries are >= 0 (max principle)."""
    dims = (5, 4, 3)
    nx, ny, nz = dims
    N = nx * ny * nz
    rng = np.random.default_rng(3)
    table = W.make_table(_MIX)
    lab = rng.integers(0, 3, size=(nz, ny, nx)).astype(np.uint8)
    A = np.zeros((N, N))
    for j in range(N):
        sim = oracle.OracleSim(dims, (0.7, 0.9, 1.3), lab, table, 0.0, 0.2, t_necrosis=1e9, conservative=True)
        e = np.zeros(N)
        e[j] = 1.0
        sim.set_temperature(e.reshape(nz, ny, nx))
        sim.step(1)
        A[:, j] = sim.T.ravel()
    rc = (table["rho"].astype(np.float64) * table["cp"])[lab].ravel()
    M = rc[:, None] * (A - np.eye(N))
    assert np.max(np.abs(M - M.T)) < 1e-9 * np.max(np.abs(M))
    assert np.max(np.abs(A.sum(axis=1) - 1.0)) < 1e-14 and A.min() >= 0.0
    # a fat|liver face couples the two voxels with dt * Kf / h^2 / (rho c_p), Kf = 2 K1 K2 / (K1 + K2)
    found = False
    for u in range(N - 1):
        if (u % nx) < nx - 1 and {int(lab.ravel()[u]), int(lab.ravel()[u + 1])} == {0, 1}:
            kf = 2 * 0.21 * 0.512 / (0.21 + 0.512)
            assert abs(A[u, u + 1] * rc[u] - 0.2 * kf / (0.7e-3) ** 2) < 1e-6 * abs(A[u, u + 1] * rc[u])
            found = True
            break
    assert found
