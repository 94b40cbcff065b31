"""GPU parity tests: the CUDA path (through the C ABI of librfa.so) against the fp64 oracle, element by
element on the same seeded inputs.

Bars (BASELINE.json north_star): max |dT| <= 1e-3 C after the configured number of steps; the necrosis
mask identical except for voxels whose oracle temperature lies within 1e-3 C of 60 C (counted).  Kernel
variants must agree bit for bit (integer/byte work and the shared fp32 arithmetic).
"""
import os

import numpy as np
import pytest

from paper_1907_05709_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1.0e-3        # deg C, north_star
BAND = 1.0e-3       # exempt band around 60 C, north_star
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def rfa():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1907_05709_b200 import binding, build
    build.build()
    binding.load_library()          # raises if librfa.so is missing: no fallback
    return binding


def run_gpu(rfa, w, steps, kernel=None, fused=0, scenario_list=None, res_prefetch=None, cons=False):
    sim = rfa.from_workload(w)
    if kernel is not None:
        sim.configure(kernel, fused)
    if res_prefetch is not None:
        sim.configure_residual_prefetch(res_prefetch)
    if cons:
        sim.set_conduction(rfa.COND_FACE)
    sim.step(steps)
    sc = range(w.batch) if scenario_list is None else scenario_list
    T = [sim.get_temperature(b) for b in sc]
    N = [sim.get_necrosis(b) for b in sc]
    q = sim.query()
    sim.close()
    return T, N, q


def compare(T_gpu, N_gpu, osim, tol=TOL):
    To = osim.T
    err = float(np.max(np.abs(T_gpu.astype(np.float64) - To)))
    assert err <= tol, f"max |dT| = {err:.3e} > {tol}"
    mism = (N_gpu != 0) != (osim.necro != 0)
    exempt = np.abs(To - 60.0) <= BAND
    bad = int((mism & ~exempt).sum())
    assert bad == 0, f"{bad} necrosis mismatches outside the +-{BAND} C band ({int(mism.sum())} inside)"
    return err, int((mism & exempt).sum())


# ----------------------------------------------------------------------------------------------
# small ragged cases: several tiles, ragged tails, all labels, both source modes
# ----------------------------------------------------------------------------------------------
RAGGED = [
    dict(dims=(136, 70, 21), spacing=(0.7, 0.9, 1.3), steps=37, mode=W.SRC_DIRICHLET, value=90.0),
    dict(dims=(72, 130, 19), spacing=(1.1, 0.8, 0.9), steps=41, mode=W.SRC_POWER, value=2.0e7),
    dict(dims=(44, 38, 29), spacing=(1.0, 1.0, 1.0), steps=50, mode=W.SRC_DIRICHLET, value=60.0),
    dict(dims=(45, 38, 29), spacing=(0.7, 0.9, 1.3), steps=30, mode=W.SRC_DIRICHLET, value=90.0),   # nx % 4 != 0
]


@pytest.mark.parametrize("case", RAGGED, ids=lambda c: "x".join(map(str, c["dims"])))
def test_ragged_parity_and_variants(rfa, oracle, case):
    w = W.ragged_phantom(dims=case["dims"], spacing=case["spacing"], steps=case["steps"], mode=case["mode"],
                         value=case["value"], q_m=10714.0, dt=0.05)
    w.table["t_init"][W.KIDNEY] = 36.0          # a label whose initial temperature differs from T_a
    osim = oracle.run_workload(w)
    Tp, Np, qp = run_gpu(rfa, w, w.steps, rfa.KERNEL_PLAIN)
    assert qp["kernel"] == rfa.KERNEL_PLAIN
    err, n_band = compare(Tp[0], Np[0], osim)
    assert err < 2e-4                            # far inside the bar on short runs
    if case["dims"][0] % 4 == 0:
        for fused in (1, 2, 3, 4):
            Tb, Nb, qb = run_gpu(rfa, w, w.steps, rfa.KERNEL_BLOCKED, fused)
            assert qb["kernel"] == rfa.KERNEL_BLOCKED and qb["fused_steps"] == fused
            assert np.array_equal(Tb[0].view(np.uint32), Tp[0].view(np.uint32)), f"fused={fused} differs from plain"
            assert np.array_equal(Nb[0], Np[0])
        # the residual-prefetch variant (fp16 residual rows of hot planes fetched one plane ahead): same bits, Eq. 12 and conservative
        for fused in (2, 3):
            Tr, Nr, _ = run_gpu(rfa, w, w.steps, rfa.KERNEL_BLOCKED, fused, res_prefetch=rfa.RES_PREFETCH_ON)
            assert np.array_equal(Tr[0].view(np.uint32), Tp[0].view(np.uint32)), f"fused={fused} with residual prefetch differs from plain"
            assert np.array_equal(Nr[0], Np[0])
        Tc0, Nc0, _ = run_gpu(rfa, w, w.steps, rfa.KERNEL_PLAIN, cons=True)
        Tc1, Nc1, _ = run_gpu(rfa, w, w.steps, rfa.KERNEL_BLOCKED, 3, res_prefetch=rfa.RES_PREFETCH_ON, cons=True)
        assert np.array_equal(Tc1[0].view(np.uint32), Tc0[0].view(np.uint32)) and np.array_equal(Nc1[0], Nc0[0])
    else:
        Ta, Na, qa = run_gpu(rfa, w, w.steps, rfa.KERNEL_AUTO)
        assert qa["kernel"] == rfa.KERNEL_PLAIN     # falls back to the plain CUDA kernel, still on the GPU
        assert np.array_equal(Ta[0], Tp[0])
        with pytest.raises(rfa.RfaError):
            rfa.from_workload(w).configure(rfa.KERNEL_BLOCKED, 2)


TMA_CASES = [
    dict(dims=(144, 70, 21), spacing=(0.7, 0.9, 1.3), steps=37, mode=W.SRC_DIRICHLET, value=90.0, batch=1),   # 3 x 3 tiles of 64 x 32, ragged
    dict(dims=(80, 130, 19), spacing=(1.1, 0.8, 0.9), steps=41, mode=W.SRC_POWER, value=2.0e7, batch=1),       # partial x tile, 5-6 y tiles
    dict(dims=(16, 38, 29), spacing=(1.0, 1.0, 1.0), steps=50, mode=W.SRC_DIRICHLET, value=60.0, batch=1),     # narrower than a tile
    dict(dims=(272, 34, 7), spacing=(0.7, 0.9, 1.3), steps=20, mode=W.SRC_DIRICHLET, value=90.0, batch=1),     # 5 x tiles, few planes
    dict(dims=(64, 66, 23), spacing=(1.0, 1.0, 1.2), steps=33, mode=W.SRC_DIRICHLET, value=90.0, batch=3),     # batched
]


@pytest.mark.parametrize("case", TMA_CASES, ids=lambda c: "x".join(map(str, c["dims"])) + f"b{c['batch']}")
def test_blocked_tma_staging_bit_identity(rfa, case):
    """The temporally blocked kernel with its level-0 planes staged by the Tensor Memory Accelerator (RFA_STAGING_TMA: one
    cp.async.bulk.tensor per tile plane, zero-filled outside the grid, replicate rule at the outer y faces by exchange
    index) against the plain kernel, bit for bit: 2 and 3 fused steps, both tile shapes, both held-copy settings."""
    w = W.ragged_phantom(dims=case["dims"], spacing=case["spacing"], steps=case["steps"], mode=case["mode"],
                         value=case["value"], q_m=10714.0, dt=0.05, batch=case["batch"])
    w.table["t_init"][W.KIDNEY] = 36.0
    Tp, Np, qp = run_gpu(rfa, w, w.steps, rfa.KERNEL_PLAIN)
    for fused in (2, 3):
        for shape in (0, 1):
            for hc in (0, 1):
                sim = rfa.from_workload(w)
                sim.configure(rfa.KERNEL_BLOCKED, fused)
                sim.configure_tile(shape)
                sim.configure_staging(rfa.STAGING_TMA)
                sim.configure_held_copy(hc)
                sim.configure_residual_prefetch(rfa.RES_PREFETCH_ON if hc else rfa.RES_PREFETCH_OFF)   # exists with TMA staging at 2 fused steps
                v = sim.query_variant()
                assert v["residual_prefetch"] == (1 if hc and fused == 2 else 0)
                assert v["staging"] == rfa.STAGING_TMA and v["fused_steps"] == fused and v["held_copy"] == hc
                assert (v["tile_bx"], v["tile_by"]) == ((64, 32), (128, 16))[shape]
                sim.step(w.steps)
                for b in range(w.batch):
                    T, N = sim.get_temperature(b), sim.get_necrosis(b)
                    assert np.array_equal(T.view(np.uint32), Tp[b].view(np.uint32)), \
                        f"TMA-staged blocked kernel differs from plain (fused {fused}, shape {shape}, hc {hc}, scenario {b})"
                    assert np.array_equal(N, Np[b])
                sim.close()
    # default staging: TMA with the 128 x 16 tile, cp.async with the 64 x 32 tile; both can be forced
    sim = rfa.from_workload(w)
    sim.configure(rfa.KERNEL_BLOCKED, 3)
    v = sim.query_variant()
    assert v["staging"] == (rfa.STAGING_TMA if v["tile_bx"] == 128 else rfa.STAGING_CP_ASYNC)
    sim.configure_staging(rfa.STAGING_CP_ASYNC)
    assert sim.query_variant()["staging"] == rfa.STAGING_CP_ASYNC
    sim.step(w.steps)
    assert np.array_equal(sim.get_temperature(0).view(np.uint32), Tp[0].view(np.uint32))
    sim.close()
    # no TMA variant: odd ny, nx % 16 != 0
    for dims in ((272, 33, 5), (136, 70, 21)):
        sim = rfa.from_workload(W.ragged_phantom(dims=dims, steps=3))
        sim.configure(rfa.KERNEL_BLOCKED, 3)
        assert sim.query_variant()["staging"] == rfa.STAGING_CP_ASYNC
        with pytest.raises(rfa.RfaError):
            sim.configure_staging(rfa.STAGING_TMA)
        sim.close()


STREAM_CASES = [
    dict(dims=(144, 70, 21), spacing=(0.7, 0.9, 1.3), steps=37, mode=W.SRC_DIRICHLET, value=90.0, batch=1),   # 2 x 3 tiles, ragged
    dict(dims=(80, 130, 19), spacing=(1.1, 0.8, 0.9), steps=41, mode=W.SRC_POWER, value=2.0e7, batch=1),       # partial x tile
    dict(dims=(16, 38, 29), spacing=(1.0, 1.0, 1.0), steps=50, mode=W.SRC_DIRICHLET, value=60.0, batch=1),     # narrower than a tile
    dict(dims=(272, 33, 5), spacing=(0.7, 0.9, 1.3), steps=20, mode=W.SRC_DIRICHLET, value=90.0, batch=1),     # 3 x tiles, 1-row tail
    dict(dims=(64, 66, 23), spacing=(1.0, 1.0, 1.2), steps=33, mode=W.SRC_DIRICHLET, value=90.0, batch=5),     # batched
]


@pytest.mark.parametrize("case", STREAM_CASES, ids=lambda c: "x".join(map(str, c["dims"])) + f"b{c['batch']}")
def test_stream_kernel_parity_and_bit_identity(rfa, oracle, case):
    """The TMA-staged one-step kernel (RFA_KERNEL_STREAM: cp.async.bulk.tensor tiles with halos, mbarrier ring) against the
    oracle and, bit for bit, against the plain kernel; both held-copy settings; also as the remainder launch of S = 3."""
    w = W.ragged_phantom(dims=case["dims"], spacing=case["spacing"], steps=case["steps"], mode=case["mode"],
                         value=case["value"], q_m=10714.0, dt=0.05, batch=case["batch"])
    w.table["t_init"][W.KIDNEY] = 36.0
    Tp, Np, qp = run_gpu(rfa, w, w.steps, rfa.KERNEL_PLAIN)
    for hc in (0, 1):
        sim = rfa.from_workload(w)
        sim.configure(rfa.KERNEL_STREAM, 1)
        sim.configure_held_copy(hc)
        q = sim.query()
        assert q["kernel"] == rfa.KERNEL_STREAM and q["fused_steps"] == 1
        v = sim.query_variant()
        assert (v["tile_bx"], v["tile_by"], v["held_copy"]) == (128, 16, hc)
        sim.step(w.steps)
        for b in range(w.batch):
            T, N = sim.get_temperature(b), sim.get_necrosis(b)
            assert np.array_equal(T.view(np.uint32), Tp[b].view(np.uint32)), f"stream kernel differs from plain (scenario {b}, hc {hc})"
            assert np.array_equal(N, Np[b])
        sim.close()
    for b in range(w.batch):
        compare(Tp[b], Np[b], oracle.run_workload(w, scenario=b))
    # default configuration: launches of 3 fused steps, a remainder of ONE step goes to the one-step kernel
    if w.steps % 3 == 1:
        Ta, Na, qa = run_gpu(rfa, w, w.steps, rfa.KERNEL_AUTO, 3)
        assert np.array_equal(Ta[0].view(np.uint32), Tp[0].view(np.uint32)) and np.array_equal(Na[0], Np[0])
    # not available: nx % 16 != 0, conservative conduction
    w2 = W.ragged_phantom(dims=(136, 70, 21), steps=3)
    sim = rfa.from_workload(w2)
    with pytest.raises(rfa.RfaError):
        sim.configure(rfa.KERNEL_STREAM, 1)
    sim.configure(rfa.KERNEL_AUTO, 1)
    assert sim.query()["kernel"] == rfa.KERNEL_BLOCKED
    sim.close()
    sim = rfa.from_workload(w)
    sim.set_conduction(rfa.COND_FACE)
    with pytest.raises(rfa.RfaError):
        sim.configure(rfa.KERNEL_STREAM, 1)
    sim.configure(rfa.KERNEL_AUTO, 1)
    assert sim.query()["kernel"] == rfa.KERNEL_BLOCKED
    sim.close()


def test_batched_scenarios(rfa, oracle):
    w = W.ragged_phantom(dims=(68, 66, 23), spacing=(1.0, 1.0, 1.2), steps=33, batch=5, dt=0.08)
    T, N, q = run_gpu(rfa, w, w.steps, rfa.KERNEL_BLOCKED, 2)
    Tp, Np, _ = run_gpu(rfa, w, w.steps, rfa.KERNEL_PLAIN)
    for b in range(w.batch):
        osim = oracle.run_workload(w, scenario=b)
        compare(T[b], N[b], osim)
        assert np.array_equal(T[b], Tp[b]) and np.array_equal(N[b], Np[b])
    assert not np.array_equal(T[0], T[1])       # the scenarios really differ


def test_needle_semantics(rfa, oracle):
    """Override (R-15), release (R-16), sticky necrosis (R-12), inclusive threshold (R-11), counts (R-13)."""
    n = 12
    lab = np.ones((n, n, n), np.uint8)
    lab[4, 4, 5] = W.VESSEL
    table = W.tissue_table()
    m1 = np.zeros((n, n, n), np.uint8)
    m1[4, 4, 4] = 1
    m1[4, 4, 5] = 1
    m2 = np.zeros((n, n, n), np.uint8)
    m2[1, 1, 1] = 1
    osim = oracle.OracleSim((n, n, n), (1.0, 1.0, 1.0), lab, table, 37.0, 0.1)
    sim = rfa.RfaSim((n, n, n), (1.0, 1.0, 1.0), lab, table, 37.0, 0.1)
    for s in (osim,):
        s.set_needle(m1, W.SRC_DIRICHLET, 90.0)
    sim.set_needle(0, m1, rfa.SRC_DIRICHLET, 90.0)
    osim.step(200)
    sim.step(200)
    compare(sim.get_temperature(0), sim.get_necrosis(0), osim)
    osim.set_needle(m2, W.SRC_DIRICHLET, 59.9995)
    sim.set_needle(0, m2, rfa.SRC_DIRICHLET, 59.9995)
    osim.step(1)
    sim.step(1)
    T = sim.get_temperature(0)
    assert T[4, 4, 5] == 90.0 and T[4, 4, 4] < 90.0 and abs(T[1, 1, 1] - 59.9995) < 1e-5
    osim.step(1500)
    sim.step(1500)
    compare(sim.get_temperature(0), sim.get_necrosis(0), osim)
    N = sim.get_necrosis(0)
    assert N[1, 1, 1] == 0 and N[4, 4, 4] == 1
    all_v, tissue_v = sim.necrotic_voxels(0)
    assert all_v == int(N.sum())
    held_or_needle = ((table["flags"][lab] & 1) != 0) | (m2 != 0)
    assert tissue_v == int((N != 0)[~held_or_needle].sum())
    sim.set_needle(0, None, rfa.SRC_OFF, 0.0)
    osim.set_needle(None, W.SRC_OFF, 0.0)
    sim.step(3)
    osim.step(3)
    compare(sim.get_temperature(0), sim.get_necrosis(0), osim)
    sim.close()


def test_edge_cases(rfa, oracle):
    table = W.tissue_table()
    # zero steps, 1x1x1, tiny grids, single plane
    for dims in ((1, 1, 1), (4, 4, 4), (8, 3, 2), (64, 64, 4), (4, 70, 9)):
        nx, ny, nz = dims
        rng = np.random.default_rng(nx * 100 + ny * 10 + nz)
        lab = rng.integers(0, 7, size=(nz, ny, nx)).astype(np.uint8)
        T0 = (37.0 + 30.0 * rng.random((nz, ny, nx))).astype(np.float32)
        osim = oracle.OracleSim(dims, (1.0, 0.8, 1.2), lab, table, 37.0, 0.05)
        osim.set_temperature(T0.astype(np.float64))
        sim = rfa.RfaSim(dims, (1.0, 0.8, 1.2), lab, table, 37.0, 0.05)
        sim.set_temperature(0, T0)
        sim.step(0)
        assert np.max(np.abs(sim.get_temperature(0) - T0)) < 4e-6      # theta = T - 37 round trip
        sim.step(13)
        osim.step(13)
        compare(sim.get_temperature(0), sim.get_necrosis(0), osim)
        sim.close()
    with pytest.raises(rfa.RfaError):
        rfa.RfaSim((4, 4, 4), (1, 1, 1), np.full((4, 4, 4), 9, np.uint8), table, 37.0, 0.1)
    with pytest.raises(rfa.RfaError) as ei:
        rfa.RfaSim((4, 4, 4), (0.5, 0.5, 0.5), np.ones((4, 4, 4), np.uint8), table, 37.0, 0.4)
    assert ei.value.code == rfa.RFA_E_UNSTABLE
    sim = rfa.RfaSim((4, 4, 4), (1, 1, 1), np.ones((4, 4, 4), np.uint8), table, 37.0, 0.1, batch=2)
    with pytest.raises(rfa.RfaError):
        sim.get_temperature(2)
    with pytest.raises(rfa.RfaError):
        sim.step(-1)
    sim.close()


def test_device_pointers_are_accepted(rfa):
    import torch
    w = W.ragged_phantom(dims=(44, 38, 29), steps=20)
    sim = rfa.from_workload(w)
    sim.step(20)
    host = sim.get_temperature(0)
    dev = torch.empty(host.shape, dtype=torch.float32, device="cuda")
    sim.get_temperature(0, out=dev)
    assert np.array_equal(dev.cpu().numpy(), host)
    ndev = torch.empty(host.shape, dtype=torch.uint8, device="cuda")
    sim.get_necrosis(0, out=ndev)
    assert np.array_equal(ndev.cpu().numpy(), sim.get_necrosis(0))
    # device-resident mask and temperature inputs
    sim2 = rfa.RfaSim(w.dims, w.spacing_mm, w.labels, w.table, w.t_blood, w.dt)
    sim2.set_needle(0, torch.from_numpy(w.needles[0].mask).cuda(), w.needles[0].mode, w.needles[0].value)
    sim2.step(20)
    assert np.array_equal(sim2.get_temperature(0), host)
    sim2.set_temperature(0, dev)
    assert np.max(np.abs(sim2.get_temperature(0) - host)) < 4e-6
    sim.close()
    sim2.close()


# ----------------------------------------------------------------------------------------------
# C1 (BASELINE configs[0]) incl. the Green's function variant, and invariants on the GPU field
# ----------------------------------------------------------------------------------------------
def test_c1_cube_and_green(rfa, oracle):
    w = W.c1_cube()
    osim = oracle.run_workload(w)
    T, N, q = run_gpu(rfa, w, w.steps)
    assert q["kernel"] == rfa.KERNEL_BLOCKED
    err, _ = compare(T[0], N[0], osim)
    # 48-fold symmetry survives fp32 exactly for the axis flips about the tip on this grid
    c = 32
    assert T[0][c, c, c + 3] == T[0][c, c, c - 3] == T[0][c + 3, c, c] == T[0][c, c - 3, c]
    wg = W.c1_green(n=64, h_mm=1.0, dt=0.1, steps=1000)
    og = oracle.run_workload(wg)
    Tg, Ng, _ = run_gpu(rfa, wg, wg.steps)
    # the delta start (37 + 1e4 C) has ulp(1e4) = 1e-3 C at t = 0; the compensated accumulation
    # carries what the first steps round away, so the smooth field after 1000 steps meets north_star's bar as it stands
    err_g, _ = compare(Tg[0], Ng[0], og, tol=TOL)
    # energy conservation on the GPU field (zero flux, no perfusion): sum(theta) constant
    e_rel = abs((Tg[0].astype(np.float64) - 37.0).sum() - 1.0e4) / 1.0e4
    print(f"C1 Green: max|dT| {err_g:.2e} C after {wg.steps} steps, energy drift {e_rel:.2e} relative")
    assert e_rel < 2e-6


def test_monotone_and_bounded_on_gpu(rfa):
    w = W.c2_phantom(steps=0)
    sim = rfa.from_workload(w)
    prev = sim.get_temperature(0)
    prev_n = sim.necrotic_voxels(0)[0]
    for _ in range(6):
        sim.step(50)
        cur = sim.get_temperature(0)
        assert np.all(cur >= prev)                       # PAPER.md:83,:159 (fp32: exact here, monotone map)
        assert cur.min() >= 37.0 and cur.max() <= 90.0
        n = sim.necrotic_voxels(0)[0]
        assert n >= prev_n
        prev, prev_n = cur, n
    sim.close()


def test_held_copy_variant_is_bit_identical(rfa):
    """Warps of held voxels only copy their rows (Alg. 1's else-branch): same bits as evaluating the bracket."""
    w = W.ragged_phantom(dims=(136, 70, 21), spacing=(0.7, 0.9, 1.3), steps=33, dt=0.05)
    res = {}
    for hc in ("0", "1"):
        sim = rfa.from_workload(w)
        sim.configure(rfa.KERNEL_BLOCKED, 3)
        sim.configure_held_copy(int(hc))
        assert sim.query_variant()["held_copy"] == int(hc) and sim.query_variant()["tile_bx"] in (64, 128)
        sim.step(w.steps)
        res[hc] = (sim.get_temperature(0), sim.get_necrosis(0))
        sim.close()
    assert np.array_equal(res["0"][0].view(np.uint32), res["1"][0].view(np.uint32))
    assert np.array_equal(res["0"][1], res["1"][1])
    # a body in air: whole tile planes are held (the CTA-wide shortcut), others are cut by the body surface
    nx, ny, nz = 200, 136, 24
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    rr = ((i - 120) / 60.0) ** 2 + ((j - 70) / 40.0) ** 2 + ((k - 11) / 9.0) ** 2
    lab = np.full((nz, ny, nx), W.EXTERIOR, np.uint8)
    lab[rr < 1.0] = W.FAT
    lab[rr < 0.5] = W.LIVER
    lab[(rr < 0.5) & (np.abs(j - 62) < 3) & (np.abs(k - 9) < 3)] = W.VESSEL
    mask = np.zeros_like(lab)
    mask[11, 70, 108:132] = 1
    body = {}
    for hc in ("0", "1"):
        for fused in (3, 2):
            sim = rfa.RfaSim((nx, ny, nz), (0.9, 0.9, 1.2), lab, W.tissue_table(), 37.0, 0.05)
            sim.configure(rfa.KERNEL_BLOCKED, fused)
            sim.configure_held_copy(int(hc))
            sim.set_needle(0, mask, rfa.SRC_DIRICHLET, 90.0)
            sim.step(40)
            body[(hc, fused)] = (sim.get_temperature(0), sim.get_necrosis(0))
            sim.close()
    ref = body[("0", 3)]
    assert float(ref[0].max()) == 90.0 and float(ref[0][11, 71, 110]) > 37.5
    for key, (T, N) in body.items():
        assert np.array_equal(T.view(np.uint32), ref[0].view(np.uint32)) and np.array_equal(N, ref[1]), key
    # blood at 59.6 C: the necrosis threshold (0.4 C above T_a) lies BELOW the 1 C bound of the cold paths, so the copied rows'
    # maxima matter to the necrosis filter (exterior held at 60.2 C: necrotic from the start; vessels at 59.6 C: not)
    tab = W.tissue_table()
    tab["t_init"][:] = 59.6
    tab["t_init"][W.EXTERIOR] = 60.2
    warm = {}
    for kern, fused, hc in ((rfa.KERNEL_PLAIN, 1, 0), (rfa.KERNEL_BLOCKED, 3, 1), (rfa.KERNEL_BLOCKED, 2, 1), (rfa.KERNEL_BLOCKED, 1, 1)):
        sim = rfa.RfaSim((nx, ny, nz), (0.9, 0.9, 1.2), lab, tab, 59.6, 0.05)
        sim.configure(kern, fused)
        if kern != rfa.KERNEL_PLAIN:
            sim.configure_held_copy(hc)
        sim.set_needle(0, mask, rfa.SRC_DIRICHLET, 90.0)
        sim.step(20)
        warm[(kern, fused)] = (sim.get_temperature(0), sim.get_necrosis(0))
        sim.close()
    ref = warm[(rfa.KERNEL_PLAIN, 1)]
    assert ref[1][0, 0, 0] == 1 and 0 < int(ref[1].sum()) < ref[1].size
    for key, (T, N) in warm.items():
        assert np.array_equal(T.view(np.uint32), ref[0].view(np.uint32)) and np.array_equal(N, ref[1]), key
    sim = rfa.from_workload(W.c1_cube())                      # no held label at all: the plain variant is chosen
    assert sim.query_variant()["held_copy"] == 0
    sim.configure_held_copy(rfa.HELD_COPY_ON)
    assert sim.query_variant()["held_copy"] == 1
    sim.configure_held_copy(rfa.HELD_COPY_AUTO)
    assert sim.query_variant()["held_copy"] == 0
    with pytest.raises(rfa.RfaError):
        sim.configure_held_copy(7)
    sim.close()
    os.environ["RFA_HELD_COPY"] = "1"                         # the library reads no environment variable
    try:
        sim = rfa.from_workload(W.c1_cube())
        assert sim.query_variant()["held_copy"] == 0
        sim.close()
    finally:
        del os.environ["RFA_HELD_COPY"]


# ----------------------------------------------------------------------------------------------
# f1: conservative conduction (harmonic-mean face conductivities, R-28)
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", RAGGED[:3], ids=lambda c: "x".join(map(str, c["dims"])))
def test_conservative_conduction_parity_and_variants(rfa, oracle, case):
    w = W.ragged_phantom(dims=case["dims"], spacing=case["spacing"], steps=case["steps"], dt=0.05,
                         mode=case["mode"], value=case["value"])
    osim = oracle.run_workload(w, conservative=True)
    plain = oracle.run_workload(w, conservative=False)
    assert np.max(np.abs(osim.T - plain.T)) > 1e-2           # the two conduction terms really differ here
    results = []
    for kernel, fused in [(rfa.KERNEL_PLAIN, 0), (rfa.KERNEL_BLOCKED, 1), (rfa.KERNEL_BLOCKED, 2),
                          (rfa.KERNEL_BLOCKED, 3), (rfa.KERNEL_BLOCKED, 4)]:
        sim = rfa.from_workload(w)
        sim.configure(kernel, fused)
        sim.set_conduction(rfa.COND_FACE)
        sim.step(w.steps)
        T, N = sim.get_temperature(0), sim.get_necrosis(0)
        sim.close()
        compare(T, N, osim)
        results.append((T, N))
    for T, N in results[1:]:
        assert np.array_equal(T.view(np.uint32), results[0][0].view(np.uint32)) and np.array_equal(N, results[0][1])


def test_conservative_three_k_stacks_at_the_outer_faces(rfa, oracle):
    """Random mix of three conductivities right up to the grid faces: the blocked kernel loads MIRRORED y/z halos
    there, which is only exact because rfa_face_correction is bit-symmetric under swapping the two sides of an axis.
    All fused depths must reproduce the plain kernel bit for bit, and the oracle to the bar."""
    dims = (72, 40, 18)
    rng = np.random.default_rng(23)
    table = W.make_table([(0.21, 911.0, 2348.0, 500.0, 0, 37.0, 0), (0.512, 1060.0, 3600.0, 24000.0, 0, 37.0, 0),
                          (1.3, 1050.0, 3700.0, 0, 0, 37.0, 0)])
    lab = (rng.random((18, 40, 72)) * 3).astype(np.uint8)
    T0 = (37.0 + 40.0 * rng.random((18, 40, 72))).astype(np.float32)
    osim = oracle.OracleSim(dims, (0.9, 1.1, 1.3), lab, table, 37.0, 0.04, conservative=True)
    osim.set_temperature(T0.astype(np.float64))
    osim.step(24)
    res = []
    for kernel, fused in [(rfa.KERNEL_PLAIN, 0), (rfa.KERNEL_BLOCKED, 1), (rfa.KERNEL_BLOCKED, 2),
                          (rfa.KERNEL_BLOCKED, 3), (rfa.KERNEL_BLOCKED, 4)]:
        sim = rfa.RfaSim(dims, (0.9, 1.1, 1.3), lab, table, 37.0, 0.04)
        sim.configure(kernel, fused)
        sim.set_conduction(rfa.COND_FACE)
        sim.set_temperature(0, T0)
        sim.step(24)
        res.append((sim.get_temperature(0), sim.get_necrosis(0)))
        sim.close()
    compare(res[0][0], res[0][1], osim)
    for T, N in res[1:]:
        assert np.array_equal(T.view(np.uint32), res[0][0].view(np.uint32)) and np.array_equal(N, res[0][1])


def test_conservative_conduction_conserves_energy_on_gpu(rfa):
    """sum rho c_p T constant (no perfusion, no sources, nothing held) to fp32 round-off."""
    dims = (72, 40, 18)
    rng = np.random.default_rng(5)
    table = W.make_table([(0.21, 911.0, 2348.0, 0, 0, 37.0, 0), (0.512, 1060.0, 3600.0, 0, 0, 37.0, 0),
                          (0.53, 1050.0, 3700.0, 0, 0, 37.0, 0)])
    lab = (rng.random((18, 40, 72)) * 3).astype(np.uint8)
    lab[:, :, 36:] = 1                                        # half random mix, half homogeneous
    T0 = (37.0 + 30.0 * rng.random((18, 40, 72))).astype(np.float32)
    sim = rfa.RfaSim(dims, (0.9, 1.1, 1.3), lab, table, 37.0, 0.05)
    sim.set_conduction(rfa.COND_FACE)
    sim.set_temperature(0, T0)
    rc = (table["rho"].astype(np.float64) * table["cp"])[lab]
    e0 = float((rc * (T0.astype(np.float64) - 37.0)).sum())
    sim.step(300)
    T = sim.get_temperature(0).astype(np.float64)
    e1 = float((rc * (T - 37.0)).sum())
    assert abs(e1 - e0) / e0 < 2e-6 and np.ptp(T) < 0.7 * np.ptp(T0)
    sim.close()


# ----------------------------------------------------------------------------------------------
# f2: probe time series (Fig. 6, Fig. 14) and the Alg. 2 frame hand-off
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("every,fused", [(1, 3), (6, 3), (4, 2)])
def test_probe_series_matches_oracle(rfa, oracle, every, fused):
    w = W.paper_probe_case(90.0, steps=240)
    pr = W.fig6_probes(w.dims, w.spacing_mm, w.meta["centre_voxel"]).ravel()
    osim = oracle.OracleSim(w.dims, w.spacing_mm, w.labels, w.table, w.t_blood, w.dt)
    osim.set_needle(w.needles[0].mask, w.needles[0].mode, w.needles[0].value)
    exp = osim.step_record(w.steps, every, pr)
    sim = rfa.from_workload(w)
    sim.configure(rfa.KERNEL_BLOCKED, fused)
    sim.set_probes(pr)
    got = sim.step_record(w.steps, every)
    assert got.shape == exp.shape == (w.steps // every, 12)
    assert float(np.max(np.abs(got.astype(np.float64) - exp))) <= TOL
    assert np.all(np.diff(got, axis=0) >= 0.0)            # monotone convergence, also in fp32
    compare(sim.get_temperature(0), sim.get_necrosis(0), osim)   # the field itself after the recorded run
    # device output buffer, probes cleared afterwards
    import torch
    dev_out = torch.empty((2, 12), dtype=torch.float32, device="cuda")
    sim.step_record(2 * every, every, out=dev_out)
    assert np.all(dev_out.cpu().numpy()[-1] >= got[-1])
    sim.set_probes([])
    with pytest.raises(rfa.RfaError):
        sim.step_record(every, every)
    sim.close()


def test_frame_handoff_double_buffer(rfa):
    """Alg. 2: the finished image stays intact while the next launch runs into the
    other buffer, so a consumer on a second stream may read it concurrently."""
    import torch
    w = W.ragged_phantom(dims=(136, 70, 21), spacing=(0.7, 0.9, 1.3), steps=9, dt=0.05)
    sim = rfa.from_workload(w)
    sim.configure(rfa.KERNEL_BLOCKED, 3)
    sim.step(9)
    sim.synchronize()
    want = sim.get_temperature(0)
    ptr, t_blood = sim.current_frame(0)
    nx, ny, nz = w.dims
    side = torch.cuda.Stream()
    host = torch.empty(nx * ny * nz, dtype=torch.float32, pin_memory=True)
    sim.step(3)                                            # ONE more launch, asynchronous, writes the other buffer
    from cuda.bindings import runtime as cudart           # raw device pointer -> pinned host, on the side stream
    (rc,) = cudart.cudaMemcpyAsync(host.data_ptr(), ptr, host.numel() * 4,
                                   cudart.cudaMemcpyKind.cudaMemcpyDeviceToHost, side.cuda_stream)
    assert int(rc) == 0
    side.synchronize()
    sim.synchronize()
    frame = host.numpy().reshape(nz, ny, nx)
    assert np.array_equal((frame + np.float32(t_blood)).view(np.uint32), want.view(np.uint32))
    ptr2, _ = sim.current_frame(0)
    assert ptr2 != ptr                                     # the buffers were swapped by the launch
    sim.close()


# ----------------------------------------------------------------------------------------------
# f3: breathing-motion warp, Eq. 14
# ----------------------------------------------------------------------------------------------
def test_warp_matches_oracle_elementwise(rfa, oracle):
    from oracle import rfa_warp_oracle as WO
    w = W.ragged_phantom(dims=(136, 70, 21), spacing=(0.7, 0.9, 1.3), steps=40, dt=0.05)
    sim = rfa.from_workload(w)
    sim.step(w.steps)
    T = sim.get_temperature(0)                               # the fp32 image the warp reads (plus T_a)
    d = W.breathing_field(w.dims, amp_mm=(2.0, 4.0, 12.0))
    for scale in (0.0, 0.37, 1.0, -1.0, 40.0):               # 40: far outside the grid -> clamped everywhere
        got = sim.warp_temperature(0, d, scale)
        exp = WO.warp_temperature(T, d, np.float32(scale), w.spacing_mm)
        # tolerance: fp32 interpolation weights (2^-24 relative on a displacement of <= 20 voxels ~ 2e-6 voxel)
        # times the steepest gradient in the image (53 C per voxel at the needle) + fp32 rounding of the result
        assert float(np.max(np.abs(got.astype(np.float64) - exp))) <= TOL
    assert np.array_equal(sim.warp_temperature(0, d, 0.0).view(np.uint32), T.view(np.uint32))
    import torch
    dd, od = torch.from_numpy(d).cuda(), torch.empty(T.shape, dtype=torch.float32, device="cuda")
    sim.warp_temperature(0, dd, 1.0, out=od)                 # device in, device out
    assert np.array_equal(od.cpu().numpy(), sim.warp_temperature(0, d, 1.0))
    assert np.array_equal(sim.get_temperature(0).view(np.uint32), T.view(np.uint32))   # state untouched
    sim.close()


def test_warp_full_size_sampled(rfa):
    """C4 size: sampled voxels near the needle first (a quick, pointed failure), then the whole field against the oracle."""
    from oracle import rfa_warp_oracle as WO
    w = W.c4_body(steps=300)
    sim = rfa.from_workload(w)
    sim.step(300)
    T = sim.get_temperature(0)
    d = W.breathing_field(w.dims)
    got = sim.warp_temperature(0, d, 0.85)
    rng = np.random.default_rng(11)
    mz, my, mx = np.nonzero(w.needles[0].mask)
    nx, ny, nz = w.dims
    pick = rng.integers(0, len(mz), 200)
    near = (np.clip(mx[pick] + rng.integers(-6, 7, 200), 0, nx - 1)
            + nx * (np.clip(my[pick] + rng.integers(-6, 7, 200), 0, ny - 1)
                    + ny * np.clip(mz[pick] + rng.integers(-12, 13, 200), 0, nz - 1)))
    idx = np.unique(np.concatenate([near, rng.integers(0, nx * ny * nz, 4000)]))
    exp = WO.warp_temperature(T, d, np.float32(0.85), w.spacing_mm, index=idx)
    assert float(np.max(np.abs(got.ravel()[idx].astype(np.float64) - exp))) <= TOL
    assert got.min() >= T.min() and got.max() <= T.max()
    assert float(np.abs(got - T).max()) > 1.0                # the heat zone really moved
    # and EVERY voxel of the 67 M: the oracle is vectorised numpy, fed 16 z planes at a time through its `index` path
    worst = 0.0
    gflat = got.ravel()
    for k0 in range(0, nz, 16):
        sl = np.arange(k0 * nx * ny, min(k0 + 16, nz) * nx * ny, dtype=np.int64)
        e = WO.warp_temperature(T, d, np.float32(0.85), w.spacing_mm, index=sl)
        worst = max(worst, float(np.max(np.abs(gflat[sl].astype(np.float64) - e))))
    assert worst <= TOL, f"warp, whole field: max |dT| = {worst:.3e}"
    print(f"warp C4: field max|dT| {worst:.2e} over all {got.size} voxels")
    sim.close()


# ----------------------------------------------------------------------------------------------
# f4: headless view of the heat zone (orthographic ray-march; Figs. 11-12)
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("direction,up", [((0, 0, 1), (0, 1, 0)), ((1, 2, 3), (0, 1, 0)), ((-2, 1, 0.5), (0, 0, 1))])
def test_render_zone_matches_oracle(rfa, direction, up):
    from oracle import rfa_render_oracle as RO
    w = W.c2_phantom(steps=900)
    sim = rfa.from_workload(w)
    sim.step(w.steps)
    T = sim.get_temperature(0)
    Wp, Hp = 96, 80
    tmax, depth = sim.render_zone(0, direction, up, Wp, Hp, 1.25, 0.5, iso_c=42.5)
    etmax, edepth, margin = RO.render_zone(T, w.spacing_mm, direction, up, Wp, Hp, 1.25, 0.5, 42.5, t_blood=w.t_blood)
    assert float(np.max(np.abs(tmax.astype(np.float64) - etmax))) <= TOL
    # first-hit decisions: identical wherever no sample of the ray lies within the band of the isotherm
    clear = margin > BAND
    assert np.array_equal(depth[clear] >= 0, edepth[clear] >= 0)
    assert float(np.max(np.abs(depth[clear].astype(np.float64) - edepth[clear]))) <= 1e-4
    assert int((~clear).sum()) < 0.02 * Wp * Hp and int((edepth >= 0).sum()) > 50      # a zone is visible
    t2, none = sim.render_zone(0, direction, up, Wp, Hp, 1.25, 0.5, want_depth=False)
    assert none is None and np.array_equal(t2, tmax)
    with pytest.raises(rfa.RfaError):
        sim.render_zone(0, (0, 0, 0), up, Wp, Hp, 1.25, 0.5)
    with pytest.raises(rfa.RfaError):
        sim.render_zone(0, up, up, Wp, Hp, 1.25, 0.5)
    sim.close()


def test_render_zone_image_sizes_around_the_old_staging_limit(rfa):
    """Host images are staged in a library-owned buffer that grows on demand: any W*H works, also above half the
    voxel count of a small volume (where the former scratch-volume staging made tmax and depth overlap)."""
    from oracle import rfa_render_oracle as RO
    w = W.ragged_phantom(dims=(44, 38, 29), spacing=(1.0, 1.0, 1.0), steps=40, dt=0.05)
    sim = rfa.from_workload(w)
    sim.step(w.steps)
    T = sim.get_temperature(0)
    nvox = w.n_voxels
    for Wp, Hp in [(150, 161), (154, 158), (168, 168), (256, 200)]:      # below, just above, above nvox/2; above nvox
        assert (Wp * Hp > nvox // 2) == ((Wp, Hp) != (150, 161))
        tmax, depth = sim.render_zone(0, (1, 2, 3), (0, 1, 0), Wp, Hp, 0.4, 0.5, iso_c=42.5)
        etmax, edepth, margin = RO.render_zone(T, w.spacing_mm, (1, 2, 3), (0, 1, 0), Wp, Hp, 0.4, 0.5, 42.5, t_blood=w.t_blood)
        assert float(np.max(np.abs(tmax.astype(np.float64) - etmax))) <= TOL
        clear = margin > BAND
        assert np.array_equal(depth[clear] >= 0, edepth[clear] >= 0)
        assert float(np.max(np.abs(depth[clear].astype(np.float64) - edepth[clear]))) <= 1e-4
        assert int((edepth >= 0).sum()) > 50
    sim.close()


def test_boundary_validation_on_a_live_simulation(rfa):
    """rfa_set_needle validates its metadata: tip inside the grid, unit axis."""
    import torch
    w = W.ragged_phantom(dims=(44, 38, 29), spacing=(1.0, 1.0, 1.0), steps=5)
    sim = rfa.from_workload(w)
    nd = w.needles[0]
    for tip in [(-0.5, 10.0, 10.0), (10.0, 38.5, 10.0), (10.0, 10.0, float("nan"))]:
        with pytest.raises(rfa.RfaError) as ei:
            sim.set_needle(0, nd.mask, nd.mode, nd.value, tip, nd.axis)
        assert ei.value.code == rfa.RFA_E_INVALID
    for axis in [(0.0, 0.0, 1.1), (0.0, 0.0, 0.0), (0.6, 0.6, 0.6)]:
        with pytest.raises(rfa.RfaError) as ei:
            sim.set_needle(0, nd.mask, nd.mode, nd.value, nd.tip_mm, axis)
        assert ei.value.code == rfa.RFA_E_INVALID
    sim.set_needle(0, nd.mask, nd.mode, nd.value, (44.0, 0.0, 29.0), (0.6, 0.0, 0.8))    # on the faces: inside
    sim.set_needle(0, nd.mask, nd.mode, nd.value, None, None)
    # the simulation stays on its own device whatever the caller's current device is (single-GPU box: device 0),
    # and host displacement fields go through the library-owned staging buffer call after call
    sim.step(5)
    d = W.breathing_field(w.dims)
    a = sim.warp_temperature(0, d, 0.5)
    b = sim.warp_temperature(0, d, 0.5)
    assert np.array_equal(a, b)
    if torch.cuda.device_count() > 1:
        T0 = sim.get_temperature(0)
        with torch.cuda.device(1):
            sim.step(3)
            T1 = sim.get_temperature(0)
        assert not np.array_equal(T0, T1)
    # output buffers are checked by the binding before their raw address reaches the library
    with pytest.raises(ValueError):
        sim.get_temperature(0, out=np.empty(w.n_voxels - 1, np.float32))
    with pytest.raises(ValueError):
        sim.get_temperature(0, out=np.empty(w.n_voxels, np.float64))
    with pytest.raises(ValueError):
        sim.render_zone(0, (0, 0, 1), (0, 1, 0), 16, 16, 1.0, 1.0, tmax=np.empty((16, 32), np.float32)[:, ::2])
    with pytest.raises(ValueError):
        sim.render_zone(0, (0, 0, 1), (0, 1, 0), 16, 16, 1.0, 1.0, depth=torch.empty(255, dtype=torch.float32, device="cuda"))
    sim.set_probes([0, 1, 2])
    with pytest.raises(ValueError):
        sim.step_record(4, 2, out=np.empty((2, 2), np.float32))
    sim.close()
    # a label id outside the tissue table is found by the device histogram of rfa_create (no host walk when a device is there)
    wbad = W.ragged_phantom(dims=(44, 38, 29), spacing=(1.0, 1.0, 1.0), steps=5)
    wbad.labels = wbad.labels.copy()
    wbad.labels[7, 11, 13] = len(wbad.table)
    with pytest.raises(rfa.RfaError) as ei:
        rfa.from_workload(wbad)
    assert ei.value.code == rfa.RFA_E_INVALID and "label" in str(ei.value)
    # a forced tile shape that cannot run is refused under every kernel setting but PLAIN (nx % 4 != 0: no blocked plan)
    sim = rfa.from_workload(W.ragged_phantom(dims=(45, 38, 29), spacing=(0.7, 0.9, 1.3), steps=3))
    for shape in (0, 1):
        with pytest.raises(rfa.RfaError) as ei:
            sim.configure_tile(shape)
        assert ei.value.code == rfa.RFA_E_INVALID
    sim.configure_tile(-1)
    sim.configure(rfa.KERNEL_PLAIN, 0)
    sim.configure_tile(1)
    sim.step(3)
    sim.close()


# ----------------------------------------------------------------------------------------------
# Full-length configs against the stored oracle results (tests/golden/, written by make_golden.py)
# ----------------------------------------------------------------------------------------------
def _golden(name):
    path = os.path.join(GOLDEN, f"{name}_golden.npz")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated yet")
    return np.load(path)


def _check_against_golden(g, prefix, T, N, dims, idx_cp=-1):
    nx, ny, nz = dims
    idx = g[prefix + "sample_idx"]
    exp = g[prefix + "sample_T"][idx_cp]
    err = float(np.max(np.abs(T.ravel()[idx].astype(np.float64) - exp)))
    assert err <= TOL, f"sampled max |dT| = {err:.3e}"
    return err


def _check_final_golden(g, prefix, T, N):
    lo = g[prefix + "crop_lo"]
    cT = g[prefix + "crop_T"]
    c = cT.shape[0]
    sub = T[lo[0]:lo[0] + c, lo[1]:lo[1] + c, lo[2]:lo[2] + c].astype(np.float64)
    err = float(np.max(np.abs(sub - cT)))
    assert err <= TOL, f"crop max |dT| = {err:.3e}"
    No = np.unpackbits(g[prefix + "necro_packed"])[:N.size].reshape(N.shape)
    mism = np.nonzero((N != 0).ravel() != (No != 0).ravel())[0]
    band = g[prefix + "band_idx"][np.abs(g[prefix + "band_T"] - 60.0) <= BAND]
    bad = np.setdiff1d(mism, band)
    assert bad.size == 0, f"{bad.size} necrosis mismatches outside the band"
    assert abs(float(T.astype(np.float64).max()) - float(g[prefix + "T_max"])) <= TOL
    return err, int(mism.size)


def _check_field_golden(g, prefix, T, w):
    """The WHOLE field against the oracle (make_golden.compact_field): inside the stored box the oracle's value is
    known to field_q / 2, outside it lies within field_outside_max of T_init = t_init[label]; both margins are taken
    off the tolerance, so passing proves |T - T_oracle| <= TOL at every voxel."""
    if prefix + "field_codes" not in g:
        pytest.fail(f"golden file lacks the compact field ({prefix}field_*): regenerate with tests/golden/make_golden.py")
    q = float(g[prefix + "field_q"])
    lo = g[prefix + "field_lo"]
    codes = g[prefix + "field_codes"]
    out_max = float(g[prefix + "field_outside_max"])
    dev = T.astype(np.float64) - np.asarray(w.table["t_init"], dtype=np.float64)[w.labels]
    bz, by, bx = codes.shape
    box = (slice(lo[0], lo[0] + bz), slice(lo[1], lo[1] + by), slice(lo[2], lo[2] + bx))
    err_in = float(np.max(np.abs(dev[box] - codes.astype(np.float64) * q)))
    assert err_in <= TOL - 0.5 * q, f"field max |dT| inside the stored box = {err_in:.3e}"
    dev[box] = 0.0
    err_out = float(np.max(np.abs(dev)))
    assert err_out <= TOL - out_max, f"far field max |T - T_init| = {err_out:.3e} (oracle: {out_max:.1e})"
    return max(err_in, err_out), int(codes.size)


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_full_length_config_vs_golden(rfa, name):
    g = _golden(name)
    w = W.BENCH_CONFIGS[name]()
    from tests.golden.make_golden import fingerprint
    assert fingerprint(w, 0) == str(g["fingerprint"]), "inputs differ from the ones the golden file was made from"
    sim = rfa.from_workload(w)                    # default configuration = what bench.py times
    done = 0
    for ci, cp in enumerate(g["checkpoints"]):
        sim.step(int(cp) - done)
        done = int(cp)
        T = sim.get_temperature(0)
        _check_against_golden(g, "", T, None, w.dims, ci)
    N = sim.get_necrosis(0)
    err, n_mism = _check_final_golden(g, "", T, N)
    err_f, n_box = _check_field_golden(g, "", T, w)            # every voxel of the volume
    all_v, tissue_v = sim.necrotic_voxels(0)
    assert abs(all_v - int(g["necro_count"])) <= n_mism and abs(tissue_v - int(g["necro_count_tissue"])) <= n_mism
    print(f"{name}: field max|dT| {err_f:.2e} over all {T.size} voxels ({n_box} in the stored box), crop {err:.2e}, "
          f"necrosis mismatches (all inside the band) {n_mism}, necrotic voxels {all_v} (oracle {int(g['necro_count'])})")
    sim.close()


def test_c4_conservative_conduction_vs_golden(rfa, oracle):
    """Row f1 at the full C4 size, in the default launch configuration: sampled voxels (needle region, uniform,
    tissue interfaces) at three checkpoints and the crop at the needle against the conservative fp64 oracle."""
    g = _golden("C4F")
    w = W.c4_face_case()
    from tests.golden.make_golden import fingerprint
    assert fingerprint(w, 0) == str(g["fingerprint"])
    sim = rfa.from_workload(w)
    sim.set_conduction(rfa.COND_FACE)
    done = 0
    for ci, cp in enumerate(g["checkpoints"]):
        sim.step(int(cp) - done)
        done = int(cp)
        T = sim.get_temperature(0)
        err_s = _check_against_golden(g, "", T, None, w.dims, ci)
    N = sim.get_necrosis(0)
    err, n_mism = _check_final_golden(g, "", T, N)
    # and the mode matters at this size: Eq. 12 as printed gives a different field at the interfaces
    sim2 = rfa.from_workload(w)
    sim2.step(done)
    T2 = sim2.get_temperature(0)
    idx = g["sample_idx"]
    assert float(np.max(np.abs(T2.ravel()[idx].astype(np.float64) - g["sample_T"][-1]))) > 0.05
    print(f"C4F: sampled max|dT| {err_s:.2e}, crop {err:.2e}, necrosis mismatches {n_mism}")
    sim2.close()
    # field-wide: every voxel of this workload moves (non-uniform start), so a compact stored field would be the whole
    # 268 MB image; the conservative oracle runs the 400 steps here instead and all 67 M voxels are compared
    osim = oracle.run_workload(w, steps=done, conservative=True)
    assert float(np.max(np.abs(osim.T.ravel()[idx] - g["sample_T"][-1]))) <= 1e-12      # the live oracle reproduces the stored one
    err_f, n_band = compare(T, N, osim)
    print(f"C4F: field max|dT| {err_f:.2e} over all {T.size} voxels, {n_band} necrosis differences inside the band")
    sim.close()


def test_c5_sweep_vs_golden(rfa):
    g = _golden("C5")
    w = W.c5_sweep()
    from tests.golden.make_golden import fingerprint
    sim = rfa.from_workload(w)
    sim.step(w.steps)
    vox = w.spacing_mm[0] * w.spacing_mm[1] * w.spacing_mm[2]
    for b in range(w.batch):
        p = f"s{b}_"
        assert fingerprint(w, b) == str(g[p + "fingerprint"])
        T = sim.get_temperature(b)
        N = sim.get_necrosis(b)
        _check_against_golden(g, p, T, N, w.dims)
        err, n_mism = _check_final_golden(g, p, T, N)
        _, tissue_v = sim.necrotic_voxels(b)
        assert abs(tissue_v * vox - float(g[p + "necro_volume_mm3"])) <= n_mism * vox
    sim.close()


def test_c5_sweep_fieldwide_vs_live_oracle(rfa, oracle):
    """Field-wide on the planning sweep: sixteen seeded scenarios of the 64 are run by the oracle here (3000 steps of
    128^3 each) and compared voxel by voxel with the batched launch bench.py times (all 64 scenarios in flight); the
    other scenarios are covered by test_c5_sweep_vs_golden (samples, crop, full necrosis mask).  A stored compact field
    for all 64 would be 35 MB of goldens."""
    w = W.c5_sweep()
    sim = rfa.from_workload(w)
    sim.step(w.steps)
    rng = np.random.default_rng(190705709)
    for b in sorted(rng.choice(w.batch, size=16, replace=False).tolist()):
        osim = oracle.run_workload(w, scenario=b)
        err, n_band = compare(sim.get_temperature(b), sim.get_necrosis(b), osim)
        print(f"C5 scenario {b}: field max|dT| {err:.2e}, {n_band} necrosis differences inside the band")
    sim.close()


# ----------------------------------------------------------------------------------------------
# Full size, field-wide, every tile / z-chunk seam of the launch configuration bench.py times
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["C4", "C3"])
def test_full_size_variants_bit_identical_fieldwide(rfa, name):
    """C4 / C3 with a smooth non-uniform start (every voxel changes every step): 30 steps of the plain kernel
    (one thread per voxel, no tiles) against the blocked kernel with S = 1, 2, 3 fused steps and the TMA-staged
    one-step kernel, each in both held-copy settings, the whole field bit for bit.  This is what exercises all work items of the full-size plan
    (C4: 540 items on 296 CTAs, the multi-item-per-CTA loop) in Eq. 12 mode."""
    w = W.with_smooth_field(W.BENCH_CONFIGS[name](steps=30))
    ref = None
    for kernel, fused, hc in [(rfa.KERNEL_PLAIN, 0, 0), (rfa.KERNEL_BLOCKED, 3, 1), (rfa.KERNEL_BLOCKED, 3, 0),
                              (rfa.KERNEL_BLOCKED, 2, 1), (rfa.KERNEL_BLOCKED, 2, 0), (rfa.KERNEL_BLOCKED, 1, 1),
                              (rfa.KERNEL_BLOCKED, 1, 0), (rfa.KERNEL_BLOCKED, 4, 1), (rfa.KERNEL_STREAM, 1, 1),
                              (rfa.KERNEL_STREAM, 1, 0)]:
        sim = rfa.from_workload(w)
        sim.configure(kernel, fused)
        sim.configure_held_copy(hc)
        sim.step(w.steps)
        T, N = sim.get_temperature(0), sim.get_necrosis(0)
        sim.close()
        if ref is None:
            ref = (T, N)
            assert float(np.ptp(T)) > 10.0
        else:
            assert np.array_equal(T.view(np.uint32), ref[0].view(np.uint32)), (name, fused, hc)
            assert np.array_equal(N, ref[1]), (name, fused, hc)


@pytest.mark.parametrize("name,conservative", [("C4", False), ("C3", False), ("C4", True)])
def test_full_size_short_run_fieldwide_vs_live_oracle(rfa, oracle, name, conservative):
    """Full size, default launch configuration, non-uniform field: 7 steps (launches of 3 + 3 + 1) against the oracle
    run here on the same inputs, EVERY voxel compared."""
    w = W.with_smooth_field(W.BENCH_CONFIGS[name](steps=7))
    osim = oracle.run_workload(w, conservative=conservative)
    sim = rfa.from_workload(w)
    if conservative:
        sim.set_conduction(rfa.COND_FACE)
    sim.step(w.steps)
    err, n_band = compare(sim.get_temperature(0), sim.get_necrosis(0), osim)
    print(f"{name}{' (conservative)' if conservative else ''}: 7 steps, field max|dT| {err:.2e} over {w.n_voxels} voxels")
    sim.close()


@pytest.mark.parametrize("name", ["C4", "C3"])
def test_full_length_default_configuration_is_bit_identical_to_plain(rfa, name):
    """The whole configured run (C4: 12 000 steps, C3: 24 000) in the default launch configuration against the
    one-thread-per-voxel kernel (no tiles, no rings, no barriers, one step per launch), field and mask bit for bit.
    Only a run of this length gets the residual-prefetch variant switched on by the library's own feedback in mid-run
    (C3) and work items that are mostly hot; a stale read of a shared-memory ring slot or of a halo plane anywhere in
    those launches would show here, which stands in for the racecheck run this pool does not allow."""
    w = W.BENCH_CONFIGS[name]()
    ref = rfa.from_workload(w)
    ref.configure(rfa.KERNEL_PLAIN, 0)
    ref.step(w.steps)
    Tp, Np = ref.get_temperature(0), ref.get_necrosis(0)
    ref.close()
    sim = rfa.from_workload(w)
    for _ in range(8):                          # several calls, as the residual-prefetch test does: the feedback is acted on at launches
        sim.step(w.steps // 8)
    hot = sim.hot_fraction()
    T, N = sim.get_temperature(0), sim.get_necrosis(0)
    v = sim.query_variant()
    sim.close()
    assert v["fused_steps"] == 3 and w.steps % 8 == 0
    assert np.array_equal(T.view(np.uint32), Tp.view(np.uint32)), f"{name}: default configuration differs from the plain kernel after {w.steps} steps"
    assert np.array_equal(N, Np)
    if name == "C3":                            # the umbrella needle warms enough of the volume: the variant switched on by itself
        assert hot["residual_prefetch"] == 1 and hot["hot_fraction"] >= 0.004, hot      # RFA_HOT_ON
    print(f"{name}: {w.steps} steps, default configuration == plain kernel bit for bit; hot fraction {hot}")


def test_residual_prefetch_switches_on_by_itself(rfa):
    """AUTO mode: the kernels count the warp-planes that take the compensated path; once the library has seen that a few
    percent of them do, it launches the residual-prefetch variant (no synchronisation involved), and the field is the same
    bit for bit as with the variant forced off."""
    w = W.ragged_phantom(dims=(144, 70, 41), spacing=(0.7, 0.9, 1.3), steps=600, mode=W.SRC_POWER, value=4.0e7, dt=0.05)
    sims = {}
    for mode in (rfa.RES_PREFETCH_AUTO, rfa.RES_PREFETCH_OFF):
        sim = rfa.from_workload(w)
        sim.configure(rfa.KERNEL_BLOCKED, 3)
        sim.configure_residual_prefetch(mode)
        for _ in range(6):                      # several calls: the feedback is looked at when a later launch is issued
            sim.step(100)
            sim.synchronize()
        sims[mode] = (sim.get_temperature(0), sim.hot_fraction(), sim.query_variant())
        sim.close()
    Ta, ha, va = sims[rfa.RES_PREFETCH_AUTO]
    To, ho, vo = sims[rfa.RES_PREFETCH_OFF]
    assert np.array_equal(Ta.view(np.uint32), To.view(np.uint32))
    assert ha["hot_fraction"] > 0.004, ha      # a power source of 4e7 W/m3 warms a good part of this small grid by >= 1 C
    assert ha["residual_prefetch"] == 1 and va["residual_prefetch"] == 1
    assert ho["residual_prefetch"] == 0 and vo["residual_prefetch"] == 0
