"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol include/rfa.h
declares, and its host-side logic (validation, stability bound, launch planning) behaves.  No compute
call is made: without a GPU rfa_create must fail loudly (there is no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1907_05709_b200 import binding, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1907_05709_b200 import build
    build.build()
    return binding.load_library()


def test_exports_match_header(lib):
    hdr = open(os.path.join(ROOT, "include", "rfa.h")).read()
    body = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(rfa_[a-z_]+)\s*\(", body))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_tissue_struct_layout():
    assert ctypes.sizeof(binding.RfaTissue) == 28 == W.TISSUE_DTYPE.itemsize


def test_stability_number_matches_bound(lib):
    t = W.tissue_table()
    s = binding.stability_number((1.0, 1.0, 1.0), t, 0.1)
    # liver: 0.1 * (2 * 0.512/(1060*3600) * 3e6 + 6.4e-3*1050*3617/(1060*3600)) ; kidney has the larger sink
    assert 0.05 < s < 0.1
    assert binding.stability_number((0.5, 0.5, 0.5), W.paper_liver_table(), 0.1) == pytest.approx(0.1 * (2 * 0.52 / (1079 * 3540) * 1.2e7 + 16.687 * 3617 / (1079 * 3540)), rel=1e-6)
    assert binding.stability_number((1.0, 1.0, -1.0), t, 0.1) < 0
    assert binding.stability_number((1.0, 1.0, 1.0), t, 0.0) < 0


def _create(lib, dims, spacing, labels, table, dt, batch=1, n_tissue=None):
    h = ctypes.c_void_p()
    lab = np.ascontiguousarray(labels, dtype=np.uint8)
    rc = lib.rfa_create(ctypes.byref(h), binding._i3(dims), binding._f3(spacing), ctypes.c_void_p(lab.ctypes.data),
                        binding.tissue_array(table), len(table) if n_tissue is None else n_tissue,
                        37.0, dt, batch, None, 0, None)
    return rc, h, lib.rfa_last_error().decode()


def test_create_validation_happens_before_cuda(lib):
    t = W.tissue_table()
    lab = np.ones((4, 4, 4), np.uint8)
    rc, h, msg = _create(lib, (4, 4, 0), (1, 1, 1), lab, t, 0.1)
    assert rc == binding.RFA_E_INVALID and not h.value
    rc, h, msg = _create(lib, (4, 4, 4), (1, 0, 1), lab, t, 0.1)
    assert rc == binding.RFA_E_INVALID
    rc, h, msg = _create(lib, (4, 4, 4), (1, 1, 1), lab * 9, t, 0.1)
    assert rc == binding.RFA_E_INVALID and "label" in msg
    rc, h, msg = _create(lib, (4, 4, 4), (1, 1, 1), lab, t, -0.1)
    assert rc == binding.RFA_E_INVALID
    rc, h, msg = _create(lib, (4, 4, 4), (1, 1, 1), lab, t, 0.1, batch=0)
    assert rc == binding.RFA_E_INVALID
    rc, h, msg = _create(lib, (4, 4, 4), (1, 1, 1), lab, t, 0.1, n_tissue=40)
    assert rc == binding.RFA_E_INVALID
    bad = t.copy()
    bad["rho"][1] = 0.0
    rc, h, msg = _create(lib, (4, 4, 4), (1, 1, 1), lab, bad, 0.1)
    assert rc == binding.RFA_E_INVALID
    # dt above the monotone bound (R-18): 0.5 mm voxels, dt = 0.4 s
    rc, h, msg = _create(lib, (4, 4, 4), (0.5, 0.5, 0.5), lab, t, 0.4)
    assert rc == binding.RFA_E_UNSTABLE and "monotone" in msg


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    rc, h, msg = _create(lib, (4, 4, 4), (1, 1, 1), np.ones((4, 4, 4), np.uint8), W.tissue_table(), 0.1)
    assert rc == binding.RFA_E_CUDA and not h.value
    assert "no CPU fallback" in msg


def test_null_handles_are_rejected(lib):
    assert lib.rfa_step(None, 1) == binding.RFA_E_INVALID
    assert lib.rfa_synchronize(None) == binding.RFA_E_INVALID
    assert lib.rfa_configure(None, 0, 0) == binding.RFA_E_INVALID
    for fn in (lib.rfa_configure_held_copy, lib.rfa_configure_staging, lib.rfa_configure_tile, lib.rfa_configure_residual_prefetch):
        assert fn(None, 0) == binding.RFA_E_INVALID
    assert lib.rfa_query_hot_fraction(None, None, None) == binding.RFA_E_INVALID
    assert lib.rfa_step_record_static(None, 1, 1, 0, None, None) == binding.RFA_E_INVALID
    lib.rfa_destroy(None)


def test_workspace_bytes(lib):
    n = lib.rfa_workspace_bytes(binding._i3((512, 512, 256)), 1)
    nv = 512 * 512 * 256
    # 2 x fp32 theta + 2 x fp16 residual + 1 state byte + 4-byte staging buffer
    assert nv * (4 + 4 + 2 + 2 + 1 + 4) <= n <= nv * 17 + 65536
    assert lib.rfa_workspace_bytes(binding._i3((0, 4, 4)), 1) == 0
    n5 = lib.rfa_workspace_bytes(binding._i3((128, 128, 128)), 64)
    assert n5 >= 64 * 128 ** 3 * 13


@pytest.mark.parametrize("dims,batch", [((512, 512, 256), 1), ((128, 128, 128), 64), ((256, 256, 256), 1),
                                        ((64, 64, 64), 1), ((44, 38, 29), 2)])
@pytest.mark.parametrize("fused", [1, 2, 3, 4])
def test_blocked_plan_covers_the_grid(lib, dims, batch, fused):
    """Tiles (x overlap 8, y halo S) and z chunks must cover every voxel; work items fill whole rounds."""
    p = binding.plan_query(dims, batch, fused, 148)
    assert p["ok"] == 1
    nx, ny, nz = dims
    BX, BY = p["bx"], p["by"]
    assert BX % 4 == 0 and BY > 2 * fused
    last_x0 = (p["tiles_x"] - 1) * (BX - 8)
    assert last_x0 + BX >= nx and (p["tiles_x"] == 1 or last_x0 + 4 < nx)
    assert p["tiles_y"] * (BY - 2 * fused) >= ny > (p["tiles_y"] - 1) * (BY - 2 * fused)
    assert p["z_chunks"] * p["planes_per_chunk"] >= nz > (p["z_chunks"] - 1) * p["planes_per_chunk"]
    assert p["work_items"] == p["tiles_x"] * p["tiles_y"] * p["z_chunks"] * batch
    assert p["ctas"] == min(p["work_items"], 148)


def test_planner_picks_the_tile_shape_by_grid(lib):
    """Two arrangements of the 256-thread CTA: 64 x 32 tiles on wide grids, whole 128-voxel rows (128 x 16 tiles) where
    that needs fewer plane iterations (the 128^3 planning-sweep volumes)."""
    assert binding.plan_query((512, 512, 256), 1, 3, 296)["bx"] == 64
    assert binding.plan_query((256, 256, 256), 1, 3, 296)["bx"] == 64
    p = binding.plan_query((128, 128, 128), 64, 3, 296)
    assert (p["bx"], p["by"], p["tiles_x"]) == (128, 16, 1)


def test_blocked_plan_rejects_unsupported_grids(lib):
    assert binding.plan_query((45, 38, 29), 1, 2, 148)["ok"] == 0      # nx % 4 != 0 -> plain kernel
    assert binding.plan_query((44, 38, 1), 1, 2, 148)["ok"] == 0       # nz < fused steps
    assert binding.plan_query((4096, 4096, 512), 1, 3, 296)["ok"] == 0  # 8.6e9 voxels: beyond 32-bit float4 offsets
    assert binding.plan_query((2048, 2048, 1024), 1, 3, 296)["ok"] == 1
    assert binding.plan_query((44, 38, 29), 1, 5, 148)["ok"] == 0


def test_plan_of_the_tma_staged_variant(lib):
    """RFA_STAGING_TMA: 2 or 3 fused steps, nx % 16 == 0, ny even; its tiles start a multiple of two rows above the grid, so
    at 3 fused steps the first tile owns one row less (tiles_y = ceil((ny + 1) / 26) for the 64 x 32 tile)."""
    TMA = binding.STAGING_TMA
    p = binding.plan_query((512, 512, 256), 1, 3, 296, TMA)
    assert p["ok"] == 1 and (p["bx"], p["by"], p["tiles_x"], p["tiles_y"]) == (64, 32, 9, 20)
    assert binding.plan_query((64, 26, 40), 1, 3, 296)["tiles_y"] == 1          # cp.async: 26 rows fit one tile ...
    assert binding.plan_query((64, 26, 40), 1, 3, 296, TMA)["tiles_y"] == 2     # ... TMA: one halo row more
    assert binding.plan_query((64, 28, 40), 1, 2, 296, TMA)["tiles_y"] == 1     # two fused steps: no extra row
    assert binding.plan_query((72, 38, 29), 1, 3, 148, TMA)["ok"] == 0          # nx % 16 != 0
    assert binding.plan_query((80, 33, 29), 1, 3, 148, TMA)["ok"] == 0          # odd ny
    assert binding.plan_query((80, 34, 29), 1, 1, 148, TMA)["ok"] == 0          # one step: the one-step kernel has its own TMA path
    assert binding.plan_query((80, 34, 29), 1, 4, 148, TMA)["ok"] == 0
    with pytest.raises(binding.RfaError):
        binding.plan_query((80, 34, 29), 1, 3, 148, 7)
