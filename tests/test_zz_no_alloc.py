"""rfa_step_record_static: the probe time series for callers that cannot allocate device memory when they ask for it.

Who that is: a frame loop that a cudaMalloc would stall (it waits for the whole GPU, so every simulation stream on the
card stops with it), and an application whose own memory pool already owns the card, where cudaMalloc just fails.  The
entry point keeps the probe list and the recorded rows in one fixed array inside librfa.so (1 MiB + 8 KiB per GPU, shared by
every call on that GPU, never cleared) instead of the buffers that rfa_set_probes / rfa_step_record allocate.

What is checked here: on the same inputs it returns the same bits as the allocating path (both run the same kernels, so the
bar is equality, which is inside the 1e-3 C the parity tests allow), on TWO calls in a row whose shapes differ -- the second
call finds the first call's list and rows still in the array and must not be affected by them -- and sizes beyond the stated
maximum are refused before anything is stepped.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure in this add-on must not hide the
parity tests.  It builds what it needs itself, so it also passes when run alone in a fresh process.
"""
import numpy as np
import pytest

from paper_1907_05709_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1.0e-3        # deg C, the bar of tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def rfa():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1907_05709_b200 import binding, build
    build.build()
    binding.load_library()          # raises if librfa.so is missing: no fallback
    return binding


def _case():
    w = W.paper_probe_case(90.0, n=48, steps=60)
    pr = W.fig6_probes(w.dims, w.spacing_mm, w.meta["centre_voxel"]).ravel()
    return w, pr


def test_static_record_equals_allocating_path_on_two_calls_in_a_row(rfa):
    import torch
    w, pr = _case()
    ref = rfa.from_workload(w)          # existing path: rfa_set_probes + rfa_step_record (cudaMalloc inside)
    sta = rfa.from_workload(w)          # new path: nothing allocated by the recording calls
    for sim in (ref, sta):
        sim.configure(rfa.KERNEL_BLOCKED, 3)

    # call 1: all 12 probes, a record after every step
    ref.set_probes(pr)
    exp1 = ref.step_record(36, 1)
    got1 = sta.step_record_static(36, 1, pr)
    assert got1.shape == exp1.shape == (36, 12)
    assert np.array_equal(got1.view(np.uint32), exp1.view(np.uint32))
    assert float(np.max(np.abs(got1.astype(np.float64) - exp1.astype(np.float64)))) <= TOL
    assert got1.min() >= 37.0 - TOL and got1.max() > 37.05         # the tip has warmed the near probes: real data, not zeros

    # call 2, straight after: fewer probes in another order, another cadence, device result buffer.  The array still
    # holds call 1's list (12 entries) and rows (432 floats); none of that may show up.
    pr2 = pr[[7, 0, 10, 3, 5]]
    ref.set_probes(pr2)
    exp2 = ref.step_record(24, 4)
    dev_out = torch.full((6, 5), -1.0, dtype=torch.float32, device="cuda")
    sta.step_record_static(24, 4, pr2, out=dev_out)
    got2 = dev_out.cpu().numpy()
    assert np.array_equal(got2.view(np.uint32), exp2.view(np.uint32))
    assert float(np.max(np.abs(got2.astype(np.float64) - exp2.astype(np.float64)))) <= TOL
    assert np.all(got2[0] >= got1[-1][[7, 0, 10, 3, 5]])             # the series goes on where call 1 stopped (monotone heating)

    # both simulations took the same 60 steps: same field, same mask, bit for bit
    assert np.array_equal(ref.get_temperature(0).view(np.uint32), sta.get_temperature(0).view(np.uint32))
    assert np.array_equal(ref.get_necrosis(0), sta.get_necrosis(0))
    # the probe list of rfa_set_probes is untouched by the static call: none was ever set on `sta`
    with pytest.raises(rfa.RfaError):
        sta.step_record(1, 1)
    ref.close()
    sta.close()


def test_static_record_refuses_sizes_beyond_its_array(rfa):
    w, pr = _case()
    sim = rfa.from_workload(w)
    before = sim.get_temperature(0)
    # too many probes
    many = np.resize(pr, rfa.STATIC_RECORD_MAX_PROBES + 1)
    with pytest.raises(rfa.RfaError) as ei:
        sim.step_record_static(1, 1, many, out=np.empty((1, many.size), np.float32))
    assert ei.value.code == rfa.RFA_E_INVALID and str(rfa.STATIC_RECORD_MAX_PROBES) in str(ei.value)
    # too many recorded values: 1024 probes x 257 records = 263168 > 262144
    full = np.resize(pr, rfa.STATIC_RECORD_MAX_PROBES)
    rows = rfa.STATIC_RECORD_MAX_FLOATS // full.size + 1
    with pytest.raises(rfa.RfaError) as ei:
        sim.step_record_static(rows, 1, full, out=np.empty((rows, full.size), np.float32))
    assert ei.value.code == rfa.RFA_E_INVALID and str(rfa.STATIC_RECORD_MAX_FLOATS) in str(ei.value)
    # an index outside the volume, no probes at all
    with pytest.raises(rfa.RfaError):
        sim.step_record_static(1, 1, [w.n_voxels * w.batch])
    with pytest.raises(rfa.RfaError):
        sim.step_record_static(1, 1, [])
    # a refused call steps nothing
    assert np.array_equal(before.view(np.uint32), sim.get_temperature(0).view(np.uint32))
    # exactly at the limit it runs: 1024 probes x 256 records
    rows = rfa.STATIC_RECORD_MAX_FLOATS // full.size
    got = sim.step_record_static(rows, 1, full)
    assert got.shape == (rows, full.size) and np.all(np.isfinite(got))
    assert np.array_equal(got[:, :12], got[:, 12:24])                  # np.resize repeats the 12 probes
    sim.close()
