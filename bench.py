#!/usr/bin/env python
"""bench.py -- headline benchmark of the RFA bioheat hot path (BASELINE.json: GVoxel-updates/s and
simulated steps/s at 512x512x256, % of the B200 HBM roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]

A "step" is ONE simulated time step of the whole hot path (load, second
differences, parameter lookup, source/sink, Euler update / hold, fused necrosis, buffer swap) over the
whole synthetic volume.  K steps are issued as ONE ``rfa_step(K)`` call through the C ABI (the library
fuses S steps per launch) and timed with CUDA events on the stream the kernels run on.

Legs of one run (ours):
  value     device-resident: state already in HBM, events around rfa_step(K)
  e2e       whole job through the public API from pinned HOST buffers: rfa_create (labels H2D),
            rfa_set_needle (mask H2D), rfa_step(K), rfa_get_temperature + rfa_get_necrosis (D2H),
            host clock around all of it (create's allocation included)
  roofline  dominant kernel: algorithmic bytes per launch / average launch duration over the timed region
  cpu_baseline  the fp64 oracle (oracle/, as it stands) on the host cores, on a bounded sample (rank 0, N=1)

N > 1 ("replicas only"): every rank runs an independent replica of the workload on
its own GPU, no data-path collective; value = all ranks' voxel-updates / max-over-ranks time.

``--impl reference`` times the oracle itself (there is no reference implementation to install: the
reference is the paper text) on a bounded z-slab sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "GVoxel-updates/s"
# Algorithmic bytes per voxel per launch of the stepping kernel.  SURVEY.md 8(d) counts
# 4 B theta read + 4 B theta write + 1 B label/flag byte + 1 B necrosis byte = 10 B, i.e. (8+2)/S per voxel-update with
# S fused steps; that is the figure roofline.frac is taken on.  This build keeps the necrosis bit inside the state
# byte (no second byte) and has a 2-B fp16 residual image for the compensated accumulation: 4 + 4 + 1 + 2 = 11 B was
# round 1's own count, reported beside it as frac_11B (since round 2 the residual is written for hot rows only: the
# measured DRAM traffic is 8.5-8.8 B per voxel per launch, the `traffic` key).
BYTES_SURVEY = {"theta_read": 4.0, "theta_write": 4.0, "label_byte": 1.0, "necrosis_byte": 1.0}
BYTES_BUILD = {"theta_read": 4.0, "theta_write": 4.0, "state_byte_read": 1.0, "residual_fp16_write": 2.0}
# Per launch of the dominant kernel, from the ncu rows summarised under profiles/: DRAM bytes (dram__bytes_read.sum +
# dram__bytes_write.sum) and warp instructions executed (smsp__inst_executed.sum).  Keyed by the variant string of the run
# (workload / fused steps / tile / held-copy / conduction / staging / residual prefetch): a run whose variant has no row
# prints "traffic": null and "issue": null.
_V = "profiles/r3_variants_ncu.md"
_AB = "profiles/r2_blocked_ab_ncu.md"
NCU_ROWS = {
    # variant: (DRAM bytes per launch, warp instructions per launch or None, profile file)
    "C4/S3/64x32/hc1/eq12": (588.2e6, 145.79e6, _V),
    "C4/S3/64x32/hc0/eq12": (577.1e6, 164.02e6, _V),
    "C4/S3/64x32/hc1/eq12/tma": (593.6e6, 153.31e6, _V),
    "C4/S2/64x32/hc1/eq12": (576.9e6, 88.84e6, _V),
    "C4/S4/64x32/hc1/eq12": (580.0e6, 197.87e6, _V),
    "C4/S1/64x32/hc1/eq12": (578.0e6, 46.66e6, _V),
    "C4/S1/128x16/hc1/eq12/tma": (569.1e6, 50.74e6, _V),
    "C4/S1/128x16/hc0/eq12/tma": (569.3e6, 57.81e6, _V),
    "C3/S3/64x32/hc0/eq12": (119.6e6, 46.51e6, _V),
    "C3/S1/128x16/hc0/eq12/tma": (113.4e6, 15.30e6, _V),
    "C5/S2/128x16/hc0/eq12/tma": (1199.9e6, 220.86e6, _V),
    "C5/S3/128x16/hc0/eq12/tma": (1186.2e6, 367.37e6, _V),
    "C2/S2/128x16/hc0/eq12/tma": (10.6e6, 6.26e6, _V),
    "C1/S3/64x32/hc0/eq12": (1.4e6, 4.43e6, _V),
    "C4/S3/64x32/hc1/face": (642.0e6, 180.77e6, _V),
    "C4F/S3/64x32/hc1/face": (851.2e6, 344.96e6, _V),
    "C4/plain": (840.3e6, 494.93e6, _V),
    # after ~2700 steps (hot region grown, residual prefetch on): rows of profiles/r2_blocked_ab_ncu.md, no instruction count there
    "C3/S3/64x32/hc0/eq12/rpf": (120.6e6, None, _AB),
    "C4F/S3/64x32/hc1/face/rpf": (870.9e6, None, _AB),
}
NCU_TRAFFIC = {k: (v[0], v[2]) for k, v in NCU_ROWS.items()}
FALLBACK_HBM_GBS = 6650.0            # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def variant_key(workload, variant):
    return "%s/S%d/%dx%d/hc%d/%s" % (workload, variant["fused_steps"], variant["tile_bx"], variant["tile_by"],
                                     variant["held_copy"], "face" if variant["conduction"] else "eq12")


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# ----------------------------------------------------------------------------------------------
# clocks during the timed region
# ----------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU every ~50 ms in a thread (NVML)."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                ids = [v for v in vis.split(",") if v.strip()]
                if index < len(ids) and ids[index].strip().isdigit():
                    phys = int(ids[index])
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.05)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ----------------------------------------------------------------------------------------------
# multi-rank plumbing (one process per GPU; replicas only -- no data-path collective)
# ----------------------------------------------------------------------------------------------
def aggregate(local_ms: float, local_units: float, dist=None, device=None):
    """(max over ranks of the time, sum over ranks of the units).  Works with any backend; unit-tested
    with gloo / world_size 2 on CPU."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_ms, local_units
    import torch
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ----------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline and --impl reference).  The only place bench.py touches oracle/.
# ----------------------------------------------------------------------------------------------
def _needle_slab(w, nzc):
    """z-slab of nzc planes of workload w centred on the needle (inputs only; no method arithmetic)."""
    nx, ny, nz = w.dims
    nzc = int(max(1, min(nz, nzc)))
    zc = int(round(np.nonzero(w.needles[0].mask)[0].mean())) if w.needles else nz // 2
    z0 = int(min(max(zc - nzc // 2, 0), nz - nzc))
    return z0, nzc


def oracle_time(w, steps, warmup, nzc, conservative=False):
    """Times `steps` oracle time steps on a z-slab of w (full slab = whole volume when nzc >= nz)."""
    from oracle import rfa_oracle
    rfa_oracle.build()
    nx, ny, nz = w.dims
    z0, nzc = _needle_slab(w, nzc)
    sim = rfa_oracle.OracleSim((nx, ny, nzc), w.spacing_mm, w.labels[z0:z0 + nzc], w.table, w.t_blood, w.dt,
                               conservative=conservative)
    if w.needles:
        nd = w.needles[0]
        sim.set_needle(nd.mask[z0:z0 + nzc], nd.mode, nd.value)
    if warmup:
        sim.step(warmup)
    t0 = time.perf_counter()
    sim.step(steps)
    secs = time.perf_counter() - t0
    return secs, nx * ny * nzc, rfa_oracle.num_threads(), (z0, nzc)


def cpu_baseline(w, budget_s=15.0, conservative=False):
    """The oracle, as it stands, on a bounded sample: whole volume, as many time steps as fit ~budget_s."""
    secs1, nv, thr, _ = oracle_time(w, 1, 0, w.dims[2], conservative)
    n = int(max(1, min(5000, budget_s / max(secs1, 1e-3))))
    secs, nv, thr, _ = oracle_time(w, n, 0, w.dims[2], conservative)
    gv = nv * n / secs / 1e9
    # the same oracle on ONE thread: a few steps, ~5 s
    from oracle import rfa_oracle
    rfa_oracle.set_num_threads(1)
    try:
        s1, nv1, _, _ = oracle_time(w, 1, 0, w.dims[2], conservative)
        n1 = int(max(1, min(50, 5.0 / max(s1, 1e-3))))
        s1, nv1, _, _ = oracle_time(w, n1, 0, w.dims[2], conservative)
        single = {"value": nv1 * n1 / s1 / 1e9, "unit": METRIC, "cores": 1, "steps": n1}
    finally:
        rfa_oracle.set_num_threads(thr)
    return {"value": gv, "unit": METRIC, "cores": thr, "kind": "oracle", "single_thread": single,
            "sample": f"{n} time steps of the full {w.dims[0]}x{w.dims[1]}x{w.dims[2]} {w.name} volume, fp64, "
                      f"OpenMP over z ({secs:.1f} s)",
            "steps_per_s": n / secs}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_1907_05709_b200 import workloads as W
    w = W.BENCH_CONFIGS[args.config]()
    nx, ny, nz = w.dims
    # calibrate on a thin slab, then size the slab so K + W steps end within ~budget seconds
    cons = args.conduction == "face"
    secs, nv, thr, _ = oracle_time(w, 2, 1, min(nz, 8), cons)
    rate = nv * 2 / secs
    budget = 100.0
    nzc = int(max(1, min(nz, budget * rate / ((args.steps + args.warmup) * nx * ny))))
    secs, nv, thr, (z0, nzc) = oracle_time(w, args.steps, args.warmup, nzc, cons)
    gv = nv * args.steps / secs / 1e9
    sample = (f"{args.steps} time steps on the z-slab [{z0},{z0 + nzc}) of {w.name} ({nx}x{ny}x{nzc} voxels around "
              f"the needle), fp64 oracle, OpenMP over z")
    line = {
        "impl": "reference", "metric": METRIC, "value": gv, "unit": METRIC, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs * 1e3 / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "dims": [nx, ny, nz], "sample_dims": [nx, ny, nzc],
                   "note": "the reference is the paper text only (no code); this arm times the repo's fp64 CPU oracle"},
        "cpu_baseline": {"value": gv, "unit": METRIC, "cores": thr, "kind": "oracle", "sample": sample},
        "e2e": {"value": gv, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------
def pinned(a):
    """Copy a numpy array into pinned host memory (torch is used for the allocation only)."""
    import torch
    t = torch.empty(a.shape, dtype=torch.from_numpy(np.empty(0, a.dtype)).dtype, pin_memory=True)
    v = t.numpy()
    v[...] = a
    return t, v


def measure_l2_and_launch_floor(dev, stream):
    """Two measured denominators for volumes that never leave the 126 MB L2 (C1, C2), where an HBM fraction says nothing:
      l2_copy_gbs      read + write bytes per second of `b.copy_(a)` between two 16 MiB device buffers, 200 copies back to
                       back on the bench stream (both buffers stay in L2 after the first copy), CUDA events
      launch_floor_us  time per launch of 400 back-to-back 4-byte copies on the same stream: what a launch costs when
                       the kernel does nothing (the floor under any one-launch-per-few-steps scheme)"""
    import torch
    a = torch.empty(4 << 20, dtype=torch.float32, device=dev)
    b = torch.empty_like(a)
    t = torch.zeros(1, dtype=torch.float32, device=dev)
    u = torch.zeros(1, dtype=torch.float32, device=dev)
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    with torch.cuda.stream(stream):
        for _ in range(10):
            b.copy_(a)
            u.copy_(t)
        e0.record(stream)
        for _ in range(200):
            b.copy_(a)
        e1.record(stream)
        for _ in range(400):
            u.copy_(t)
        e2.record(stream)
        e2.synchronize()
    return 2.0 * a.numel() * 4 * 200 / (e0.elapsed_time(e1) * 1e-3) / 1e9, e1.elapsed_time(e2) * 1e3 / 400


def run_ours(args):
    import torch
    from paper_1907_05709_b200 import binding, workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: librfa has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    binding.load_library()                      # raises if librfa.so is missing

    w = W.BENCH_CONFIGS[args.config]()
    nx, ny, nz = w.dims
    nvox_all = w.n_voxels * w.batch
    K, Wu = args.steps, args.warmup
    stream = torch.cuda.Stream(device=dev)

    # ---- device-resident leg ------------------------------------------------------------------
    hc_env = os.environ.get("RFA_HELD_COPY")          # A/B switch of the bench only; the library reads no environment
    with torch.cuda.stream(stream):
        sim = binding.from_workload(w, device=dev, stream=stream)
        sim.configure(args.kernel, args.fused)
        if hc_env in ("0", "1"):
            sim.configure_held_copy(int(hc_env))
        if args.staging != "auto":
            sim.configure_staging(binding.STAGING_TMA if args.staging == "tma" else binding.STAGING_CP_ASYNC)
        if args.tile >= 0:
            sim.configure_tile(args.tile)
        if args.res_prefetch != "auto":
            sim.configure_residual_prefetch(binding.RES_PREFETCH_ON if args.res_prefetch == "on" else binding.RES_PREFETCH_OFF)
        if args.conduction == "face":
            sim.set_conduction(binding.COND_FACE)
        sim.step(Wu)
        sim.synchronize()
        q0 = sim.query()
        S = max(q0["fused_steps"], 1)
        k_main, k_rem = K - K % S, K % S                # full S-step launches, then the remainder launch
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)
        with ClockSampler(local) as clk:
            e0.record(stream)
            sim.step(k_main)
            e1.record(stream)
            sim.step(k_rem)
            e2.record(stream)
            e2.synchronize()
            torch.cuda.synchronize(dev)
            if dist is not None:
                dist.barrier()
            ms_local = float(e0.elapsed_time(e2))
            ms_main = float(e0.elapsed_time(e1))
            q1 = sim.query()
            # the timed region of a short run (the driver's --steps 20 is 2 ms) is shorter than one NVML sample: keep
            # the same stepping loop running, untimed, until the sampler has seen >= 0.4 s under this load
            t_probe = time.perf_counter()
            while time.perf_counter() - t_probe < max(0.0, 0.4 - ms_local * 1e-3):
                sim.step(30 * S)
                sim.synchronize()
        variant = sim.query_variant()
        variant.update(sim.hot_fraction())
        necro_all, necro_tissue = sim.necrotic_voxels(0)
        tmax = float(sim.get_temperature(0).max())
        sim.close()
        del sim
    launches = q1["kernel_launches"] - q0["kernel_launches"]
    n_main = k_main // S
    ms, units = aggregate(ms_local, float(nvox_all) * K, dist, dev)
    gvox = units / (ms * 1e-3) / 1e9
    peak, peak_src = measured_peak()

    # dominant kernel = the stepping kernel: the timed region holds nothing else on this stream.  Its launch time is
    # taken over the full S-step launches only; the remainder launch (K % S steps) is reported separately.
    blocked = q1["kernel"] == binding.KERNEL_BLOCKED
    stream_k = q1["kernel"] == binding.KERNEL_STREAM
    launch_us = ms_main * 1e3 / max(n_main, 1) if n_main else ms_local * 1e3 / max(launches, 1)
    b_survey = sum(BYTES_SURVEY.values()) * nvox_all
    b_build = sum(BYTES_BUILD.values()) * nvox_all
    # Bytes the launch really moves.  Where an ncu capture of this variant exists: its DRAM traffic.  Otherwise this
    # build's own count: 4 B theta read + 4 B theta write + 1 B state byte (label, flags and the necrosis bit share it;
    # it is written back only where it changes), plus the fp16 residual (2 B read + 2 B written) for the share of rows
    # that are hot, which the kernels count themselves (rfa_query_hot_fraction).  SURVEY.md 8(d)'s 10 B per voxel has a
    # separate necrosis byte that this build does not move: kept as frac_survey_10B, not as the headline fraction.
    vkey = (variant_key(w.name, variant) + ("/tma" if variant.get("staging") == binding.STAGING_TMA else "") +
            ("/rpf" if variant.get("residual_prefetch") else "")) if (blocked or stream_k) else f"{w.name}/plain"
    traffic, traffic_src = NCU_TRAFFIC.get(vkey, (None, None))
    hot = float(variant.get("hot_fraction", 0.0) or 0.0) if (blocked or stream_k) else 1.0
    bytes_counted = {"theta_read": 4.0, "theta_write": 4.0, "state_byte_read": 1.0, "residual_fp16_read_write_hot_rows": 4.0 * hot}
    b_counted = sum(bytes_counted.values()) * nvox_all
    b_moved = traffic if traffic is not None else b_counted
    achieved = b_moved / (launch_us * 1e-6) / 1e9
    achieved_survey = b_survey / (launch_us * 1e-6) / 1e9
    # Issue-side roofline for the launches whose busiest unit is the warp schedulers: warp instructions per launch
    # (the variant's ncu row) / measured launch time / (SMs x 4 schedulers x the SM clock sampled during this run);
    # one warp instruction per scheduler and clock is the limit.
    clk_now = clk.summary()
    n_sm = int(torch.cuda.get_device_properties(dev).multi_processor_count)
    warp_inst = NCU_ROWS.get(vkey, (None, None, None))[1]
    issue = None
    if warp_inst is not None and clk_now.get("sm_mhz"):
        issue_peak = n_sm * 4 * float(clk_now["sm_mhz"]) * 1e6
        issue_ach = warp_inst / (launch_us * 1e-6)
        issue = {"achieved": issue_ach / 1e9, "peak": issue_peak / 1e9, "unit": "G warp-instructions/s",
                 "frac": issue_ach / issue_peak, "warp_instructions_per_launch": warp_inst,
                 "warp_instructions_source": NCU_ROWS[vkey][2] + " (smsp__inst_executed.sum)",
                 "peak_source": "%d SMs x 4 schedulers x %.0f MHz (SM clock sampled during the timed region, NVML), "
                                "1 warp instruction per scheduler and clock" % (n_sm, float(clk_now["sm_mhz"]))}
    roofline = {
        # S = 1: one pass over the field per step, the HBM stream binds.  S >= 2: the kernel moves the same bytes per
        # launch but does S steps of arithmetic on them; ncu shows the issue slots, not DRAM, as the busiest unit
        # (profiles/): frac stays the true share of the HBM peak, it is just not what limits the kernel
        "bound": "hbm" if (not blocked or S == 1) else "issue",      # (the one-step kernels, blocked S = 1 or TMA-staged: HBM)
        "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "bytes_basis": ("DRAM bytes per launch of this variant's ncu capture (traffic_source)" if traffic is not None else
                        "this build's count: 9 B per voxel + 4 B for the hot share of rows (no ncu capture of this variant)"),
        "bytes_per_launch": b_moved, "bytes_per_voxel_counted": bytes_counted,
        "achieved_survey_10B": achieved_survey, "frac_survey_10B": achieved_survey / peak,
        "traffic": traffic, "traffic_source": traffic_src, "variant": vkey, "peak_source": peak_src,
        "issue": issue,
        "kernel": f"rfa_blocked_kernel<S={S}>" if blocked else ("rfa_stream_kernel (TMA, S=1)" if stream_k else "rfa_plain_kernel"),
        "launches": launches, "full_launches": n_main, "avg_launch_us": launch_us,
        "remainder_launch": {"steps": k_rem, "us": (ms_local - ms_main) * 1e3} if k_rem else None,
        "algorithmic_bytes_per_launch": b_survey, "bytes_per_voxel": BYTES_SURVEY,
        "bytes_per_voxel_update": sum(BYTES_SURVEY.values()) / S,
        "frac_11B": b_build / (launch_us * 1e-6) / 1e9 / peak, "bytes_per_voxel_build": BYTES_BUILD,
        "fused_steps_per_launch": S,
        # north_star's roofline-EQUIVALENT: voxel-updates/s x 8 B (one 4-B read + one 4-B write of the field per TIME
        # STEP) over the copy peak.  A speed-up-equivalent that temporal blocking raises by design, not an HBM utilisation.
        "equiv_8B_frac": gvox / world * 8.0 / peak,
    }

    fits_l2 = nvox_all * 9 <= 126e6              # the same test as config.l2 below: what one step touches (2 fields + state) vs the 126 MB L2
    if fits_l2 and world == 1:
        # the volume stays in L2 from launch to launch: report against a measured L2 copy rate and the launch floor,
        # and keep the HBM share only as a labelled side figure
        l2_gbs, floor_us = measure_l2_and_launch_floor(dev, stream)
        achieved = b_counted / (launch_us * 1e-6) / 1e9      # bytes through L2 (this build's count), not the DRAM trickle
        roofline.update({
            "bound": "l2+launch", "achieved": achieved, "peak": l2_gbs, "frac": achieved / l2_gbs,
            "bytes_per_launch": b_counted, "bytes_basis": "this build's count through L2: 9 B per voxel + 4 B for the hot share of rows "
                                                          "(the DRAM traffic of an L2-resident volume, `traffic`, is next to nothing)",
            "peak_source": "measured here: torch b.copy_(a) between two 16 MiB device buffers, 200 copies back to back (L2-resident), read + write bytes; a 6 us copy kernel carries its own launch and tail overhead, so this is a floor of the L2 rate and frac an upper estimate",
            "frac_of_hbm_copy_peak": achieved / peak, "hbm_copy_peak": peak,
            "launch_floor_us": floor_us, "launch_floor_frac": floor_us / launch_us,
            "launch_floor_source": "measured here: 400 back-to-back 4-byte device copies on the bench stream, time per launch",
        })

    # ---- end-to-end leg: host buffers in, host buffers out --------------------------------------
    e2e = None
    if not args.no_e2e:
        _, lab_h = pinned(np.ascontiguousarray(w.labels, dtype=np.uint8))
        masks = [pinned(np.ascontiguousarray(nd.mask, dtype=np.uint8))[1] for nd in w.needles]
        _, T_h = pinned(np.empty((nz, ny, nx), np.float32))
        _, N_h = pinned(np.empty((nz, ny, nx), np.uint8))
        # The whole job three times, each through the public API from host buffers to host buffers; the MEDIAN is reported
        # and all three are listed.  A single shot is at the mercy of one cudaMalloc of the 0.7 GB workspace, which on a
        # fresh process takes anything between 1 and 25 ms (measured: jobs of 12.9 / 18.2 / 39.0 ms for the same 20 steps).
        e2e_runs = []
        for _rep in range(3):
            torch.cuda.synchronize(dev)
            if dist is not None:
                dist.barrier()
            t0 = time.perf_counter()
            with torch.cuda.stream(stream):
                s2 = binding.RfaSim(w.dims, w.spacing_mm, lab_h, w.table, w.t_blood, w.dt, batch=w.batch,
                                    device=dev, stream=stream)
                s2.configure(args.kernel, args.fused)
                if hc_env in ("0", "1"):
                    s2.configure_held_copy(int(hc_env))
                if args.conduction == "face":
                    s2.set_conduction(binding.COND_FACE)
                for b, nd in enumerate(w.needles):
                    s2.set_needle(b, masks[b], nd.mode, nd.value, nd.tip_mm, nd.axis)
                s2.step(K)
                for b in range(w.batch):
                    s2.get_temperature(b, out=T_h)
                    s2.get_necrosis(b, out=N_h)
                s2.synchronize()
            torch.cuda.synchronize(dev)
            e2e_runs.append((time.perf_counter() - t0) * 1e3)
            s2.close()
        e2e_ms_local = float(np.median(e2e_runs))
        e2e_ms, e2e_units = aggregate(e2e_ms_local, float(nvox_all) * K, dist, dev)
        h2d = w.n_voxels * (1 + len(w.needles))
        d2h = w.n_voxels * 5 * w.batch
        e2e = {"value": e2e_units / (e2e_ms * 1e-3) / 1e9, "unit": METRIC,
               "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K,
               "h2d_bytes_per_job": h2d, "d2h_bytes_per_job": d2h, "job_ms": e2e_ms, "job_ms_runs": e2e_runs,
               "what": "rfa_create(host labels) + rfa_set_needle(host mask) + rfa_step(K) + rfa_get_temperature/"
                       "rfa_get_necrosis into pinned host buffers, host clock, allocation included; median of 3 whole jobs"}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_baseline(w, conservative=(args.conduction == "face"))

    if rank == 0:
        line = {
            "metric": METRIC, "value": gvox, "unit": METRIC, "n_gpus": world, "steps": K, "warmup": Wu,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "dims": [nx, ny, nz], "batch": w.batch, "spacing_mm": list(w.spacing_mm),
                       "dt_s": w.dt, "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "l2": "inputs larger than L2 (2 x %d MiB fields + %d MiB state vs 126 MB L2)" % (
                           nvox_all * 4 >> 20, nvox_all >> 20) if nvox_all * 9 > 126e6 else
                             "working set fits L2 (reported, not held to the HBM bar)",
                       "kernel": roofline["kernel"], "conduction": args.conduction, "variant": variant},
            "sim_steps_per_s": K / (ms * 1e-3) * (1 if world == 1 else world),
            # BASELINE.json's "% of B200 HBM roofline" as north_star defines it: voxel-updates/s x 8 B (one read + one
            # write of the fp32 field per time step) over the measured copy bandwidth -- a roofline-EQUIVALENT (speed-up
            # over a one-step kernel at the copy peak), not an HBM utilisation; the true HBM fraction is roofline.frac
            "roofline_equiv_8B_frac": roofline["equiv_8B_frac"],
            "roofline": roofline, "e2e": e2e, "cpu_baseline": cpu, "gpu_launches": launches,
            "clocks": clk.summary(),
            "check": {"t_max_c": tmax, "necrotic_voxels": necro_all, "necrotic_tissue_voxels": necro_tissue},
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_warp(args):
    """Row f3 (Eq. 14 warp) on the C4 volume: K warps of the heated image through a device-resident displacement
    field; algorithmic bytes per voxel = 12 (displacement) + 4 (image, read once through L2) + 4 (output)."""
    import torch
    from paper_1907_05709_b200 import binding, workloads as W
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    w = W.BENCH_CONFIGS[args.config]()
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        sim = binding.from_workload(w, device=dev, stream=stream)
        sim.step(300)
        d = torch.from_numpy(W.breathing_field(w.dims)).to(dev)
        out = torch.empty((w.dims[2], w.dims[1], w.dims[0]), dtype=torch.float32, device=dev)
        for _ in range(max(args.warmup, 3)):
            sim.warp_temperature(0, d, 0.85, out=out)
        K = min(args.steps, 200)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(dev.index or 0) as clk:
            e0.record(stream)
            for _ in range(K):
                sim.warp_temperature(0, d, 0.85, out=out)       # device in / device out: asynchronous
            e1.record(stream)
            e1.synchronize()
        ms = float(e0.elapsed_time(e1))
        sim.close()
    peak, peak_src = measured_peak()
    gv = w.n_voxels * K / (ms * 1e-3) / 1e9
    ach = 20.0 * w.n_voxels * K / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "GVoxel/s (Eq. 14 warp)", "value": gv, "unit": "GVoxel/s", "n_gpus": 1, "steps": K,
                      "warmup": max(args.warmup, 3), "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": w.name + " warp", "dims": list(w.dims), "field": "breathing_field, scale 0.85"},
                      "roofline": {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                                   "traffic": None, "peak_source": peak_src, "kernel": "rfa_warp_kernel",
                                   "algorithmic_bytes_per_launch": 20.0 * w.n_voxels},
                      "gpu_launches": K, "clocks": clk.summary()}), flush=True)
    return 0


def run_record(args):
    """Row f2 and the paper's own regime (Alg. 2: ONE time iteration of Alg. 1 per displayed frame,
    :330; probe curves of Fig. 6 / Fig. 14, :147).  Two legs on the configured volume, both one step per frame:
      record   rfa_step_record(K, every=1): K single-step launches, each followed by the probe read-out kernel
      handoff  the Alg. 2 frame loop: rfa_step(1) -> event -> a consumer on a SECOND stream reads the finished image
               (rfa_current_frame; here a device-to-device copy into a "display" buffer stands in for the renderer)
               while the next step runs into the other buffer; the step after that waits for the consumer's event,
               because it overwrites the image the consumer was given."""
    import torch
    from cuda.bindings import runtime as cudart
    from paper_1907_05709_b200 import binding, workloads as W
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    w = W.BENCH_CONFIGS[args.config]()
    nx, ny, nz = w.dims
    K = min(args.steps, 3000)
    stream, side = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
    mz, my, mx = np.nonzero(w.needles[0].mask)
    centre = (int(round(mx.mean())), int(round(my.mean())), int(round(mz.mean())))
    probes = W.fig6_probes(w.dims, w.spacing_mm, centre).ravel()
    with torch.cuda.stream(stream):
        sim = binding.from_workload(w, device=dev, stream=stream)
        sim.configure(args.kernel, 1)                      # one time step per launch: the interactive regime
        hc_env = os.environ.get("RFA_HELD_COPY")
        if hc_env in ("0", "1"):
            sim.configure_held_copy(int(hc_env))
        sim.set_probes(probes)
        rec = torch.empty((K, probes.size), dtype=torch.float32, device=dev)
        sim.step_record(max(args.warmup, 3), 1, out=rec)
        q0 = sim.query()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(dev.index or 0) as clk:
            e0.record(stream)
            sim.step_record(K, 1, out=rec)
            e1.record(stream)
            e1.synchronize()
            ms_rec = float(e0.elapsed_time(e1))
            q1 = sim.query()
            # ---- Alg. 2 hand-off loop with an overlapped consumer
            display = torch.empty(nx * ny * nz, dtype=torch.float32, device=dev)
            prod = [torch.cuda.Event() for _ in range(K)]
            cons = [torch.cuda.Event() for _ in range(K)]
            nbytes = nx * ny * nz * 4
            sim.step(3)
            torch.cuda.synchronize(dev)
            e0.record(stream)
            for f in range(K):
                if f >= 2:
                    stream.wait_event(cons[f - 2])         # step f overwrites the image consumer f-2 was reading
                sim.step(1)
                prod[f].record(stream)
                ptr, _ = sim.current_frame(0)
                side.wait_event(prod[f])
                (rc,) = cudart.cudaMemcpyAsync(display.data_ptr(), ptr, nbytes,
                                               cudart.cudaMemcpyKind.cudaMemcpyDeviceToDevice, side.cuda_stream)
                assert int(rc) == 0
                cons[f].record(side)
            e1.record(stream)
            side.synchronize()
            e1.synchronize()
            torch.cuda.synchronize(dev)
            ms_hand = float(e0.elapsed_time(e1))
        variant = sim.query_variant()
        last = rec[-1].cpu().numpy()
        sim.close()
    peak, peak_src = measured_peak()
    fps_rec, fps_hand = K / (ms_rec * 1e-3), K / (ms_hand * 1e-3)
    # the TMA-staged one-step kernel moves 8.48 B per voxel (569.1 MB per C4 launch, profiles/r3_variants_ncu.md);
    # without a capture of the workload: 9 B (theta read + write, state byte).  SURVEY's 10 B is kept as frac_survey_10B.
    stream_used = q1["kernel"] == binding.KERNEL_STREAM      # what rfa_query reports for one-step launches of this simulation
    tr = NCU_TRAFFIC.get("C4/S1/128x16/hc%d/eq12/tma" % variant.get("held_copy", 0)) if (w.name == "C4" and stream_used) else None
    b_step = tr[0] if tr else 9.0 * w.n_voxels
    b_step_survey = sum(BYTES_SURVEY.values()) * w.n_voxels
    ach = b_step * fps_rec / 1e9
    print(json.dumps({
        "metric": "frames/s (Alg. 2 frame loop: one time step per frame, probes recorded every frame)",
        "value": fps_rec, "unit": "frames/s", "n_gpus": 1, "steps": K, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_rec / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": w.name + " frame loop", "dims": list(w.dims), "probes": int(probes.size), "variant": variant,
                   "paper_context": "PAPER.md:13/:290: > 480 Hz on a 256^2 x 234 volume (GTX 1080 / 1080 Ti), other hardware"},
        "gvoxel_updates_per_s": w.n_voxels * fps_rec / 1e9,
        "handoff": {"frames_per_s": fps_hand, "ms_per_frame": ms_hand / K, "gvoxel_updates_per_s": w.n_voxels * fps_hand / 1e9,
                    "consumer": "device-to-device copy of the finished image (%d MiB) on a second stream, overlapped with "
                                "the next step" % (nbytes >> 20)},
        "roofline": {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None,
                     "peak_source": peak_src,
                     "kernel": ("rfa_stream_kernel (TMA, S=1)" if stream_used else "rfa_blocked_kernel<S=1>") + " + rfa_probe_kernel",
                     "bytes_per_launch": b_step, "bytes_basis": (tr[1] + " (DRAM bytes of the one-step kernel)") if tr else "this build's count: 9 B per voxel",
                     "algorithmic_bytes_per_launch": b_step_survey, "bytes_per_voxel": BYTES_SURVEY,
                     "frac_survey_10B": b_step_survey * fps_rec / 1e9 / peak,
                     "equiv_8B_frac": w.n_voxels * fps_rec * 8.0 / 1e9 / peak},
        "gpu_launches": q1["kernel_launches"] - q0["kernel_launches"], "clocks": clk.summary(),
        "check": {"probe_t_c_last_frame": [float(x) for x in last]}}), flush=True)
    return 0


def run_render(args):
    """Row f4 (headless view of the heat zone) on the C4 volume: K frames of 512 x 512 pixels, oblique view,
    0.5 mm steps.  Reported as frame time (host images), kernel time (device images) and trilinear samples per second.
    The kernel is a gather: eight 4-byte loads per sample that counts, served by L1 (ncu: 95 % hit rate).  Its roofline is
    the L1 request rate: one warp-wide load per SM and clock if the 32 addresses fell into one 128-byte line; the oblique
    view needs about five lines per load (ncu), which is what bounds it (profiles/r2_view_kernels_ncu.md)."""
    import torch
    from paper_1907_05709_b200 import binding, workloads as W
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    w = W.BENCH_CONFIGS[args.config]()
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        sim = binding.from_workload(w, device=dev, stream=stream)
        sim.step(600)
        for _ in range(3):
            tmax, depth = sim.render_zone(0, (1, 2, 3), (0, 1, 0), 512, 512, 0.7, 0.5, 42.5)
        K = min(args.steps, 20)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(K):
            sim.render_zone(0, (1, 2, 3), (0, 1, 0), 512, 512, 0.7, 0.5, 42.5)
        e1.record(stream)
        e1.synchronize()
        ms = float(e0.elapsed_time(e1)) / K
        # kernel alone: both images stay on the device
        t_dev = torch.empty(512 * 512, dtype=torch.float32, device=dev)
        d_dev = torch.empty(512 * 512, dtype=torch.float32, device=dev)
        sim.render_zone(0, (1, 2, 3), (0, 1, 0), 512, 512, 0.7, 0.5, 42.5, tmax=t_dev, depth=d_dev)
        e0.record(stream)
        for _ in range(K):
            sim.render_zone(0, (1, 2, 3), (0, 1, 0), 512, 512, 0.7, 0.5, 42.5, tmax=t_dev, depth=d_dev)
        e1.record(stream)
        e1.synchronize()
        ms_dev = float(e0.elapsed_time(e1)) / K
        sim.close()
    ext = [n * h for n, h in zip(w.dims, w.spacing_mm)]
    ns = int(np.floor(np.sqrt(sum(e * e for e in ext)) / 0.5)) + 1
    # samples that count (inside the box of voxel centres), from the geometry of the view (include/rfa.h: rfa_render_zone)
    wv = np.array([1.0, 2.0, 3.0]); wv /= np.linalg.norm(wv)
    e1v = np.cross(np.array([0.0, 1.0, 0.0]), wv); e1v /= np.linalg.norm(e1v)
    e2v = np.cross(wv, e1v)
    c = 0.5 * np.array(ext); R = 0.5 * float(np.sqrt(sum(e * e for e in ext)))
    uu = (np.arange(512) - 255.5) * 0.7
    o = c[None, None, :] + uu[None, :, None] * e1v + uu[:, None, None] * e2v - R * wv
    h = np.array(w.spacing_mm, dtype=np.float64); nn = np.array(w.dims, dtype=np.float64)
    q0, dq = o / h - 0.5, 0.5 * wv / h
    lo = np.zeros((512, 512)); hi = np.full((512, 512), ns - 1.0)
    for a in range(3):
        t0, t1 = (0.0 - q0[..., a]) / dq[a], (nn[a] - 1.0 - q0[..., a]) / dq[a]
        lo, hi = np.maximum(lo, np.minimum(t0, t1)), np.minimum(hi, np.maximum(t0, t1))
    inside = float(np.maximum(np.floor(hi) - np.ceil(lo) + 1.0, 0.0).sum())
    sm_count, sm_hz = 148, 1.965e9
    req = inside * 8 / 32 / (ms_dev * 1e-3)                 # warp-wide gather loads per second
    roof = {"bound": "l1", "achieved": req / 1e9, "peak": sm_count * sm_hz / 1e9, "unit": "G warp-wide loads/s",
            "frac": req / (sm_count * sm_hz), "traffic": None,
            "peak_source": "148 SMs x 1965 MHz x one 128-byte L1 line per clock (B200_PROFILING.md unit counts and clocks); a load "
                           "of this view touches ~5 lines (ncu), so the L1 is ~5x busier than frac says",
            "kernel": "rfa_render_kernel", "kernel_ms": ms_dev, "samples_inside_box": inside,
            "gsamples_inside_per_s": inside / (ms_dev * 1e-3) / 1e9}
    print(json.dumps({"metric": "frames/s (heat-zone view, 512x512, host images)", "value": 1e3 / ms, "unit": "frames/s",
                      "n_gpus": 1, "steps": K, "warmup": 3, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": w.name + " view", "dims": list(w.dims), "image": [512, 512], "step_mm": 0.5,
                                 "samples_per_ray": ns, "visible_pixels": int((depth >= 0).sum())},
                      "gsamples_per_s": 512 * 512 * ns / (ms * 1e-3) / 1e9, "roofline": roof, "gpu_launches": 2 * K + 1}), flush=True)
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=12000)
    ap.add_argument("--warmup", type=int, default=120)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C4", choices=["C1", "C2", "C3", "C4", "C5", "C4F"])
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 plain, 2 blocked, 3 TMA-staged one-step (rfa_configure)")
    ap.add_argument("--fused", type=int, default=0, help="fused time steps per launch, 0 = library default")
    ap.add_argument("--conduction", default="eq12", choices=["eq12", "face"],
                    help="eq12: Eq. 12 as printed (default, the headline); face: conservative div(K grad T), row f1")
    ap.add_argument("--op", default="step", choices=["step", "warp", "render", "record"],
                    help="step: the time-stepping hot path (the headline); warp: the Eq. 14 motion warp (row f3)")
    ap.add_argument("--staging", default="auto", choices=["auto", "tma", "cp_async"],
                    help="A/B switch: how the blocked kernel stages its input planes (rfa_configure_staging)")
    ap.add_argument("--res-prefetch", default="auto", choices=["auto", "on", "off"],
                    help="A/B switch: residual-prefetch variant of the blocked kernel (rfa_configure_residual_prefetch)")
    ap.add_argument("--tile", type=int, default=-1, choices=[-1, 0, 1],
                    help="A/B switch: tile shape of the blocked kernel, 0 = 64x32, 1 = 128x16 (rfa_configure_tile)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args(argv)
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    if args.op == "warp":
        return run_warp(args)
    if args.op == "render":
        return run_render(args)
    if args.op == "record":
        return run_record(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
