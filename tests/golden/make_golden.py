"""Writes the stored expected values under tests/golden/ for the full-length configs.

Calls ONLY the fp64 oracle (oracle/) and the seeded input generators
(paper_1907_05709_b200/workloads.py, which hold no method arithmetic).  Nothing here touches the
CUDA library.  Usage (CPU box, takes ~2 h of all-core time for everything):

    python tests/golden/make_golden.py C2 C5 C3 C4 [--threads 6]

Per config <C> it writes tests/golden/<C>_golden.npz with, at checkpoints (steps/4, steps/2, steps):
  sample_idx   flat voxel indices (half within +-24 voxels of the needle, half uniform), seeded
  sample_T     fp64 oracle temperatures at those voxels, per checkpoint
and for the final state: a 32^3 crop around the needle centroid (crop_lo, crop_T), the bit-packed
necrosis mask, necrotic voxel counts (all / without held-label and needle voxels), the voxels whose
temperature lies within 2e-3 C of 60 C (band_idx, band_T: the exempt band of BASELINE.json's
north_star is 1e-3), the field sum and maximum, a fingerprint of the inputs, and the oracle's speed,
and the WHOLE final field in a compact form (field_*): with T_init = t_init[label] (the label ->
temperature image of PAPER.md:139, which a test rebuilds from the inputs alone), the bounding box of the
voxels with |T - T_init| > 1e-6 C is stored as integer codes rint((T - T_init) / field_q), field_q = 1e-5 C
(so a stored value is within field_q / 2 of the oracle's), together with the largest |T - T_init| outside
the box (field_outside_max <= 1e-6).  A test that finds its field within TOL - field_q / 2 of the decoded
box and within TOL - field_outside_max of T_init elsewhere has shown |T - T_oracle| <= TOL at EVERY voxel.
For the batched config C5 the same is stored per scenario (fewer samples each).  "C4F" = the C4 body model with a
smooth non-uniform initial field and the conservative conduction term (row f1), 400 steps, with extra
samples on tissue interfaces.
"""
from __future__ import annotations

import argparse
import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import rfa_oracle  # noqa: E402
from paper_1907_05709_b200 import workloads as W  # noqa: E402


def fingerprint(w, scenario: int) -> str:
    h = hashlib.sha256()
    h.update(np.ascontiguousarray(w.labels).tobytes())
    h.update(np.ascontiguousarray(w.table).tobytes())
    h.update(np.ascontiguousarray(w.needles[scenario].mask).tobytes())
    h.update(np.asarray([w.dt, *w.spacing_mm, w.needles[scenario].value, w.needles[scenario].mode],
                        dtype=np.float64).tobytes())
    return h.hexdigest()


def sample_indices(w, scenario: int, n: int, seed: int) -> np.ndarray:
    rng = np.random.Generator(np.random.PCG64(seed))
    nx, ny, nz = w.dims
    mz, my, mx = np.nonzero(w.needles[scenario].mask)
    pick = rng.integers(0, len(mz), size=n // 2)
    off = rng.integers(-24, 25, size=(n // 2, 3))
    z = np.clip(mz[pick] + off[:, 0], 0, nz - 1)
    y = np.clip(my[pick] + off[:, 1], 0, ny - 1)
    x = np.clip(mx[pick] + off[:, 2], 0, nx - 1)
    near = x + nx * (y + ny * z)
    far = rng.integers(0, nx * ny * nz, size=n - n // 2)
    return np.unique(np.concatenate([near, far]).astype(np.int64))


def interface_indices(w, n: int, seed: int) -> np.ndarray:
    """Flat indices of voxels whose +x neighbour carries a different label (tissue interfaces), a seeded subset."""
    lab = w.labels
    z, y, x = np.nonzero(lab[:, :, :-1] != lab[:, :, 1:])
    rng = np.random.Generator(np.random.PCG64(seed))
    pick = rng.choice(len(z), size=min(n, len(z)), replace=False)
    nx, ny, nz = w.dims
    return (x[pick] + nx * (y[pick] + ny * z[pick])).astype(np.int64)


FIELD_Q = 1.0e-5        # deg C per code of the compact field
FIELD_EPS = 1.0e-6      # voxels that moved less than this from T_init stay outside the stored box


def compact_field(T, w) -> dict:
    """The whole fp64 field as integer codes over the bounding box of the voxels that left T_init (see the
    module docstring).  Data handling only: no method arithmetic."""
    dev = T - np.asarray(w.table["t_init"], dtype=np.float64)[w.labels]
    moved = np.abs(dev) > FIELD_EPS
    if not moved.any():
        lo, hi = np.zeros(3, np.int64), np.ones(3, np.int64)
    else:
        lo = np.array([np.nonzero(moved.any(axis=tuple(a for a in range(3) if a != ax)))[0][0] for ax in range(3)])
        hi = np.array([np.nonzero(moved.any(axis=tuple(a for a in range(3) if a != ax)))[0][-1] + 1 for ax in range(3)])
    box = dev[lo[0]:hi[0], lo[1]:hi[1], lo[2]:hi[2]]
    codes = np.rint(box / FIELD_Q)
    assert np.abs(codes).max() < 2 ** 31 and np.abs(codes * FIELD_Q - box).max() <= 0.5 * FIELD_Q * (1 + 1e-9)
    out = np.abs(dev)
    out[lo[0]:hi[0], lo[1]:hi[1], lo[2]:hi[2]] = 0.0
    return {"field_q": np.float64(FIELD_Q), "field_lo": lo.astype(np.int64), "field_codes": codes.astype(np.int32),
            "field_outside_max": np.float64(out.max())}


def run_scenario(w, scenario: int, n_samples: int, crop: int, checkpoints, conservative: bool = False):
    nx, ny, nz = w.dims
    sim = rfa_oracle.OracleSim(w.dims, w.spacing_mm, w.labels, w.table, w.t_blood, w.dt, conservative=conservative)
    if w.t0 is not None:
        sim.set_temperature(w.t0)
    nd = w.needles[scenario]
    sim.set_needle(nd.mask, nd.mode, nd.value)
    idx = sample_indices(w, scenario, n_samples, 190705709 + 17 * scenario + len(w.name))
    if conservative:
        idx = np.unique(np.concatenate([idx, interface_indices(w, n_samples, 190705709 + 99)]))
    out_T = []
    prev = None
    done = 0
    t0 = time.time()
    for cp in checkpoints:
        sim.step(cp - done)
        done = cp
        cur = sim.T.ravel()[idx].copy()
        if prev is not None and w.t0 is None:      # constant heating from T_a: non-decreasing
            assert np.all(cur >= prev - 1e-12), "oracle field not monotone between checkpoints"
        prev = cur
        out_T.append(cur)
        print(f"  {w.name}[{scenario}] step {cp}: {time.time() - t0:.1f} s, Tmax {sim.T.max():.4f}", flush=True)
    secs = time.time() - t0
    T = sim.T
    mz, my, mx = np.nonzero(nd.mask)
    c = np.array([int(round(mz.mean())), int(round(my.mean())), int(round(mx.mean()))])
    lo = np.clip(c - crop // 2, 0, np.array([nz, ny, nx]) - crop)
    crop_T = T[lo[0]:lo[0] + crop, lo[1]:lo[1] + crop, lo[2]:lo[2] + crop].copy()
    flat = T.ravel()
    band = np.nonzero(np.abs(flat - 60.0) <= 2e-3)[0]
    field = compact_field(T, w)
    res = {
        "sample_idx": idx,
        "sample_T": np.stack(out_T),
        "crop_lo": lo,
        "crop_T": crop_T,
        "necro_packed": np.packbits(sim.necro.ravel()),
        "necro_count": np.int64(sim.necro.sum()),
        "necro_count_tissue": np.int64(((sim.necro != 0) & (sim.label_held == 0) & (sim.needle_mask == 0)).sum()),
        "necro_volume_mm3": np.float64(sim.necrotic_volume_mm3()),
        "band_idx": band,
        "band_T": flat[band],
        "T_sum": np.float64(flat.sum()),
        "T_max": np.float64(flat.max()),
        "fingerprint": np.array(fingerprint(w, scenario)),
        "oracle_gvox_per_s": np.float64(w.n_voxels * checkpoints[-1] / secs / 1e9),
        "oracle_threads": np.int64(rfa_oracle.num_threads()),
    }
    res.update(field)
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("configs", nargs="+")
    ap.add_argument("--threads", type=int, default=0)
    args = ap.parse_args()
    rfa_oracle.build()
    if args.threads:
        rfa_oracle.set_num_threads(args.threads)
    for name in args.configs:
        # "C4F" = the C4 body model with a non-uniform initial field, conservative conduction term (row f1)
        cons = name.endswith("F")
        w = W.BENCH_CONFIGS[name]()
        cps = [w.steps // 4, w.steps // 2, w.steps]
        print(f"{name}: dims {w.dims} steps {w.steps} batch {w.batch}", flush=True)
        out = {"dims": np.array(w.dims), "checkpoints": np.array(cps), "batch": np.int64(w.batch)}
        if w.batch == 1:
            out.update(run_scenario(w, 0, 4096, 32, cps, conservative=cons))
        else:
            for b in range(w.batch):
                r = run_scenario(w, b, 512, 16, [w.steps])
                for k, v in r.items():
                    out[f"s{b}_{k}"] = v
        path = os.path.join(HERE, f"{name}_golden.npz")
        np.savez_compressed(path, **out)
        print(f"wrote {path} ({os.path.getsize(path) / 1024:.0f} KiB)", flush=True)


if __name__ == "__main__":
    main()
