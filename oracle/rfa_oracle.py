"""fp64 CPU oracle for the RFA bioheat hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes driver around ``oracle/rfa_oracle.c`` (plain C, fp64, the un-factored Eq. 12 of
PAPER.md:117 voxel by voxel).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this module.  It imports nothing from the
CUDA package (the seeded input generators in ``paper_1907_05709_b200/workloads.py`` hold no method
arithmetic and are handed to both sides by the caller).

State handling follows the paper's set-up and DESIGN.md's readings:
  * label -> initial temperature image (Fig. 5):  T[v] = table[label[v]].t_init
  * vessel / fixed labels and Dirichlet needle voxels are held (Alg. 1 :306/:313)
  * the needle mask overrides the label (R-15); moving the needle releases the old voxels, which keep
    their current temperature and become ordinary tissue again (R-16)
  * constant-power needle voxels are updated like tissue with +Q in the bracket; a held label under the
    mask stays held (R-17)
  * necrosis: sticky OR over time of (T >= 60 C), tested on the initial / post-set_needle state and after
    every step (R-11, R-12, R-14)

Parity with the paper's printed curves: UNPINNED (the paper tabulates no temperature).  Everything
else is pinned by tests/test_oracle_pins.py (see the header of rfa_oracle.c).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rfa_oracle.c")
_LIB = os.path.join(_HERE, "librfa_oracle.so")

TISSUE_HELD = 1
SRC_OFF, SRC_DIRICHLET, SRC_POWER = 0, 1, 2
T_NECROSIS = 60.0  # deg C

_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (``-O2 -fopenmp``; never tuned beyond that)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        up = ctypes.POINTER(ctypes.c_uint8)
        common = [ctypes.c_int] * 3 + [ctypes.c_double] * 3 + [up, up, up] + [dp] * 5 + [ctypes.c_double] * 4
        lib.rfa_oracle_step.argtypes = common + [dp, dp, up]
        lib.rfa_oracle_step.restype = None
        lib.rfa_oracle_run.argtypes = common + [ctypes.c_int, dp, dp, up, ctypes.c_int]
        lib.rfa_oracle_run.restype = None
        lib.rfa_oracle_num_threads.restype = ctypes.c_int
        lib.rfa_oracle_set_num_threads.argtypes = [ctypes.c_int]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().rfa_oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().rfa_oracle_set_num_threads(int(n))


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _up(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8))


class OracleSim:
    """One scenario.  ``labels`` uint8 (nz, ny, nx); ``table`` structured rows with fields
    k, rho, cp, wb_cb, q_m, t_init, flags; ``spacing_mm`` (dx, dy, dz) in millimetres."""

    def __init__(self, dims, spacing_mm, labels, table, t_blood: float, dt: float,
                 t_necrosis: float = T_NECROSIS, conservative: bool = False):
        nx, ny, nz = (int(d) for d in dims)
        self.conservative = bool(conservative)      # row f1: harmonic-mean face conductivities (R-28)
        self.dims = (nx, ny, nz)
        self.h_m = tuple(float(s) * 1.0e-3 for s in spacing_mm)     # mm -> m (R-2)
        self.lab = np.ascontiguousarray(labels, dtype=np.uint8).reshape(nz, ny, nx).copy()
        if int(self.lab.max()) >= len(table):
            raise ValueError("label id outside the tissue table")
        self.K = np.ascontiguousarray(table["k"], dtype=np.float64)
        self.rho = np.ascontiguousarray(table["rho"], dtype=np.float64)
        self.cp = np.ascontiguousarray(table["cp"], dtype=np.float64)
        self.wb_cb = np.ascontiguousarray(table["wb_cb"], dtype=np.float64)
        self.q_m = np.ascontiguousarray(table["q_m"], dtype=np.float64)
        self.t_init = np.ascontiguousarray(table["t_init"], dtype=np.float64)
        self.flags = np.ascontiguousarray(table["flags"], dtype=np.uint32)
        self.t_a = float(t_blood)
        self.dt = float(dt)
        self.t_necro = float(t_necrosis)
        self.q_power = 0.0
        # label -> initial temperature image
        self.T = self.t_init[self.lab].astype(np.float64)
        self._buf = np.empty_like(self.T)
        self.label_held = ((self.flags[self.lab] & TISSUE_HELD) != 0).astype(np.uint8)
        self.needle_held = np.zeros_like(self.lab)
        self.power = np.zeros_like(self.lab)
        self.needle_mask = np.zeros_like(self.lab)
        self.necro = np.zeros_like(self.lab)
        self._refresh_necrosis()
        self.steps_done = 0

    # -- state -----------------------------------------------------------------------------
    def _refresh_necrosis(self):
        self.necro |= (self.T >= self.t_necro).astype(np.uint8)        # R-14

    def set_temperature(self, T):
        self.T[...] = np.asarray(T, dtype=np.float64).reshape(self.T.shape)
        self._refresh_necrosis()

    def set_needle(self, mask, mode: int, value: float):
        self.needle_held[...] = 0                                       # R-16: release old voxels
        self.power[...] = 0
        self.needle_mask[...] = 0
        self.q_power = 0.0
        if mode == SRC_OFF or mask is None:
            return
        m = np.asarray(mask).reshape(self.lab.shape) != 0
        self.needle_mask[m] = 1
        if mode == SRC_DIRICHLET:
            self.needle_held[m] = 1                                     # R-15: overrides the label
            self.T[m] = float(value)
        elif mode == SRC_POWER:
            self.power[m] = 1                                           # R-17
            self.q_power = float(value)
        else:
            raise ValueError("bad source mode")
        self._refresh_necrosis()

    @property
    def held(self):
        return (self.label_held | self.needle_held).astype(np.uint8)

    # -- stepping --------------------------------------------------------------------------
    def step(self, n: int = 1):
        lib = _load()
        nx, ny, nz = self.dims
        held = np.ascontiguousarray(self.held)
        lib.rfa_oracle_run(nx, ny, nz, self.h_m[0], self.h_m[1], self.h_m[2],
                           _up(self.lab), _up(held), _up(self.power),
                           _dp(self.K), _dp(self.rho), _dp(self.cp), _dp(self.wb_cb), _dp(self.q_m),
                           self.t_a, self.q_power, self.dt, self.t_necro,
                           int(n), _dp(self.T), _dp(self._buf), _up(self.necro), int(self.conservative))
        self.steps_done += int(n)

    def step_record(self, n: int, every: int, index) -> np.ndarray:
        """Probe time series (Fig. 6, Fig. 14): row m = T at the flat voxel indices after
        (m+1)*every steps."""
        idx = np.asarray(index, dtype=np.int64)
        rows = []
        for _ in range(int(n) // int(every)):
            self.step(every)
            rows.append(self.T.ravel()[idx].copy())
        return np.array(rows, dtype=np.float64).reshape(len(rows), idx.size)

    # -- results ---------------------------------------------------------------------------
    def temperature(self) -> np.ndarray:
        return self.T.copy()

    def necrosis(self) -> np.ndarray:
        return self.necro.copy()

    def necrotic_volume_mm3(self, exclude_held: bool = True) -> float:
        """Volume of the necrosis mask; by default without needle-mask and held-label voxels (R-13)."""
        m = self.necro != 0
        if exclude_held:
            m &= (self.label_held == 0) & (self.needle_mask == 0)
        vox = self.h_m[0] * self.h_m[1] * self.h_m[2] * 1e9
        return float(m.sum()) * vox

    def stability_number(self) -> float:
        """max over labels of dt*(2 alpha (1/dx^2+1/dy^2+1/dz^2) + beta/(rho cp)); the explicit update
        is a monotone (entrywise non-negative) map iff this is <= 1 (R-18)."""
        s = sum(1.0 / (h * h) for h in self.h_m)
        alpha = self.K / (self.rho * self.cp)
        if self.conservative:
            # worst face conductivity seen by a voxel of label l: 2 K_l K_max / (K_l + K_max)
            kmax = float(self.K.max())
            alpha = (2.0 * self.K * kmax / (self.K + kmax)) / (self.rho * self.cp)
        return float(np.max(self.dt * (2.0 * alpha * s + self.wb_cb / (self.rho * self.cp))))


def run_workload(w, steps: int | None = None, scenario: int = 0, conservative: bool = False) -> OracleSim:
    """Run one scenario of a ``workloads.Workload`` for ``steps`` (default: the configured count)."""
    sim = OracleSim(w.dims, w.spacing_mm, w.labels, w.table, w.t_blood, w.dt, conservative=conservative)
    if w.t0 is not None:
        sim.set_temperature(w.t0)
    if w.needles:
        nd = w.needles[scenario]
        sim.set_needle(nd.mask, nd.mode, nd.value)
    sim.step(w.steps if steps is None else steps)
    return sim
