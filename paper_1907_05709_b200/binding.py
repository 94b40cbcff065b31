"""Thin ctypes binding over the C ABI of librfa.so (include/rfa.h): argument marshalling only.

PyTorch is used for exactly two things: the device workspace (a uint8 CUDA tensor handed to
``rfa_create``) and the CUDA stream.  Every step of the hot path runs in the library's kernels; there
is no Python / PyTorch / CPU fallback -- if librfa.so is missing, loading raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# RFA_LIBRARY lets a developer load another build of the same library (e.g. a tile-shape experiment)
LIB_PATH = os.environ.get("RFA_LIBRARY") or os.path.join(_HERE, "librfa.so")

RFA_OK, RFA_E_INVALID, RFA_E_UNSTABLE, RFA_E_CUDA, RFA_E_NOMEM = 0, -1, -2, -3, -4
SRC_OFF, SRC_DIRICHLET, SRC_POWER = 0, 1, 2
KERNEL_AUTO, KERNEL_PLAIN, KERNEL_BLOCKED, KERNEL_STREAM = 0, 1, 2, 3
TISSUE_HELD = 1
MAX_TISSUES = 16
COND_EQ12, COND_FACE = 0, 1
HELD_COPY_AUTO, HELD_COPY_OFF, HELD_COPY_ON = -1, 0, 1
STAGING_AUTO, STAGING_CP_ASYNC, STAGING_TMA = -1, 0, 1
RES_PREFETCH_AUTO, RES_PREFETCH_OFF, RES_PREFETCH_ON = -1, 0, 1
STATIC_RECORD_MAX_PROBES, STATIC_RECORD_MAX_FLOATS = 1024, 262144   # rfa_step_record_static (include/rfa.h)

# every symbol include/rfa.h declares
EXPORTS = [
    "rfa_workspace_bytes", "rfa_stability_number", "rfa_create", "rfa_set_needle", "rfa_set_temperature",
    "rfa_step", "rfa_get_temperature", "rfa_get_necrosis", "rfa_necrotic_voxels", "rfa_configure",
    "rfa_set_conduction", "rfa_query", "rfa_query_variant", "rfa_configure_held_copy", "rfa_configure_staging", "rfa_configure_tile", "rfa_configure_residual_prefetch", "rfa_query_hot_fraction", "rfa_plan_query", "rfa_set_probes", "rfa_step_record", "rfa_step_record_static", "rfa_current_frame",
    "rfa_warp_temperature", "rfa_render_zone",
    "rfa_synchronize", "rfa_destroy", "rfa_last_error",
]


class RfaTissue(ctypes.Structure):
    _fields_ = [("k", ctypes.c_float), ("rho", ctypes.c_float), ("cp", ctypes.c_float),
                ("wb_cb", ctypes.c_float), ("q_m", ctypes.c_float), ("t_init", ctypes.c_float),
                ("flags", ctypes.c_uint32)]


class RfaView(ctypes.Structure):
    _fields_ = [("dir", ctypes.c_float * 3), ("up", ctypes.c_float * 3), ("width", ctypes.c_int),
                ("height", ctypes.c_int), ("pixel_mm", ctypes.c_float), ("step_mm", ctypes.c_float),
                ("iso_c", ctypes.c_float)]


class RfaError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"librfa error {code}: {msg}")
        self.code = code


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen librfa.so and declare the prototypes.  Raises if the library has not been built
    (``python -m paper_1907_05709_b200.build`` or ``__graft_entry__.build()``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build the CUDA library first "
                           "(python paper_1907_05709_b200/build.py). There is no CPU fallback.")
    lib = ctypes.CDLL(LIB_PATH)
    i3 = ctypes.POINTER(ctypes.c_int)
    f3 = ctypes.POINTER(ctypes.c_float)
    vp = ctypes.c_void_p
    lib.rfa_workspace_bytes.argtypes = [i3, ctypes.c_int]
    lib.rfa_workspace_bytes.restype = ctypes.c_size_t
    lib.rfa_stability_number.argtypes = [f3, ctypes.POINTER(RfaTissue), ctypes.c_int, ctypes.c_float]
    lib.rfa_stability_number.restype = ctypes.c_double
    lib.rfa_create.argtypes = [ctypes.POINTER(vp), i3, f3, vp, ctypes.POINTER(RfaTissue), ctypes.c_int,
                               ctypes.c_float, ctypes.c_float, ctypes.c_int, vp, ctypes.c_size_t, vp]
    lib.rfa_create.restype = ctypes.c_int
    lib.rfa_set_needle.argtypes = [vp, ctypes.c_int, f3, f3, vp, ctypes.c_int, ctypes.c_float]
    lib.rfa_set_needle.restype = ctypes.c_int
    lib.rfa_set_temperature.argtypes = [vp, ctypes.c_int, vp]
    lib.rfa_set_temperature.restype = ctypes.c_int
    lib.rfa_step.argtypes = [vp, ctypes.c_int]
    lib.rfa_step.restype = ctypes.c_int
    lib.rfa_get_temperature.argtypes = [vp, ctypes.c_int, vp]
    lib.rfa_get_temperature.restype = ctypes.c_int
    lib.rfa_get_necrosis.argtypes = [vp, ctypes.c_int, vp]
    lib.rfa_get_necrosis.restype = ctypes.c_int
    lib.rfa_necrotic_voxels.argtypes = [vp, ctypes.c_int, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64)]
    lib.rfa_necrotic_voxels.restype = ctypes.c_int
    lib.rfa_configure.argtypes = [vp, ctypes.c_int, ctypes.c_int]
    lib.rfa_configure.restype = ctypes.c_int
    lib.rfa_set_conduction.argtypes = [vp, ctypes.c_int]
    lib.rfa_set_conduction.restype = ctypes.c_int
    lib.rfa_query.argtypes = [vp, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int64)]
    lib.rfa_query.restype = ctypes.c_int
    lib.rfa_query_variant.argtypes = [vp, ctypes.POINTER(ctypes.c_int)]
    lib.rfa_query_variant.restype = ctypes.c_int
    lib.rfa_configure_held_copy.argtypes = [vp, ctypes.c_int]
    lib.rfa_configure_held_copy.restype = ctypes.c_int
    lib.rfa_configure_staging.argtypes = [vp, ctypes.c_int]
    lib.rfa_configure_staging.restype = ctypes.c_int
    lib.rfa_configure_residual_prefetch.argtypes = [vp, ctypes.c_int]
    lib.rfa_configure_residual_prefetch.restype = ctypes.c_int
    lib.rfa_query_hot_fraction.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)]
    lib.rfa_query_hot_fraction.restype = ctypes.c_int
    lib.rfa_configure_tile.argtypes = [vp, ctypes.c_int]
    lib.rfa_configure_tile.restype = ctypes.c_int
    lib.rfa_plan_query.argtypes = [i3, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_int)]
    lib.rfa_plan_query.restype = ctypes.c_int
    lib.rfa_set_probes.argtypes = [vp, ctypes.c_int, ctypes.POINTER(ctypes.c_int64)]
    lib.rfa_set_probes.restype = ctypes.c_int
    lib.rfa_step_record.argtypes = [vp, ctypes.c_int, ctypes.c_int, vp]
    lib.rfa_step_record.restype = ctypes.c_int
    lib.rfa_step_record_static.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_int64), vp]
    lib.rfa_step_record_static.restype = ctypes.c_int
    lib.rfa_current_frame.argtypes = [vp, ctypes.c_int, ctypes.POINTER(vp), ctypes.POINTER(ctypes.c_float)]
    lib.rfa_current_frame.restype = ctypes.c_int
    lib.rfa_warp_temperature.argtypes = [vp, ctypes.c_int, vp, ctypes.c_float, vp]
    lib.rfa_warp_temperature.restype = ctypes.c_int
    lib.rfa_render_zone.argtypes = [vp, ctypes.c_int, ctypes.POINTER(RfaView), vp, vp]
    lib.rfa_render_zone.restype = ctypes.c_int
    lib.rfa_synchronize.argtypes = [vp]
    lib.rfa_synchronize.restype = ctypes.c_int
    lib.rfa_destroy.argtypes = [vp]
    lib.rfa_destroy.restype = None
    lib.rfa_last_error.argtypes = []
    lib.rfa_last_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _check(rc: int):
    if rc != RFA_OK:
        raise RfaError(rc, load_library().rfa_last_error().decode("utf-8", "replace"))


def tissue_array(table) -> ctypes.Array:
    """numpy structured rows (k, rho, cp, wb_cb, q_m, t_init, flags) -> rfa_tissue[]"""
    arr = (RfaTissue * len(table))()
    for i, r in enumerate(table):
        arr[i] = RfaTissue(float(r["k"]), float(r["rho"]), float(r["cp"]), float(r["wb_cb"]),
                           float(r["q_m"]), float(r["t_init"]), int(r["flags"]))
    return arr


def _i3(v):
    return (ctypes.c_int * 3)(*[int(x) for x in v])


def _f3(v):
    return (ctypes.c_float * 3)(*[float(x) for x in v])


def stability_number(spacing_mm, table, dt) -> float:
    lib = load_library()
    return float(lib.rfa_stability_number(_f3(spacing_mm), tissue_array(table), len(table), float(dt)))


def plan_query(dims, batch, fused, resident_ctas, staging: int = 0) -> dict:
    lib = load_library()
    out = (ctypes.c_int * 9)()
    _check(lib.rfa_plan_query(_i3(dims), int(batch), int(fused), int(resident_ctas), int(staging), out))
    keys = ["ok", "tiles_x", "tiles_y", "z_chunks", "planes_per_chunk", "work_items", "ctas", "bx", "by"]
    return dict(zip(keys, [int(x) for x in out]))


def _ptr(x):
    """host numpy array or torch tensor (host or CUDA) -> raw address (the library tells them apart)"""
    if isinstance(x, np.ndarray):
        return ctypes.c_void_p(x.ctypes.data)
    return ctypes.c_void_p(x.data_ptr())


def _check_out(x, n_elem: int, what: str, np_dtype=np.float32):
    """An output buffer handed to the library by raw address: it must hold >= n_elem contiguous elements of the
    right type, or the library would write past its end (host) / fault (device)."""
    if isinstance(x, np.ndarray):
        ok = x.dtype == np_dtype and x.flags["C_CONTIGUOUS"] and x.flags["WRITEABLE"]
        size = x.size
    else:
        import torch
        want = {np.float32: torch.float32, np.uint8: torch.uint8}[np_dtype]
        ok = x.dtype == want and x.is_contiguous()
        size = x.numel()
    if not ok:
        raise ValueError(f"{what}: need a contiguous {np.dtype(np_dtype).name} buffer")
    if size < n_elem:
        raise ValueError(f"{what}: buffer of {size} elements, need {n_elem}")


class RfaSim:
    """One simulation: ``batch`` scenarios sharing a label volume.  Mirrors include/rfa.h one to one."""

    def __init__(self, dims, spacing_mm, labels, table, t_blood: float, dt: float, batch: int = 1,
                 device="cuda:0", stream=None):
        import torch
        self._torch = torch
        lib = load_library()
        self._lib = lib
        self.dims = tuple(int(d) for d in dims)
        self.batch = int(batch)
        self.nvox = self.dims[0] * self.dims[1] * self.dims[2]
        self.device = torch.device(device)
        lab = np.ascontiguousarray(labels, dtype=np.uint8).reshape(-1)
        if lab.size != self.nvox:
            raise ValueError("labels do not match dims")
        need = int(lib.rfa_workspace_bytes(_i3(dims), self.batch))
        self._handle = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            # PyTorch's only roles: device memory and the stream
            self.workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=self.device)
            st = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.stream = st
            rc = lib.rfa_create(ctypes.byref(self._handle), _i3(dims), _f3(spacing_mm),
                                ctypes.c_void_p(lab.ctypes.data), tissue_array(table), len(table),
                                float(t_blood), float(dt), self.batch,
                                ctypes.c_void_p(self.workspace.data_ptr()), need, ctypes.c_void_p(st.cuda_stream))
        _check(rc)

    # -- lifetime ----------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_handle", None) is not None and self._handle.value:
            self._lib.rfa_destroy(self._handle)
            self._handle = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the ABI, same names -------------------------------------------------------------------
    def set_needle(self, scenario: int, mask, mode: int, value: float, tip_mm=None, axis=None):
        m = None
        if mode != SRC_OFF:
            m = mask if not isinstance(mask, np.ndarray) else np.ascontiguousarray(mask, dtype=np.uint8)
        _check(self._lib.rfa_set_needle(self._handle, int(scenario),
                                        _f3(tip_mm) if tip_mm is not None else None,
                                        _f3(axis) if axis is not None else None,
                                        _ptr(m) if m is not None else None, int(mode), float(value)))

    def set_temperature(self, scenario: int, t_c):
        t = t_c if not isinstance(t_c, np.ndarray) else np.ascontiguousarray(t_c, dtype=np.float32)
        _check(self._lib.rfa_set_temperature(self._handle, int(scenario), _ptr(t)))

    def step(self, n: int = 1):
        _check(self._lib.rfa_step(self._handle, int(n)))

    def get_temperature(self, scenario: int = 0, out=None):
        nx, ny, nz = self.dims
        if out is None:
            out = np.empty((nz, ny, nx), dtype=np.float32)
        _check_out(out, nx * ny * nz, "get_temperature out", np.float32)
        _check(self._lib.rfa_get_temperature(self._handle, int(scenario), _ptr(out)))
        return out

    def get_necrosis(self, scenario: int = 0, out=None):
        nx, ny, nz = self.dims
        if out is None:
            out = np.empty((nz, ny, nx), dtype=np.uint8)
        _check_out(out, nx * ny * nz, "get_necrosis out", np.uint8)
        _check(self._lib.rfa_get_necrosis(self._handle, int(scenario), _ptr(out)))
        return out

    def necrotic_voxels(self, scenario: int = 0):
        a, t = ctypes.c_int64(), ctypes.c_int64()
        _check(self._lib.rfa_necrotic_voxels(self._handle, int(scenario), ctypes.byref(a), ctypes.byref(t)))
        return int(a.value), int(t.value)

    def configure(self, kernel: int = KERNEL_AUTO, fused_steps: int = 0):
        _check(self._lib.rfa_configure(self._handle, int(kernel), int(fused_steps)))

    def configure_held_copy(self, mode: int = HELD_COPY_AUTO):
        _check(self._lib.rfa_configure_held_copy(self._handle, int(mode)))

    def configure_staging(self, mode: int = STAGING_AUTO):
        _check(self._lib.rfa_configure_staging(self._handle, int(mode)))

    def configure_residual_prefetch(self, mode: int = RES_PREFETCH_AUTO):
        _check(self._lib.rfa_configure_residual_prefetch(self._handle, int(mode)))

    def hot_fraction(self) -> dict:
        f, on = ctypes.c_double(), ctypes.c_int()
        _check(self._lib.rfa_query_hot_fraction(self._handle, ctypes.byref(f), ctypes.byref(on)))
        return {"hot_fraction": float(f.value), "residual_prefetch": int(on.value)}

    def configure_tile(self, shape: int = -1):
        _check(self._lib.rfa_configure_tile(self._handle, int(shape)))

    def set_conduction(self, mode: int):
        _check(self._lib.rfa_set_conduction(self._handle, int(mode)))

    def query(self) -> dict:
        k, f, n = ctypes.c_int(), ctypes.c_int(), ctypes.c_int64()
        _check(self._lib.rfa_query(self._handle, ctypes.byref(k), ctypes.byref(f), ctypes.byref(n)))
        return {"kernel": int(k.value), "fused_steps": int(f.value), "kernel_launches": int(n.value)}

    def query_variant(self) -> dict:
        out = (ctypes.c_int * 8)()
        _check(self._lib.rfa_query_variant(self._handle, out))
        return dict(zip(["fused_steps", "tile_bx", "tile_by", "ctas", "held_copy", "conduction", "staging", "residual_prefetch"],
                        [int(x) for x in out]))

    def set_probes(self, index):
        idx = np.ascontiguousarray(index, dtype=np.int64).reshape(-1)
        self.n_probes = int(idx.size)
        _check(self._lib.rfa_set_probes(self._handle, self.n_probes,
                                        idx.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)) if idx.size else None))

    def step_record(self, n: int, every: int = 1, out=None):
        rows = int(n) // max(int(every), 1)
        if out is None:
            out = np.empty((rows, getattr(self, "n_probes", 0)), dtype=np.float32)
        _check_out(out, rows * getattr(self, "n_probes", 0), "step_record out")
        _check(self._lib.rfa_step_record(self._handle, int(n), int(every), _ptr(out)))
        return out

    def step_record_static(self, n: int, every: int, index, out=None):
        """``step_record`` for callers that must not allocate device memory at this point (a running frame loop, which a
        cudaMalloc would stall; an application whose memory pool owns the whole card): the probe list ``index`` is passed
        here instead of to ``set_probes``, and list and rows go through a fixed 1 MiB array inside librfa.so, so at most
        ``STATIC_RECORD_MAX_PROBES`` probes and ``STATIC_RECORD_MAX_FLOATS`` recorded values per call.  One array per GPU:
        do not run two of these calls on one GPU at the same time.  Same bits as ``step_record``."""
        idx = np.ascontiguousarray(index, dtype=np.int64).reshape(-1)
        rows = int(n) // max(int(every), 1)
        if out is None:
            out = np.empty((rows, int(idx.size)), dtype=np.float32)
        _check_out(out, rows * int(idx.size), "step_record_static out")
        _check(self._lib.rfa_step_record_static(self._handle, int(n), int(every), int(idx.size),
                                                idx.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)) if idx.size else None,
                                                _ptr(out)))
        return out

    def current_frame(self, scenario: int = 0):
        """(device address of theta = T - t_blood of the finished image, t_blood): Alg. 2 hand-off"""
        p, tb = ctypes.c_void_p(), ctypes.c_float()
        _check(self._lib.rfa_current_frame(self._handle, int(scenario), ctypes.byref(p), ctypes.byref(tb)))
        return int(p.value), float(tb.value)

    def warp_temperature(self, scenario: int, disp, scale: float = 1.0, out=None):
        """Eq. 14: the temperature image seen through a displacement field (3, nz, ny, nx) in mm"""
        nx, ny, nz = self.dims
        d = disp if not isinstance(disp, np.ndarray) else np.ascontiguousarray(disp, dtype=np.float32)
        if out is None:
            out = np.empty((nz, ny, nx), dtype=np.float32)
        _check_out(out, nx * ny * nz, "warp_temperature out")
        _check(self._lib.rfa_warp_temperature(self._handle, int(scenario), _ptr(d), float(scale), _ptr(out)))
        return out

    def render_zone(self, scenario: int, direction, up, width: int, height: int, pixel_mm: float, step_mm: float,
                    iso_c: float = 42.5, want_depth: bool = True, tmax=None, depth=None):
        """Orthographic ray-march of the heat zone: (tmax image, depth-of-isotherm image), each (height, width).
        ``tmax`` / ``depth``: optional caller buffers of width*height floats (numpy or CUDA tensors); returned as given."""
        v = RfaView((ctypes.c_float * 3)(*[float(x) for x in direction]), (ctypes.c_float * 3)(*[float(x) for x in up]),
                    int(width), int(height), float(pixel_mm), float(step_mm), float(iso_c))
        if tmax is None:
            tmax = np.empty((height, width), dtype=np.float32)
        if depth is None and want_depth:
            depth = np.empty((height, width), dtype=np.float32)
        _check_out(tmax, int(width) * int(height), "render_zone tmax")
        if depth is not None:
            _check_out(depth, int(width) * int(height), "render_zone depth")
        _check(self._lib.rfa_render_zone(self._handle, int(scenario), ctypes.byref(v), _ptr(tmax),
                                         _ptr(depth) if depth is not None else None))
        return tmax, depth

    def synchronize(self):
        _check(self._lib.rfa_synchronize(self._handle))


def from_workload(w, device="cuda:0", stream=None) -> RfaSim:
    """Convenience: create a simulation from a ``workloads.Workload`` and place its needles."""
    sim = RfaSim(w.dims, w.spacing_mm, w.labels, w.table, w.t_blood, w.dt, batch=w.batch,
                 device=device, stream=stream)
    if w.t0 is not None:
        for b in range(w.batch):
            sim.set_temperature(b, np.asarray(w.t0, dtype=np.float32))
    for b, nd in enumerate(w.needles):
        sim.set_needle(b, nd.mask, nd.mode, nd.value, nd.tip_mm, nd.axis)
    return sim
