"""Thin Python binding of the C ABI in ``include/avm.h`` (argument marshalling only).

Every step of the hot path runs inside ``libavm_b200.so``; this module only
  * loads the library (and fails loudly if it has not been built — there is no fallback),
  * allocates device memory with PyTorch and passes ``data_ptr()`` / the current CUDA stream,
  * mirrors the entry points one to one: ``avm_create``, ``avm_step``, ``avm_get_state``,
    ``avm_compute_forces`` (+ the ``*_host`` twins and the test hooks).
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# AVM_B200_LIB overrides the location (an alternative build of the same library)
LIB_PATH = os.environ.get("AVM_B200_LIB") or os.path.join(_HERE, "libavm_b200.so")
# the same ABI with reduced-precision storage (NEXT-3); loaded on demand, never the default
LIB_MIXED_PATH = os.path.join(_HERE, "libavm_b200_mixed.so")

# every symbol include/avm.h declares (tests check that the library exports all of them)
ABI_SYMBOLS = [
    "avm_workspace_bytes", "avm_create", "avm_create_host", "avm_step", "avm_step_profile", "avm_compute_forces",
    "avm_forces_static",
    "avm_compute_forces_host", "avm_energy", "avm_observe", "avm_step_observe", "avm_spv_geometry", "avm_spv_forces", "avm_spv_step", "avm_spv_test_triangulation", "avm_set_cell_targets", "avm_set_cell_moduli", "avm_msd_reset", "avm_get_state", "avm_get_state_host", "avm_debug_t1",
    "avm_t1_pass", "avm_set_positions", "avm_resort", "avm_philox_words", "avm_hilbert_index",
    "avm_hilbert_index_host", "avm_destroy", "avm_strerror", "avm_last_cuda_error", "avm_precision",
]

AVM_FLAG_SORT_AT_CREATE = 1
AVM_FLAG_SCHEDULE_FUSED = 4
AVM_FLAG_SCHEDULE_UNFUSED = 8
AVM_FLAG_SCHEDULE_PERSISTENT = 16
AVM_FLAG_T1_PASSES_SHIFT = 8


class AvmParams(ctypes.Structure):
    _fields_ = [("n_cells", ctypes.c_int32), ("n_vertices", ctypes.c_int32),
                ("max_cell_vertices", ctypes.c_int32), ("sort_every", ctypes.c_int32),
                ("Lx", ctypes.c_double), ("Ly", ctypes.c_double),
                ("KA", ctypes.c_double), ("KP", ctypes.c_double), ("A0", ctypes.c_double), ("P0", ctypes.c_double),
                ("v0", ctypes.c_double), ("Dr", ctypes.c_double), ("mu", ctypes.c_double), ("dt", ctypes.c_double),
                ("l_c", ctypes.c_double),
                ("seed", ctypes.c_uint64), ("step0", ctypes.c_uint64),
                ("device", ctypes.c_int32), ("flags", ctypes.c_int32)]


class AvmStats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int64) for n in
                ("step", "t1_short", "t1_candidates", "t1_flips", "t1_blocked", "overflow_rejects", "error",
                 "n_sorts", "kernel_launches")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class AvmObservables(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in ("energy", "sum_area", "sum_perimeter", "mean_shape_index", "area_min",
                                               "area_max", "area_variance")] + \
               [(n, ctypes.c_int64) for n in ("n_nonpositive_area", "step", "t1_flips")] + [("msd", ctypes.c_double)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class AvmError(RuntimeError):
    pass


def _load(path: str = LIB_PATH) -> ctypes.CDLL:
    if not os.path.exists(path):
        raise AvmError(
            f"{path} is missing: build the CUDA library first (python -m paper_1702_02939_b200.build). "
            "There is no CPU fallback.")
    lib = ctypes.CDLL(path)
    p, i64, u64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_uint64, ctypes.c_int32
    PP = ctypes.POINTER(AvmParams)
    lib.avm_workspace_bytes.restype = ctypes.c_size_t
    lib.avm_workspace_bytes.argtypes = [PP]
    for name in ("avm_create", "avm_create_host"):
        f = getattr(lib, name)
        f.restype = ctypes.c_int
        f.argtypes = [PP, p, p, p, p, p, p, p, ctypes.c_size_t, p, ctypes.POINTER(p)]
    lib.avm_step.argtypes = [p, i64]
    lib.avm_step_profile.argtypes = [p, i64, p]
    lib.avm_compute_forces.argtypes = [p, p, p]
    lib.avm_compute_forces_host.argtypes = [p, p, p]
    lib.avm_forces_static.argtypes = [PP, p, p, p, p, p, p, p, p]
    lib.avm_energy.argtypes = [p, ctypes.POINTER(ctypes.c_double)]
    lib.avm_observe.argtypes = [p, ctypes.POINTER(AvmObservables)]
    lib.avm_step_observe.argtypes = [p, i64, ctypes.POINTER(AvmObservables)]
    lib.avm_spv_geometry.argtypes = [p, p, p, p]
    lib.avm_spv_forces.argtypes = [p, p, p, p]
    lib.avm_spv_step.argtypes = [p, p, i64, p, p]
    lib.avm_spv_test_triangulation.argtypes = [p, p, p, p]
    for name in ("avm_get_state", "avm_get_state_host"):
        getattr(lib, name).argtypes = [p, p, p, p, p, p, p, ctypes.POINTER(AvmStats)]
    lib.avm_debug_t1.argtypes = [p, p, ctypes.POINTER(i64), p, ctypes.POINTER(i64), i64]
    lib.avm_t1_pass.argtypes = [p]
    lib.avm_set_positions.argtypes = [p, p]
    lib.avm_set_cell_targets.argtypes = [p, p, p]
    lib.avm_set_cell_moduli.argtypes = [p, p, p]
    lib.avm_msd_reset.argtypes = [p]
    lib.avm_resort.argtypes = [p]
    lib.avm_philox_words.argtypes = [p, u64, u64, u64, i64, p]
    lib.avm_hilbert_index.argtypes = [p, i32, i64, p, p, p]
    lib.avm_hilbert_index_host.argtypes = [i32, ctypes.c_uint32, ctypes.c_uint32]
    lib.avm_hilbert_index_host.restype = ctypes.c_uint32
    lib.avm_destroy.argtypes = [p]
    lib.avm_destroy.restype = None
    lib.avm_strerror.argtypes = [ctypes.c_int]
    lib.avm_strerror.restype = ctypes.c_char_p
    lib.avm_last_cuda_error.restype = ctypes.c_char_p
    lib.avm_precision.restype = ctypes.c_char_p
    return lib


lib = _load()
_LIBS = {"f64": lib}


_VARIANTS = {}


def register_library(name: str, path: str) -> None:
    """an alternative build of the same sources and ABI under a name of its own (test builds with timing knobs);
    `from_tiling(..., precision=name)` then runs on it"""
    _VARIANTS[name] = _load(path)


def library(precision: str = "f64") -> ctypes.CDLL:
    """the C-ABI library for a storage precision: "f64" (default) or "mixed" (libavm_b200_mixed.so, NEXT-3)"""
    if precision in _VARIANTS:
        return _VARIANTS[precision]
    if precision not in _LIBS:
        if precision != "mixed":
            raise AvmError(f"unknown precision {precision!r}")
        _LIBS[precision] = _load(LIB_MIXED_PATH)
    assert _LIBS[precision].avm_precision().decode() == precision
    return _LIBS[precision]


def _check(rc: int) -> None:
    if rc != 0:
        msg = lib.avm_strerror(rc).decode()
        if rc == -4:
            msg += ": " + lib.avm_last_cuda_error().decode()
        raise AvmError(f"avm error {rc}: {msg}")


def hilbert_index_host(m: int, ix: int, iy: int) -> int:
    return int(lib.avm_hilbert_index_host(m, ix, iy))


def make_params(N: int, S: int, *, Lx, Ly, KA=1.0, KP=1.0, A0=1.0, P0=3.8, v0=0.0, Dr=0.0, mu=1.0, dt=0.01,
                l_c=0.0, seed=0, step0=0, sort_every=0, sort_at_create=False, device=0, flags=0, t1_max_passes=1,
                schedule="auto", **_ignored) -> AvmParams:
    if sort_at_create:
        flags |= AVM_FLAG_SORT_AT_CREATE
    flags |= {"auto": 0, "fused": AVM_FLAG_SCHEDULE_FUSED, "unfused": AVM_FLAG_SCHEDULE_UNFUSED,
              "persistent": AVM_FLAG_SCHEDULE_PERSISTENT}[schedule]
    if t1_max_passes > 1:
        flags |= (min(int(t1_max_passes), 255) << AVM_FLAG_T1_PASSES_SHIFT)
    return AvmParams(N, 2 * N, S, sort_every, Lx, Ly, KA, KP, A0, P0, v0, Dr, mu, dt, l_c, seed, step0, device, flags)


def _dptr(t) -> Optional[int]:
    return None if t is None else ctypes.c_void_p(t.data_ptr())


AVM_FORCES_STATIC_MAX_CELLS = 65536


def forces_static(params: AvmParams, pos, cell_vertex_num, cell_vertices, vertex_neighbors, vertex_cell_neighbors,
                  force_out, area_perim_out, precision: str = "f64") -> None:
    """``avm_forces_static``: geometry and forces of a tiling given as CUDA tensors in user order, written into the
    caller's ``force_out`` [V,2] / ``area_perim_out`` [N,2] (either may be None), on the current stream.  Needs no
    AvmSim and no workspace, and the library allocates nothing: the per-cell (A, P) pairs pass through a 1 MiB array
    built into the library.  Raises AvmError (code -6) beyond AVM_FORCES_STATIC_MAX_CELLS cells.  Calls that can
    overlap on the GPU share that array and must be ordered by the caller (see include/avm.h)."""
    import torch
    stream = torch.cuda.current_stream(torch.device("cuda", params.device))
    _check(library(precision).avm_forces_static(
        ctypes.byref(params), _dptr(pos), _dptr(cell_vertex_num), _dptr(cell_vertices), _dptr(vertex_neighbors),
        _dptr(vertex_cell_neighbors), _dptr(force_out), _dptr(area_perim_out), ctypes.c_void_p(stream.cuda_stream)))


def _hptr(a: Optional[np.ndarray]):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


class AvmSim:
    """One simulation living on a CUDA device.  Tensors in/out are torch CUDA tensors (device
    entry points) or numpy arrays (``*_host`` entry points), always in user order."""

    def __init__(self, tiling, params: AvmParams, host: bool = False, precision: str = "f64"):
        import torch
        self.torch = torch
        self.lib = library(precision)
        self.precision = precision
        self.params = params
        self.N, self.V, self.S = params.n_cells, params.n_vertices, params.max_cell_vertices
        self.device = torch.device("cuda", params.device)
        nbytes = self.lib.avm_workspace_bytes(ctypes.byref(params))
        if nbytes == 0:
            raise AvmError("avm_workspace_bytes rejected the parameters")
        self.workspace_bytes = int(nbytes)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        assert self.workspace.data_ptr() % 256 == 0
        self.stream = torch.cuda.current_stream(self.device)
        self._h = ctypes.c_void_p()
        arrays = [np.ascontiguousarray(tiling.pos, dtype=np.float64),
                  np.ascontiguousarray(tiling.cell_vertex_num, dtype=np.int32),
                  np.ascontiguousarray(tiling.cell_vertices, dtype=np.int32),
                  np.ascontiguousarray(tiling.vertex_neighbors, dtype=np.int32),
                  np.ascontiguousarray(tiling.vertex_cell_neighbors, dtype=np.int32),
                  np.ascontiguousarray(tiling.theta, dtype=np.float64)]
        assert arrays[2].shape == (self.N, self.S) and arrays[0].shape == (self.V, 2)
        if host:
            self._inputs = arrays
            ptrs = [_hptr(a) for a in arrays]
            fn = self.lib.avm_create_host
        else:
            self._inputs = [torch.from_numpy(a).to(self.device) for a in arrays]
            ptrs = [_dptr(t) for t in self._inputs]
            fn = self.lib.avm_create
        _check(fn(ctypes.byref(params), *ptrs, ctypes.c_void_p(self.workspace.data_ptr()),
                  self.workspace_bytes, ctypes.c_void_p(self.stream.cuda_stream), ctypes.byref(self._h)))
        self._inputs = None

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self.torch.cuda.synchronize(self.device)
            self.lib.avm_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- hot path ------------------------------------------------------------------------------
    def step(self, n: int = 1) -> None:
        _check(self.lib.avm_step(self._h, n))

    KERNEL_NAMES = ("force_move", "cell_update", "t1_flip")

    def step_profile(self, n: int) -> dict:
        """n steps with every kernel bracketed by CUDA events; summed device ms per kernel class."""
        ms = (ctypes.c_double * len(self.KERNEL_NAMES))()
        _check(self.lib.avm_step_profile(self._h, n, ms))
        return dict(zip(self.KERNEL_NAMES, list(ms)))

    def compute_forces(self):
        t = self.torch
        F = t.empty((self.V, 2), dtype=t.float64, device=self.device)
        ap = t.empty((self.N, 2), dtype=t.float64, device=self.device)
        _check(self.lib.avm_compute_forces(self._h, _dptr(F), _dptr(ap)))
        return F, ap

    def compute_forces_host(self):
        F = np.empty((self.V, 2), dtype=np.float64)
        ap = np.empty((self.N, 2), dtype=np.float64)
        _check(self.lib.avm_compute_forces_host(self._h, _hptr(F), _hptr(ap)))
        return F, ap

    def energy(self) -> float:
        e = ctypes.c_double(0.0)
        _check(self.lib.avm_energy(self._h, ctypes.byref(e)))
        return e.value

    def _set_cell_pair(self, fn, a0, b0) -> None:
        t = self.torch
        if a0 is None and b0 is None:
            _check(fn(self._h, None, None))
            return
        dev = []
        for a in (a0, b0):
            if isinstance(a, np.ndarray):
                a = t.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(self.device)
            assert a.shape == (self.N,) and a.dtype == t.float64 and a.is_contiguous()
            dev.append(a)
        _check(fn(self._h, _dptr(dev[0]), _dptr(dev[1])))
        t.cuda.synchronize(self.device)        # the inputs are copied by then

    def set_cell_targets(self, area0=None, perimeter0=None) -> None:
        """per-cell preferred area / perimeter (numpy or CUDA tensors, user order); None, None = uniform"""
        self._set_cell_pair(self.lib.avm_set_cell_targets, area0, perimeter0)

    def set_cell_moduli(self, KA=None, KP=None) -> None:
        """per-cell moduli K_A,i / K_P,i (numpy or CUDA tensors, user order); None, None = uniform"""
        self._set_cell_pair(self.lib.avm_set_cell_moduli, KA, KP)

    def msd_reset(self) -> None:
        _check(self.lib.avm_msd_reset(self._h))

    def observe(self) -> dict:
        o = AvmObservables()
        _check(self.lib.avm_observe(self._h, ctypes.byref(o)))
        return o.as_dict()

    # ---- SPV on a fixed triangulation (cell_xy: torch float64 [N,2] on the device, user order) ----
    def spv_geometry(self, cell_xy):
        t = self.torch
        vor = t.empty((self.V, 2), dtype=t.float64, device=self.device)
        ap = t.empty((self.N, 2), dtype=t.float64, device=self.device)
        _check(self.lib.avm_spv_geometry(self._h, cell_xy.data_ptr(), vor.data_ptr(), ap.data_ptr()))
        return vor, ap

    def spv_forces(self, cell_xy, sets: bool = True):
        t = self.torch
        F = t.empty((self.N, 2), dtype=t.float64, device=self.device)
        fs = t.empty((self.N, self.S, 2), dtype=t.float64, device=self.device) if sets else None
        _check(self.lib.avm_spv_forces(self._h, cell_xy.data_ptr(), F.data_ptr(), fs.data_ptr() if sets else None))
        return F, fs

    def spv_step(self, cell_xy, n: int = 1):
        """advances cell_xy in place; returns (failed tests after the last step, first failing step or -1, flags [N])"""
        t = self.torch
        out = (ctypes.c_int64 * 2)()
        flags = t.empty(self.N, dtype=t.int32, device=self.device)
        _check(self.lib.avm_spv_step(self._h, cell_xy.data_ptr(), n, out, flags.data_ptr()))
        return int(out[0]), int(out[1]), flags

    def spv_test_triangulation(self, cell_xy):
        t = self.torch
        out = (ctypes.c_int64 * 1)()
        flags = t.empty(self.N, dtype=t.int32, device=self.device)
        _check(self.lib.avm_spv_test_triangulation(self._h, cell_xy.data_ptr(), out, flags.data_ptr()))
        return int(out[0]), flags

    def step_observe(self, n: int = 1) -> dict:
        """n steps; the geometry pass of the last one also reduces the observables of its moved tiling"""
        o = AvmObservables()
        _check(self.lib.avm_step_observe(self._h, n, ctypes.byref(o)))
        return o.as_dict()

    def get_state(self, stats: bool = True) -> dict:
        t = self.torch
        pos = t.empty((self.V, 2), dtype=t.float64, device=self.device)
        cvn = t.empty(self.N, dtype=t.int32, device=self.device)
        cv = t.empty((self.N, self.S), dtype=t.int32, device=self.device)
        vn = t.empty((self.V, 3), dtype=t.int32, device=self.device)
        vc = t.empty((self.V, 3), dtype=t.int32, device=self.device)
        th = t.empty(self.N, dtype=t.float64, device=self.device)
        st = AvmStats()
        _check(self.lib.avm_get_state(self._h, _dptr(pos), _dptr(cvn), _dptr(cv), _dptr(vn), _dptr(vc), _dptr(th),
                                 ctypes.byref(st) if stats else None))
        return dict(pos=pos, cell_vertex_num=cvn, cell_vertices=cv, vertex_neighbors=vn,
                    vertex_cell_neighbors=vc, theta=th, stats=st.as_dict() if stats else None)

    def get_state_host(self, out: Optional[dict] = None) -> dict:
        if out is None:
            out = dict(pos=np.empty((self.V, 2), dtype=np.float64), cell_vertex_num=np.empty(self.N, dtype=np.int32),
                       cell_vertices=np.empty((self.N, self.S), dtype=np.int32),
                       vertex_neighbors=np.empty((self.V, 3), dtype=np.int32),
                       vertex_cell_neighbors=np.empty((self.V, 3), dtype=np.int32),
                       theta=np.empty(self.N, dtype=np.float64))
        st = AvmStats()
        _check(self.lib.avm_get_state_host(self._h, _hptr(out.get("pos")), _hptr(out.get("cell_vertex_num")),
                                      _hptr(out.get("cell_vertices")), _hptr(out.get("vertex_neighbors")),
                                      _hptr(out.get("vertex_cell_neighbors")), _hptr(out.get("theta")),
                                      ctypes.byref(st)))
        out["stats"] = st.as_dict()
        return out

    def stats(self) -> dict:
        st = AvmStats()
        _check(self.lib.avm_get_state(self._h, None, None, None, None, None, None, ctypes.byref(st)))
        return st.as_dict()

    # ---- test hooks ----------------------------------------------------------------------------
    def debug_t1(self):
        cap = 3 * self.N
        cand = np.empty((cap, 2), dtype=np.int32)
        win = np.empty((cap, 2), dtype=np.int32)
        nc, nw = ctypes.c_int64(0), ctypes.c_int64(0)
        _check(self.lib.avm_debug_t1(self._h, _hptr(cand), ctypes.byref(nc), _hptr(win), ctypes.byref(nw), cap))
        return cand[:nc.value].copy(), win[:nw.value].copy()

    def t1_pass(self) -> None:
        _check(self.lib.avm_t1_pass(self._h))

    def set_positions(self, pos) -> None:
        t = self.torch
        if isinstance(pos, np.ndarray):
            pos = t.from_numpy(np.ascontiguousarray(pos, dtype=np.float64)).to(self.device)
        assert pos.shape == (self.V, 2) and pos.dtype == t.float64 and pos.is_contiguous()
        _check(self.lib.avm_set_positions(self._h, _dptr(pos)))
        t.cuda.current_stream(self.device).synchronize()   # keep `pos` alive until consumed

    def resort(self) -> None:
        _check(self.lib.avm_resort(self._h))

    def philox_words(self, seed: int, step: int, cell0: int, n: int):
        t = self.torch
        out = t.empty((n, 4), dtype=t.int32, device=self.device)
        _check(self.lib.avm_philox_words(self._h, seed, step, cell0, n, _dptr(out)))
        return out.cpu().numpy().view(np.uint32)

    def hilbert_index(self, m: int, ix: np.ndarray, iy: np.ndarray) -> np.ndarray:
        t = self.torch
        dx = t.from_numpy(ix.astype(np.int64)).to(self.device).to(t.int32)
        dy = t.from_numpy(iy.astype(np.int64)).to(self.device).to(t.int32)
        out = t.empty(ix.shape[0], dtype=t.int32, device=self.device)
        _check(self.lib.avm_hilbert_index(self._h, m, ix.shape[0], _dptr(dx), _dptr(dy), _dptr(out)))
        return out.cpu().numpy().view(np.uint32)


def from_tiling(tiling, host: bool = False, precision: str = "f64", **params) -> AvmSim:
    p = make_params(tiling.N, tiling.S, **dict(params, Lx=tiling.Lx, Ly=tiling.Ly))
    return AvmSim(tiling, p, host=host, precision=precision)
