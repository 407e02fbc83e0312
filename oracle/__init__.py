"""CPU oracle for the AVM hot path — TEST INFRASTRUCTURE, not product code.

ctypes wrapper around ``avm_oracle.cpp`` (single-threaded C++17, fp64, built with
``-O2 -ffp-contract=off``).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports nothing from
``paper_1702_02939_b200`` and shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "avm_oracle.cpp")
_LIB = os.path.join(_HERE, "libavm_oracle.so")
_lib: Optional[ctypes.CDLL] = None


class OracleParams(ctypes.Structure):
    _fields_ = [("n_cells", ctypes.c_int32), ("n_vertices", ctypes.c_int32),
                ("max_cell_vertices", ctypes.c_int32), ("t1_max_passes", ctypes.c_int32),
                ("Lx", ctypes.c_double), ("Ly", ctypes.c_double),
                ("KA", ctypes.c_double), ("KP", ctypes.c_double), ("A0", ctypes.c_double), ("P0", ctypes.c_double),
                ("v0", ctypes.c_double), ("Dr", ctypes.c_double), ("mu", ctypes.c_double),
                ("dt", ctypes.c_double), ("l_c", ctypes.c_double),
                ("seed", ctypes.c_uint64), ("step0", ctypes.c_uint64)]


class OracleStats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int64) for n in
                ("step", "t1_short", "t1_candidates", "t1_flips", "t1_blocked", "overflow_rejects", "error")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


def build(force: bool = False) -> str:
    """Compile the oracle (host C++ only; building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC",
                               "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        p, i64, u64 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_uint64
        lib.oracle_create.restype = p
        lib.oracle_create.argtypes = [ctypes.POINTER(OracleParams), p, p, p, p, p, p]
        lib.oracle_destroy.argtypes = [p]
        lib.oracle_destroy.restype = None
        lib.oracle_geometry.argtypes = [p, p]
        lib.oracle_energy.argtypes = [p]
        lib.oracle_energy.restype = ctypes.c_double
        lib.oracle_compute_forces.argtypes = [p, p, p]
        lib.oracle_step.argtypes = [p, i64]
        lib.oracle_step_move_and_rotate.argtypes = [p]
        lib.oracle_step_topology_and_advance.argtypes = [p]
        lib.oracle_t1_pass.argtypes = [p]
        lib.oracle_set_cell_targets.argtypes = [p, p, p]
        lib.oracle_set_cell_moduli.argtypes = [p, p, p]
        lib.oracle_msd.argtypes = [p]
        lib.oracle_msd.restype = ctypes.c_double
        lib.oracle_msd_reset.argtypes = [p]
        lib.oracle_debug_t1.argtypes = [p, p, p, p, p, i64]
        lib.oracle_get_state.argtypes = [p, p, p, p, p, p, p, ctypes.POINTER(OracleStats)]
        lib.oracle_set_positions.argtypes = [p, p]
        lib.oracle_philox4x32_10.argtypes = [p, p, p]
        lib.oracle_philox4x32_10.restype = None
        lib.oracle_philox_words.argtypes = [u64, u64, u64, i64, p]
        lib.oracle_philox_words.restype = None
        lib.oracle_director_noise.argtypes = [u64, u64, u64, i64, p]
        lib.oracle_director_noise.restype = None
        _lib = lib
    return _lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.empty(4, dtype=np.uint32)
    _load().oracle_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
    return out


def philox_words(seed: int, step: int, cell0: int, n: int) -> np.ndarray:
    """Raw Philox output words for (seed, step, cell0..cell0+n-1), shape [n,4]."""
    out = np.empty((n, 4), dtype=np.uint32)
    _load().oracle_philox_words(seed, step, cell0, n, _ptr(out))
    return out


def director_noise(seed: int, step: int, cell0: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _load().oracle_director_noise(seed, step, cell0, n, _ptr(out))
    return out


class OracleSim:
    """One AVM system advanced on the CPU.  All arrays are numpy, user order."""

    def __init__(self, pos, cell_vertex_num, cell_vertices, vertex_neighbors, vertex_cell_neighbors, theta, *,
                 Lx, Ly, KA=1.0, KP=1.0, A0=1.0, P0=3.8, v0=0.0, Dr=0.0, mu=1.0, dt=0.01, l_c=0.0,
                 seed=0, step0=0, t1_max_passes=1, **_ignored):
        lib = _load()
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        cvn = np.ascontiguousarray(cell_vertex_num, dtype=np.int32)
        cv = np.ascontiguousarray(cell_vertices, dtype=np.int32)
        vn = np.ascontiguousarray(vertex_neighbors, dtype=np.int32)
        vc = np.ascontiguousarray(vertex_cell_neighbors, dtype=np.int32)
        th = np.ascontiguousarray(theta, dtype=np.float64)
        self.N, self.S = cv.shape
        self.V = pos.shape[0]
        self.params = OracleParams(self.N, self.V, self.S, int(t1_max_passes), Lx, Ly, KA, KP, A0, P0, v0, Dr, mu, dt, l_c, seed, step0)
        self._h = lib.oracle_create(ctypes.byref(self.params), _ptr(pos), _ptr(cvn), _ptr(cv), _ptr(vn), _ptr(vc), _ptr(th))
        if not self._h:
            raise ValueError("oracle_create rejected the input")

    def __del__(self):
        if getattr(self, "_h", None):
            _load().oracle_destroy(self._h)
            self._h = None

    def geometry(self) -> np.ndarray:
        ap = np.empty((self.N, 2), dtype=np.float64)
        _load().oracle_geometry(self._h, _ptr(ap))
        return ap

    def energy(self) -> float:
        return float(_load().oracle_energy(self._h))

    def observables(self) -> dict:
        """NEXT-2: the definitions, written out with numpy on the oracle's own geometry: energy of
        Eq. 1, totals, mean shape index <P / sqrt(A)> over cells with A > 0, area
        extremes and (population) variance, number of cells with non-positive signed area."""
        ap = self.geometry()
        A, P = ap[:, 0], ap[:, 1]
        pos = A > 0
        return {"energy": self.energy(), "msd": self.msd(), "sum_area": float(A.sum()), "sum_perimeter": float(P.sum()),
                "mean_shape_index": float((P[pos] / np.sqrt(A[pos])).mean()) if pos.any() else 0.0,
                "area_min": float(A.min()), "area_max": float(A.max()),
                "area_variance": float((A * A).mean() - A.mean() ** 2),
                "n_nonpositive_area": int((~pos).sum())}

    def compute_forces(self):
        F = np.empty((self.V, 2), dtype=np.float64)
        ap = np.empty((self.N, 2), dtype=np.float64)
        _load().oracle_compute_forces(self._h, _ptr(F), _ptr(ap))
        return F, ap

    def step(self, n: int = 1) -> None:
        _load().oracle_step(self._h, n)

    def step_move_and_rotate(self) -> None:
        """first half of one step: geometry, forces, move, director update"""
        _load().oracle_step_move_and_rotate(self._h)

    def step_topology_and_advance(self) -> None:
        """second half: the T1 pass(es) on the moved positions and the step counter"""
        _load().oracle_step_topology_and_advance(self._h)

    def set_cell_targets(self, A0=None, P0=None) -> None:
        """per-cell preferred area / perimeter of Eq. 1 (user order); None, None = uniform again"""
        a = None if A0 is None else np.ascontiguousarray(A0, dtype=np.float64)
        b = None if P0 is None else np.ascontiguousarray(P0, dtype=np.float64)
        if _load().oracle_set_cell_targets(self._h, _ptr(a), _ptr(b)) != 0:
            raise ValueError("oracle_set_cell_targets: give both arrays or neither")

    def set_cell_moduli(self, KA=None, KP=None) -> None:
        """per-cell moduli K_{A,i}, K_{P,i} of Eq. 1 (user order); None, None = uniform again"""
        a = None if KA is None else np.ascontiguousarray(KA, dtype=np.float64)
        b = None if KP is None else np.ascontiguousarray(KP, dtype=np.float64)
        if _load().oracle_set_cell_moduli(self._h, _ptr(a), _ptr(b)) != 0:
            raise ValueError("oracle_set_cell_moduli: give both arrays or neither")

    def msd(self) -> float:
        """mean-square displacement of the vertices since creation / the latest msd_reset (unwrapped)"""
        return float(_load().oracle_msd(self._h))

    def msd_reset(self) -> None:
        _load().oracle_msd_reset(self._h)

    def t1_pass(self) -> None:
        _load().oracle_t1_pass(self._h)

    def debug_t1(self):
        cap = 3 * self.N
        cand = np.empty((cap, 2), dtype=np.int32)
        win = np.empty((cap, 2), dtype=np.int32)
        nc, nw = ctypes.c_int64(0), ctypes.c_int64(0)
        _load().oracle_debug_t1(self._h, _ptr(cand), ctypes.byref(nc), _ptr(win), ctypes.byref(nw), cap)
        return cand[:nc.value].copy(), win[:nw.value].copy()

    def set_positions(self, pos) -> None:
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        assert pos.shape == (self.V, 2)
        _load().oracle_set_positions(self._h, _ptr(pos))

    def get_state(self) -> dict:
        pos = np.empty((self.V, 2), dtype=np.float64)
        cvn = np.empty(self.N, dtype=np.int32)
        cv = np.empty((self.N, self.S), dtype=np.int32)
        vn = np.empty((self.V, 3), dtype=np.int32)
        vc = np.empty((self.V, 3), dtype=np.int32)
        th = np.empty(self.N, dtype=np.float64)
        st = OracleStats()
        _load().oracle_get_state(self._h, _ptr(pos), _ptr(cvn), _ptr(cv), _ptr(vn), _ptr(vc), _ptr(th), ctypes.byref(st))
        return dict(pos=pos, cell_vertex_num=cvn, cell_vertices=cv, vertex_neighbors=vn,
                    vertex_cell_neighbors=vc, theta=th, stats=st.as_dict())


def from_tiling(t, **params) -> OracleSim:
    """Convenience: build an OracleSim from any object with the Tiling attribute names."""
    return OracleSim(t.pos, t.cell_vertex_num, t.cell_vertices, t.vertex_neighbors, t.vertex_cell_neighbors,
                     t.theta, Lx=t.Lx, Ly=t.Ly, **{k: v for k, v in params.items() if k not in ("Lx", "Ly")})
