"""Seeded synthetic workloads for the AVM hot path (input generation only).

This module builds the initial states the BASELINE.json configs describe ("Voronoi of N
uniform-random points (seed k)", PAPER.md:66 for the three topology lists) plus the small
hand-built tilings the tests use (regular hexagons).  It holds none of the method's arithmetic
and is the only code the CPU oracle's tests and the CUDA path's tests/bench have in common.

The heavy lifting is in ``tiling.cpp`` (periodic Voronoi by per-cell half-plane clipping),
compiled on demand with g++ into ``libavm_tiling.so`` next to this file.
"""
from __future__ import annotations

import ctypes
import dataclasses
import math
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tiling.cpp")
_LIB = os.path.join(_HERE, "libavm_tiling.so")
_lib: Optional[ctypes.CDLL] = None


def build(force: bool = False) -> str:
    """Compile tiling.cpp -> libavm_tiling.so (host code only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        i64, f64, u64, i32 = ctypes.c_int64, ctypes.c_double, ctypes.c_uint64, ctypes.c_int32
        p = ctypes.c_void_p
        lib.tiling_points.argtypes = [i64, f64, f64, u64, p]
        lib.tiling_thetas.argtypes = [i64, u64, p]
        lib.tiling_from_rows.argtypes = [i64, i64, i32, p, p, p, p]
        lib.tiling_voronoi.argtypes = [i64, f64, f64, p, i32, p, p, p, p, p, p]
        for f in (lib.tiling_points, lib.tiling_thetas, lib.tiling_from_rows, lib.tiling_voronoi):
            f.restype = ctypes.c_int
        _lib = lib
    return _lib


_ERR = {-1: "bad argument", -2: "open cell (box too small for neighbour search)",
        -3: "a cell has more than max_cell_vertices vertices",
        -4: "vertex triple not produced exactly three times (degenerate points)",
        -5: "V != 2N", -6: "clip overflow", -7: "rows are not a 3-coordinated tiling"}


def _ptr(a: np.ndarray) -> ctypes.c_void_p:
    return ctypes.c_void_p(a.ctypes.data)


@dataclasses.dataclass
class Tiling:
    """Initial AVM state in user (tag) order.  Arrays are C-contiguous numpy."""
    Lx: float
    Ly: float
    S: int                      # max_cell_vertices = row stride
    pos: np.ndarray             # float64 [V,2]
    cell_vertex_num: np.ndarray  # int32 [N]
    cell_vertices: np.ndarray   # int32 [N,S], CCW, unused = -1
    vertex_neighbors: np.ndarray       # int32 [V,3]
    vertex_cell_neighbors: np.ndarray  # int32 [V,3]
    theta: np.ndarray           # float64 [N]
    points: Optional[np.ndarray] = None  # generator points (Voronoi tilings only)

    @property
    def N(self) -> int:
        return int(self.cell_vertex_num.shape[0])

    @property
    def V(self) -> int:
        return int(self.pos.shape[0])

    def copy(self) -> "Tiling":
        return dataclasses.replace(
            self, pos=self.pos.copy(), cell_vertex_num=self.cell_vertex_num.copy(),
            cell_vertices=self.cell_vertices.copy(), vertex_neighbors=self.vertex_neighbors.copy(),
            vertex_cell_neighbors=self.vertex_cell_neighbors.copy(), theta=self.theta.copy())


def random_points(N: int, Lx: float, Ly: float, seed: int) -> np.ndarray:
    pts = np.empty((N, 2), dtype=np.float64)
    rc = _load().tiling_points(N, Lx, Ly, seed, _ptr(pts))
    if rc:
        raise ValueError(_ERR.get(rc, str(rc)))
    return pts


def random_thetas(N: int, seed: int) -> np.ndarray:
    th = np.empty(N, dtype=np.float64)
    rc = _load().tiling_thetas(N, seed, _ptr(th))
    if rc:
        raise ValueError(_ERR.get(rc, str(rc)))
    return th


def lists_from_rows(cvn: np.ndarray, cv: np.ndarray, V: int):
    """vertexNeighbors / vertexCellNeighbors (slot convention of DESIGN.md) from CCW rows."""
    N, S = cv.shape
    cvn = np.ascontiguousarray(cvn, dtype=np.int32)
    cv = np.ascontiguousarray(cv, dtype=np.int32)
    vn = np.empty((V, 3), dtype=np.int32)
    vc = np.empty((V, 3), dtype=np.int32)
    rc = _load().tiling_from_rows(N, V, S, _ptr(cvn), _ptr(cv), _ptr(vn), _ptr(vc))
    if rc:
        raise ValueError(_ERR.get(rc, str(rc)))
    return vn, vc


def voronoi_tiling(N: int, L: float, seed: int, S: int = 16, Ly: Optional[float] = None,
                   points: Optional[np.ndarray] = None) -> Tiling:
    """Periodic Voronoi tiling of N seeded uniform points in [0,L)x[0,Ly)."""
    Lx = float(L)
    Ly = float(L if Ly is None else Ly)
    pts = random_points(N, Lx, Ly, seed) if points is None else np.ascontiguousarray(points, dtype=np.float64)
    V = 2 * N
    pos = np.empty((V, 2), dtype=np.float64)
    cvn = np.empty(N, dtype=np.int32)
    cv = np.empty((N, S), dtype=np.int32)
    vn = np.empty((V, 3), dtype=np.int32)
    vc = np.empty((V, 3), dtype=np.int32)
    info = np.zeros(2, dtype=np.int64)
    rc = _load().tiling_voronoi(N, Lx, Ly, _ptr(pts), S, _ptr(pos), _ptr(cvn), _ptr(cv), _ptr(vn),
                                _ptr(vc), _ptr(info))
    if rc:
        raise ValueError(f"tiling_voronoi: {_ERR.get(rc, rc)} (max n seen {int(info[0])})")
    return Tiling(Lx, Ly, S, pos, cvn, cv, vn, vc, random_thetas(N, seed), points=pts)


def hex_tiling(nx: int, ny: int, a: float = 1.0, S: int = 16, theta: Optional[np.ndarray] = None) -> Tiling:
    """Regular pointy-top hexagons of side a on a torus: ny (even) rows of nx cells.

    Lx = nx*sqrt(3)*a, Ly = ny*1.5*a tiles the torus exactly (reading R13: a regular
    hexagonal tiling is periodic in a rectangle, not in a square).  nx, ny >= 4 keeps every cell
    narrower than half the box so that minimum-image unwrapping is valid.
    """
    if ny % 2 or nx < 3 or ny < 4:
        raise ValueError("need even ny >= 4 and nx >= 3")
    s3 = math.sqrt(3.0)
    Lx, Ly = nx * s3 * a, ny * 1.5 * a
    N, V = nx * ny, 2 * nx * ny
    # vertices live on a lattice with spacing (sqrt(3)/2*a, a/2): integer key (kx, ky)
    key_to_id = {}
    pos = []
    cv = np.full((N, S), -1, dtype=np.int32)
    cvn = np.full(N, 6, dtype=np.int32)
    # CCW corner offsets in lattice units starting at angle 30 degrees
    offs = [(1, 1), (0, 2), (-1, 1), (-1, -1), (0, -2), (1, -1)]
    for iy in range(ny):
        for ix in range(nx):
            c = iy * nx + ix
            ckx, cky = 2 * ix + (iy % 2), 3 * iy   # centre in lattice units
            for m, (ox, oy) in enumerate(offs):
                k = ((ckx + ox) % (2 * nx), (cky + oy) % (3 * ny))
                if k not in key_to_id:
                    key_to_id[k] = len(pos)
                    pos.append((k[0] * 0.5 * s3 * a, k[1] * 0.5 * a))
                cv[c, m] = key_to_id[k]
    assert len(pos) == V
    pos = np.asarray(pos, dtype=np.float64)
    vn, vc = lists_from_rows(cvn, cv, V)
    th = np.zeros(N, dtype=np.float64) if theta is None else np.asarray(theta, dtype=np.float64).copy()
    return Tiling(Lx, Ly, S, pos, cvn, cv, vn, vc, th)


# ---------------------------------------------------------------------------------------------
# The five BASELINE.json configs.  mu = K_A = K_P = A0 = 1 everywhere;
# P0 = p0*sqrt(A0) = p0.  "steps" is the config's nominal run length.
# ---------------------------------------------------------------------------------------------
CONFIGS = [
    dict(name="cfg0", N=64, L=8.0, points_seed=1, p0=3.8, v0=0.05, Dr=1.0, dt=0.01, l_c=0.04,
         seed=7, steps=100, sort_every=0, sort_at_create=False),
    dict(name="cfg1", N=4096, L=64.0, points_seed=2, p0=3.8, v0=0.1, Dr=1.0, dt=0.01, l_c=0.04,
         seed=7, steps=10000, sort_every=0, sort_at_create=False),
    dict(name="cfg2", N=65536, L=256.0, points_seed=3, p0=3.9, v0=0.5, Dr=0.5, dt=0.01, l_c=0.04,
         seed=7, steps=10000, sort_every=0, sort_at_create=True),
    dict(name="cfg3", N=1048576, L=1024.0, points_seed=4, p0=3.6, v0=0.01, Dr=1.0, dt=0.01, l_c=0.04,
         seed=7, steps=1000, sort_every=0, sort_at_create=True),
    dict(name="cfg4", N=4194304, L=2048.0, points_seed=5, p0=4.0, v0=1.0, Dr=0.1, dt=0.005, l_c=0.06,
         seed=7, steps=500, sort_every=100, sort_at_create=True),
]


def config_tiling(k: int, S: int = 16) -> Tiling:
    cfg = CONFIGS[k]
    return voronoi_tiling(cfg["N"], cfg["L"], cfg["points_seed"], S=S)


def config_params(k: int) -> dict:
    """Model parameters of config k as plain numbers (the caller builds its own param struct)."""
    cfg = CONFIGS[k]
    return dict(Lx=cfg["L"], Ly=cfg["L"], KA=1.0, KP=1.0, A0=1.0, P0=cfg["p0"], v0=cfg["v0"],
                Dr=cfg["Dr"], mu=1.0, dt=cfg["dt"], l_c=cfg["l_c"], seed=cfg["seed"],
                sort_every=cfg["sort_every"], sort_at_create=cfg["sort_at_create"])
