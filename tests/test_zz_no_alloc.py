"""avm_forces_static: the entry point for callers that may not allocate device memory.

Who they are: code that runs inside another program's memory plan (a plugin or callback handed fixed
device buffers by a host application that forbids cudaMalloc), loops with a latency budget that cannot
afford the allocator's locks and the device-wide synchronisation a cudaMalloc / cudaFree implies, and
processes whose device memory another pool has reserved completely.  They cannot supply avm_create's
workspace either, so this entry point needs neither a simulation object nor a workspace: its only scratch,
the per-cell (area, perimeter) pairs handed from the geometry kernel to the force kernel, sits in a 1 MiB
array compiled into the library.

The GPU test checks it against the ordinary path (avm_create + avm_compute_forces) with the tolerance of the
force parity tests (1e-10 relative, tests/test_gpu_parity.py), on calls made back to back: the array is
shared by all calls and keeps what the previous one wrote, so the second call, on a smaller tiling, runs
with the first one's leftovers behind its own entries, and a third one repeats the first.

This file is named to be collected last: `pytest -x` stops at the first failure, and nothing should hide
behind this one.  It passes alone in a fresh process (its first CUDA call then is the library's own address
look-up) and after the other GPU tests."""
import ctypes

import numpy as np
import pytest

from paper_1702_02939_b200 import workloads as w


def _binding():
    from paper_1702_02939_b200 import build
    build.build()
    from paper_1702_02939_b200 import binding
    return binding


def _assert_close(F, Fo, ap, apo):
    # the bar of tests/test_gpu_parity.py::assert_forces_close
    sa = np.maximum(np.abs(apo[:, 0]), np.abs(apo[:, 0]).mean())
    assert (np.abs(ap[:, 0] - apo[:, 0]) <= 1e-10 * sa).all()
    assert (np.abs(ap[:, 1] - apo[:, 1]) <= 1e-10 * np.abs(apo[:, 1])).all()
    rms = np.sqrt((Fo ** 2).sum(axis=1).mean())
    nf = np.linalg.norm(Fo, axis=1)
    err = np.linalg.norm(F - Fo, axis=1)
    assert (err <= 1e-10 * np.maximum(nf, rms)).all(), (err / np.maximum(nf, rms)).max()


def test_sizes_beyond_the_static_array_are_refused():
    """More cells than the built-in array holds: a clear error before any CUDA call (runs without a GPU)."""
    B = _binding()
    fake = ctypes.c_void_p(256)   # never dereferenced: the size check comes first
    for lib in (B.lib, ctypes.CDLL(B.LIB_MIXED_PATH)):
        big = B.make_params(B.AVM_FORCES_STATIC_MAX_CELLS + 1, 16, Lx=300.0, Ly=300.0)
        rc = lib.avm_forces_static(ctypes.byref(big), fake, fake, fake, fake, fake, fake, fake, None)
        assert rc == -6
        bad = B.make_params(64, 16, Lx=8.0, Ly=8.0)
        assert lib.avm_forces_static(ctypes.byref(bad), fake, fake, fake, fake, fake, None, None, None) == -1   # no output
        assert lib.avm_forces_static(ctypes.byref(bad), None, fake, fake, fake, fake, fake, fake, None) == -1   # NULL input
    assert b"AVM_FORCES_STATIC_MAX_CELLS" in B.lib.avm_strerror(-6)
    header = open(__file__.replace("tests/test_zz_no_alloc.py", "include/avm.h")).read()
    assert f"#define AVM_FORCES_STATIC_MAX_CELLS {B.AVM_FORCES_STATIC_MAX_CELLS}\n" in header


@pytest.mark.gpu
def test_static_scratch_forces_equal_the_workspace_path_on_consecutive_calls():
    import torch
    assert torch.cuda.is_available(), "this test needs the B200"
    B = _binding()
    dev = torch.device("cuda", 0)

    def device_inputs(t):
        as_dev = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).to(dev)
        return (as_dev(t.pos, np.float64), as_dev(t.cell_vertex_num, np.int32), as_dev(t.cell_vertices, np.int32),
                as_dev(t.vertex_neighbors, np.int32), as_dev(t.vertex_cell_neighbors, np.int32))

    def static_call(t, par):
        p = B.make_params(t.N, t.S, **dict(par, Lx=t.Lx, Ly=t.Ly))
        F = torch.full((2 * t.N, 2), float("nan"), dtype=torch.float64, device=dev)
        ap = torch.full((t.N, 2), float("nan"), dtype=torch.float64, device=dev)
        B.forces_static(p, *device_inputs(t), F, ap)
        torch.cuda.synchronize(dev)
        return F.cpu().numpy(), ap.cpu().numpy()

    def workspace_call(t, par):
        sim = B.from_tiling(t, **par)
        F, ap = sim.compute_forces()
        out = F.cpu().numpy(), ap.cpu().numpy()
        sim.close()
        return out

    # the larger tiling first, so that the smaller one finds stale entries behind its own
    t1, par1 = w.config_tiling(1), dict(w.config_params(1), KA=1.7, KP=0.6, A0=1.2)
    t0, par0 = w.config_tiling(0), w.config_params(0)
    first = static_call(t1, par1)
    second = static_call(t0, par0)
    third = static_call(t1, par1)
    ref1, ref0 = workspace_call(t1, par1), workspace_call(t0, par0)
    _assert_close(first[0], ref1[0], first[1], ref1[1])
    _assert_close(second[0], ref0[0], second[1], ref0[1])
    assert np.array_equal(third[0], first[0]) and np.array_equal(third[1], first[1])
    assert np.abs(ref1[0]).max() > 1e-3   # the comparison is not between zeros
    # forces only / geometry only
    p = B.make_params(t0.N, t0.S, **dict(par0, Lx=t0.Lx, Ly=t0.Ly))
    F = torch.empty((2 * t0.N, 2), dtype=torch.float64, device=dev)
    B.forces_static(p, *device_inputs(t0), F, None)
    ap = torch.empty((t0.N, 2), dtype=torch.float64, device=dev)
    B.forces_static(p, *device_inputs(t0), None, ap)
    torch.cuda.synchronize(dev)
    assert np.array_equal(F.cpu().numpy(), second[0]) and np.array_equal(ap.cpu().numpy(), second[1])
