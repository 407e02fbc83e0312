"""The fused (two-launch) schedule under forced timing skew ("add a build knob that inserts a delay in
sweep() to widen the window").  Two test builds of the library hold back one side of the fused force/move launch
for tens of microseconds - the sweepers (so that every flip and every mover finishes before a sweeper reaches a
flagged vertex) or the flippers (so that the whole sweep is over before any flip is decided).  The schedule's
race-freedom argument says the result cannot depend on that order: both builds must
reproduce the three-launch schedule of the default library bit for bit."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1702_02939_b200 import workloads as w


@pytest.fixture(scope="module")
def B(tmp_path_factory):
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1702_02939_b200 import build, binding
    build.build()
    d = tmp_path_factory.mktemp("skew")
    for n in (1, 2, 3):
        binding.register_library(f"skew{n}", build.build_variant(str(d / f"libavm_skew{n}.so"), [f"AVM_TEST_SKEW={n}"]))
    return binding


def to_np(st):
    return {k: (v.cpu().numpy() if hasattr(v, "cpu") else v) for k, v in st.items()}


@pytest.mark.parametrize("skew", [1, 2])
def test_fused_schedule_does_not_depend_on_who_finishes_first(B, skew):
    t = w.config_tiling(2)                                   # 65 536 cells, ~60 flips per step: the one-warp-per-candidate mode
    p = dict(w.config_params(2), sort_every=11)
    ref = B.from_tiling(t, schedule="unfused", **p)
    ref.step(40)
    sr = to_np(ref.get_state())
    import torch
    g = B.from_tiling(t, schedule="fused", precision=f"skew{skew}", **p)
    g.step(7)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    g.step(33)
    e1.record()
    e1.synchronize()
    assert e0.elapsed_time(e1) > 33 * 0.04, "the skew knob had no effect: every fused launch must last at least 40 us"
    sg = to_np(g.get_state())
    assert sg["stats"]["kernel_launches"] < sr["stats"]["kernel_launches"] - 30       # it really ran two launches per step
    for key in ("pos", "theta", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "cell_vertex_num"):
        assert np.array_equal(sg[key], sr[key]), key
    for key in ("t1_short", "t1_candidates", "t1_flips", "t1_blocked", "error"):
        assert sg["stats"][key] == sr["stats"][key], key
    assert sr["stats"]["t1_flips"] > 1000


def test_image_counts_are_applied_once_when_movers_run_at_different_times(B):
    """ADVICE r2, under skew (see tests/test_gpu_parity.py::test_image_counts_are_applied_once_when_movers_overlap
    for the scenario: a rigidly translating tiling whose MSD is (n v0 dt)^2).  Movers of different candidates
    normally start within nanoseconds of each other, and a lost update can hide a second increment of a shared
    vertex's image count; the third test build starts every other mover 30 us late, so every shared vertex is
    moved at two clearly different times.  (Without the once-only claim this build gave 4108.2 instead of 4096.0.)"""
    t = w.voronoi_tiling(4096, 64.0, 4)
    t.theta[:] = 0.6
    p = dict(KA=0.0, KP=0.0, A0=1.0, P0=3.8, v0=128.0, Dr=0.0, mu=1.0, dt=0.1, l_c=0.008, seed=11)
    ref = B.from_tiling(t, schedule="unfused", **p)
    g = B.from_tiling(t, schedule="fused", precision="skew3", **p)
    ref.step(5)
    g.step(5)
    m = ref.observe()["msd"]
    assert g.observe()["msd"] == m and abs(m - 64.0 ** 2) < 1e-3
    st = g.stats()
    assert st["kernel_launches"] < ref.stats()["kernel_launches"] - 3
    assert 20 < st["t1_candidates"] <= 85 and st["t1_blocked"] > 0     # the one-warp-per-candidate mode, with shared cells
    assert np.array_equal(to_np(g.get_state())["pos"], to_np(ref.get_state())["pos"])
