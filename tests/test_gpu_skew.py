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
    for n in (1, 2):
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
