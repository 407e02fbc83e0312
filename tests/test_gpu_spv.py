"""GPU parity of the SPV pieces on a fixed triangulation (avm_spv_*; csrc/avm_spv.cu) against oracle/spv.py,
element by element on the same seeded inputs (App. A.2).  Run with `pytest -m gpu`."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import spv
from paper_1702_02939_b200 import workloads as w
from tests import helpers as h


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1702_02939_b200 import build
    build.build()
    from paper_1702_02939_b200 import binding
    return binding


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


CASES = [(64, 8.0, 1, False), (4096, 64.0, 2, True), (20000, 141.0, 9, True)]   # several CTAs and a ragged tail


@pytest.mark.parametrize("N,L,seed,sort", CASES)
def test_spv_geometry_and_forces_match_the_oracle(B, N, L, seed, sort):
    t = w.voronoi_tiling(N, L, seed)
    p = dict(KA=1.0, KP=1.0, A0=1.0, P0=3.8, v0=0.1, Dr=1.0, mu=1.0, dt=1e-4, l_c=0.0, seed=7)
    g = B.from_tiling(t, sort_at_create=sort, **p)
    o = spv.SpvOracle(t, t.points, **p)
    r = dev(t.points)
    vor, ap = g.spv_geometry(r)
    ho, apo = o.geometry()
    d = h.min_image(vor.cpu().numpy() - ho, L)
    assert np.abs(d).max() <= 1e-10 * L
    assert np.abs(ap.cpu().numpy() - apo).max() <= 1e-10 * np.abs(apo).max()
    # the Voronoi vertices are now the simulation's vertex positions
    assert np.abs(h.min_image(g.get_state()["pos"].cpu().numpy() - ho, L)).max() <= 1e-10 * L
    # ... replaced, not moved: the mean-square displacement restarts from them, whatever was counted before
    if N == 64:
        g2 = B.from_tiling(t, sort_at_create=sort, **dict(p, v0=3.0, dt=0.02))
        g2.step(200)
        assert g2.observe()["msd"] > 1.0
        g2.spv_geometry(r)
        assert g2.observe()["msd"] == 0.0
    F, fs = g.spv_forces(r)
    Fo = o.forces()
    rms = np.sqrt((Fo ** 2).sum(1).mean())
    err = np.linalg.norm(F.cpu().numpy() - Fo, axis=1) / np.maximum(np.linalg.norm(Fo, axis=1), rms)
    assert err.max() <= 1e-9, err.max()       # the circumcentre Jacobian of a thin triangle amplifies rounding: 1e-9, not 1e-10
    if N <= 4096:
        fso = o.force_sets()
        scale = np.abs(fso).max()
        assert np.abs(fs.cpu().numpy() - fso).max() <= 1e-9 * scale
        assert np.abs(fs.cpu().numpy().sum(axis=1) - F.cpu().numpy()).max() <= 1e-12 * scale


@pytest.mark.parametrize("mu,KA,KP", [(1.0, 1.0, 1.0), (0.37, 1.7, 0.6)])
def test_spv_steps_match_the_oracle(B, mu, KA, KP):
    """ten steps of Eq. 3 on the fixed triangulation: positions, directors (Philox keyed on the same seed, step,
    cell), the simulation's saved Voronoi vertices, and the circumcircle verdict after every call; also with a
    mobility and moduli other than 1 (the oracle's mu is pinned by tests/test_oracle_spv.py)"""
    t = w.voronoi_tiling(1024, 32.0, 3)
    p = dict(KA=KA, KP=KP, A0=1.0, P0=3.8, v0=0.2, Dr=1.0, mu=mu, dt=2e-5, l_c=0.0, seed=11)
    g = B.from_tiling(t, sort_at_create=True, **p)
    o = spv.SpvOracle(t, t.points, **p)
    r = dev(t.points)
    for rep in range(5):
        nf, first, flags = g.spv_step(r, 2)
        o.step(2)
        d = h.min_image(r.cpu().numpy() - o.r, 32.0)
        assert np.abs(d).max() <= 1e-9, (rep, np.abs(d).max())
        st = g.get_state()
        assert np.abs(st["theta"].cpu().numpy() - o.theta).max() <= 1e-8
        assert st["stats"]["step"] == o.step_count
        assert np.abs(h.min_image(st["pos"].cpu().numpy() - o.circumcentres(), 32.0)).max() <= 1e-8
        failed, margin, opp = o.test_triangulation()
        sure = np.abs(margin) > 1e-7
        assert (failed & sure).sum() <= nf <= (failed | ~sure).sum()


def test_spv_circumcircle_test_matches_the_oracle(B):
    t = w.voronoi_tiling(4096, 64.0, 5)
    g = B.from_tiling(t, **dict(w.config_params(1), sort_at_create=True))
    o = spv.SpvOracle(t, t.points)
    nf, flags = g.spv_test_triangulation(dev(t.points))
    assert nf == 0 and int(flags.sum()) == 0              # a Voronoi start is Delaunay
    rng = np.random.default_rng(2)
    for amp in (1e-4, 1e-2, 0.1, 0.3):
        r = np.mod(t.points + amp * rng.standard_normal(t.points.shape), 64.0)
        nf, flags = g.spv_test_triangulation(dev(r))
        failed, margin, opp = o.test_triangulation(r)
        assert np.abs(margin).min() > 1e-9                # no test sits on the circle: the comparison is exact
        assert nf == int(failed.sum())
        want = np.zeros(t.N, dtype=np.int32)
        vbad, kbad = np.nonzero(failed)
        want[t.vertex_cell_neighbors[vbad].ravel()] = 1
        want[opp[vbad, kbad]] = 1
        assert np.array_equal(flags.cpu().numpy(), want)
    assert nf > 100
