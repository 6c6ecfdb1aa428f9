"""GPU parity of the G-buffer extras (osog_render_gbuffer: depth map and instance-id map, reading A24)
against the oracle.  Both sides decide "which particle is on top" in float64; the GPU rounds the depth to float32.
Where two top surfaces cross, a 1e-12 difference between the two float64 evaluations may flip the owner of a pixel: such
pixels must be (very) rare and their depth must still agree (several owners are then correct: compare what is unique)."""
from dataclasses import replace

import numpy as np
import pytest

from workloads import make_config, make_scene

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def og():
    import torch
    assert torch.cuda.is_available()
    import paper_2606_21381_b200 as m
    m.lib()
    return m


@pytest.fixture(scope="module")
def o():
    from oracle import oracle
    return oracle


def with_heights(sc, seed, spread=6.0):
    """The BASELINE workloads put every centre at z = 0; give them seeded random heights."""
    rng = np.random.default_rng(seed)
    cols = dict(sc.cols)
    cols["cz"] = rng.uniform(-spread, spread, sc.N).astype(np.float32)
    return replace(sc, cols=cols)


def check(og, o, sc):
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P = og.Particles.from_scene(sc)
    opt = og.optics_from_scene(sc)
    tid, dep = ctx.render_gbuffer(P, opt)
    tid, dep = tid.cpu().numpy(), dep.cpu().numpy().astype(np.float64)
    assert ctx.status()[0] == 0
    ctx.close()
    rid, rdep = o.render_gbuffer(sc)
    tol = 1e-6 + 2e-7 * np.abs(rdep)
    assert np.all(np.abs(dep - rdep) <= tol), float(np.abs(dep - rdep).max())
    differ = tid != rid
    assert differ.mean() <= 1e-5, f"{int(differ.sum())} pixels with another owner"
    assert np.array_equal(tid < 0, rid < 0) or (differ & ((tid < 0) | (rid < 0))).sum() <= 2
    return tid, dep, rid, rdep


@pytest.mark.parametrize("k,n", [(1, None), (2, None), (3, None), (4, None), (5, None)])
def test_gbuffer_matches_oracle_on_the_baseline_workloads(og, o, k, n):
    """All five workloads at full size, with seeded random centre heights (config 5: 16 frames, ids relative to the frame)."""
    sc = with_heights(make_config(k, n_override=n), seed=40 + k)
    tid, dep, rid, rdep = check(og, o, sc)
    assert len(np.unique(tid)) > min(sc.N // sc.B, 40)      # many different owners
    if k == 5:
        assert tid.max() < sc.N // sc.B            # indices restart with every frame


def test_gbuffer_flat_heights_ties_and_no_cz(og, o):
    import torch
    # all centres at the same height (the workloads as they are) and a NULL cz give the same maps
    sc = make_config(2)
    tid, dep, _, _ = check(og, o, sc)
    ctx = og.Context(sc.H, sc.W, sc.N)
    cols = {k: v for k, v in sc.cols.items() if k != "cz"}
    P = og.Particles(cols, None)
    assert "cz" not in P.t
    t2, d2 = ctx.render_gbuffer(P, og.optics_from_scene(sc))
    assert np.array_equal(t2.cpu().numpy(), tid) and np.array_equal(d2.cpu().numpy().astype(np.float64), dep)
    # the hot path is untouched by the heights: same OPD bits with and without random cz
    a = ctx.render_opd(og.Particles.from_scene(sc), og.optics_from_scene(sc)).clone()
    b = ctx.render_opd(og.Particles.from_scene(with_heights(sc, 3)), og.optics_from_scene(sc))
    assert torch.equal(a, b)
    ctx.close()
    # an exact tie (two identical particles) goes to the smaller index; a particle with a NaN height is left out
    cols = dict(cx=[3.2, 3.2, 1.0], cy=[3.2, 3.2, 1.0], cz=[0.2, 0.2, float("nan")], d0=[1.5, 1.5, 0.5], d1=[1.5, 1.5, 0.5],
                d2=[1.5, 1.5, 0.5], n_p=[1.4] * 3)
    tid, dep, rid, _ = check(og, o, make_scene("tie", 64, 64, cols))
    assert set(np.unique(tid)) == {-1, 0}


def test_gbuffer_ragged_frame_prisms_with_vertical_faces(og, o):
    r = np.sqrt(0.5)
    cols = dict(cx=[3.213, 9.047, 6.131, 5.0], cy=[3.377, 4.021, 9.563, 5.2], cz=[0.5, -1.0, 2.0, 0.0], qw=[1.0, r, r, 0.9],
                qx=[0.0, r, 0.0, 0.1], qy=[0.0, 0.0, r, 0.3], qz=[0.0, 0.0, 0.0, 0.3], d0=[2.03, 1.57, 1.21, 3.0],
                d1=[3.3, 4.1, 2.9, 2.0], d2=[1.0, 0.8, 0.6, 1.2], n_p=[1.45, 1.40, 1.42, 1.4],
                kind=np.array([1, 1, 1, 0], np.uint8))
    check(og, o, make_scene("vertical_g", 100, 130, cols))
