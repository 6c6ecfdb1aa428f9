"""Pins for the oracle's binning restatement (B1-B4).

Expected values come from brute force: the bounding box is compared with the set of pixels the thickness
oracle actually covers (conservative, and tight to a pixel), the half-extents with a dense sampling of the
body's surface, and the tile lists with a dumb loop over every (tile, particle) pair.
"""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from oracle import oracle as o
from workloads import make_config, make_scene, subset


def _scene(n=60, H=160, W=144, seed=21):
    rng = np.random.default_rng(seed)
    q = rng.standard_normal((n, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    kind = (rng.uniform(size=n) < 0.5).astype(np.uint8)
    s = rng.uniform(0.5, 2.5, n)
    d = np.where(kind[:, None] == 1, np.stack([s, s * rng.uniform(1, 3, n), 0.5 * s], 1), rng.uniform(0.3, 3.0, (n, 3)))
    cols = dict(cx=rng.uniform(-1.0, W * 0.1 + 1.0, n), cy=rng.uniform(-1.0, H * 0.1 + 1.0, n),
                qw=q[:, 0], qx=q[:, 1], qy=q[:, 2], qz=q[:, 3], d0=d[:, 0], d1=d[:, 1], d2=d[:, 2],
                n_p=rng.uniform(1.36, 1.5, n), kind=kind)
    return make_scene("bins", H, W, cols)


def test_B1_half_extents_against_sampled_surface():
    sc = _scene(n=30)
    hx, hy = o.half_extents(sc.cols)
    rng = np.random.default_rng(1)
    u = rng.standard_normal((200000, 3)); u /= np.linalg.norm(u, axis=1, keepdims=True)
    for n in range(sc.N):
        q = np.array([sc.qw[n], sc.qx[n], sc.qy[n], sc.qz[n]], dtype=np.float64)
        R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()
        d = np.array([sc.d0[n], sc.d1[n], sc.d2[n]], dtype=np.float64)
        if sc.kind[n] == 0:
            P = (u * d) @ R.T                                    # points on the ellipsoid surface
            assert np.abs(P[:, 0]).max() <= hx[n] * (1 + 1e-6)
            assert np.abs(P[:, 0]).max() >= hx[n] * (1 - 2e-3)  # and the bound is attained
            assert np.abs(P[:, 1]).max() >= hy[n] * (1 - 2e-3)
        else:
            s, L, hc = d
            V = np.array([(a * s / 2, b * s / 2, c * L / 2) for a in (1, -1) for b in (1, -1) for c in (1, -1)]
                         + [(0, 0, L / 2 + hc), (0, 0, -L / 2 - hc)])
            lam = rng.dirichlet(np.ones(10), size=20000)          # the body is the hull of its vertices
            P = (lam @ V) @ R.T
            assert np.abs(P[:, 0]).max() <= hx[n] * (1 + 1e-6)
            assert np.abs((V @ R.T)[:, 0]).max() == pytest.approx(hx[n], rel=1e-6)
            assert np.abs((V @ R.T)[:, 1]).max() == pytest.approx(hy[n], rel=1e-6)


def test_B2_bbox_is_conservative_and_tight_against_covered_pixels():
    sc = _scene()
    H, W = sc.H, sc.W
    j0, j1, i0, i1, listed = o.bboxes(sc.cols, H, W, sc.pitch_um)
    n_tight = 0
    n_inside = 0
    for n in range(sc.N):
        one = o.render_opd(subset(sc, [n]), "full")[0]
        ii, jj = np.nonzero(one)
        if ii.size == 0:
            continue
        assert listed[n]
        assert j0[n] <= jj.min() and jj.max() <= j1[n] and i0[n] <= ii.min() and ii.max() <= i1[n]
        # tight to one pixel on every side, for bodies whose box the frame does not clip (a clipped body's
        # widest section may lie off-frame, so its visible pixels can be narrower than the box)
        if j0[n] == 0 or i0[n] == 0 or j1[n] == W - 1 or i1[n] == H - 1:
            continue
        n_inside += 1
        assert jj.min() - j0[n] <= 1 and j1[n] - jj.max() <= 1 and ii.min() - i0[n] <= 1 and i1[n] - ii.max() <= 1
        n_tight += int(jj.min() == j0[n]) + int(jj.max() == j1[n]) + int(ii.min() == i0[n]) + int(ii.max() == i1[n])
    assert n_inside >= 20 and n_tight > 2.5 * n_inside            # most edges are exact
    # clamping and emptiness
    assert (j0[listed] >= 0).all() and (j1[listed] <= W - 1).all() and (i0[listed] >= 0).all() and (i1[listed] <= H - 1).all()


def test_B2_edge_cases():
    H = W = 64
    cols = dict(cx=[-3.0, 3.2, 3.2, 6.399, 3.2499999], cy=[3.2, -3.0, 3.2, 3.2, 3.2500001],
                d0=[1.0, 1.0, 0.01, 1.0, 0.004], d1=[1.0, 1.0, 0.01, 1.0, 0.004], d2=[1.0, 1.0, 0.01, 1.0, 0.004],
                n_p=[1.4] * 5)
    sc = make_scene("edge", H, W, cols)
    j0, j1, i0, i1, listed = o.bboxes(sc.cols, H, W, 0.1)
    assert list(listed[:2]) == [False, False]                     # fully off-frame
    # a 10 nm sphere centred on a pixel corner (3.2 um = corner between pixels 31 and 32) covers no centre
    assert not listed[2]
    assert listed[3] and j1[3] == W - 1 and j0[3] == 54           # clamped at the right edge (6.399 - 1)/0.1 - 0.5 = 53.49
    # a 4 nm sphere within 1e-5 px of a pixel centre (3.25 um = centre of pixel 32): listed, exactly that pixel
    assert listed[4] and (j0[4], j1[4], i0[4], i1[4]) == (32, 32, 32, 32)


@pytest.mark.parametrize("T", [8, 16, 32])
def test_B3_B4_lists_against_dumb_double_loop(T):
    sc = _scene(n=80, H=100, W=90, seed=33)          # H, W not multiples of T: ragged last tiles
    count, offset, lst = o.binning(sc, T)
    j0, j1, i0, i1, listed = o.bboxes(sc.cols, sc.H, sc.W, sc.pitch_um)
    ntx = -(-sc.W // T); nty = -(-sc.H // T)
    assert count.size == ntx * nty and offset.size == count.size + 1 and offset[0] == 0
    assert np.array_equal(np.diff(offset.astype(np.int64)), count.astype(np.int64))
    assert lst.size == offset[-1]
    for ty in range(nty):
        for tx in range(ntx):
            want = [n for n in range(sc.N) if listed[n]
                    and not (j1[n] < tx * T or j0[n] > tx * T + T - 1 or i1[n] < ty * T or i0[n] > ty * T + T - 1)]
            t = ty * ntx + tx
            assert list(lst[offset[t]:offset[t + 1]]) == want      # ascending particle index


def test_B4_batched_frames_concatenate():
    sc = make_config(5, n_override=40)
    T = 16
    count, offset, lst = o.binning(sc, T)
    tpf = (sc.H // T) * (sc.W // T)
    assert count.size == sc.B * tpf
    fs = sc.frame_start
    for b in (0, 7, 15):
        seg = lst[offset[b * tpf]:offset[(b + 1) * tpf]]
        assert seg.size > 0 and seg.min() >= fs[b] and seg.max() < fs[b + 1]   # global indices, own frame only


def test_pair_counts_of_the_configs_are_sane():
    """Workload statistics quoted in DESIGN.md section 4 (tile 16): total (particle, tile) pairs."""
    c1 = make_config(1)
    count, offset, lst = o.binning(c1, 16)
    assert 400 < offset[-1] < 1200 and count.max() <= 12
    c2 = make_config(2)
    count, offset, lst = o.binning(c2, 16)
    assert 10000 < offset[-1] < 25000
