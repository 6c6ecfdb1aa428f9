"""Pins for the oracle's oriented-bounding-box labels (reading A23): closed forms, containment and
tightness against sampled surface points and against the covered pixels of the thickness oracle."""
import math

import numpy as np

from oracle import oracle as o
from workloads import make_config, make_scene, subset

P = 0.1


def _scene(cols, H=64, W=64):
    return make_scene("obb", H, W, cols)


def _qz(alpha):
    return dict(qw=[math.cos(alpha / 2)], qx=[0.0], qy=[0.0], qz=[math.sin(alpha / 2)])


def test_closed_forms():
    # sphere: a circle, the axis is arbitrary, both half lengths R / p
    b = o.particle_obbs(_scene(dict(cx=[3.21], cy=[2.87], d0=[1.3], d1=[1.3], d2=[1.3], n_p=[1.4])))[0]
    f = lambda v: float(np.float32(v))
    assert abs(b[0] - (f(3.21) / P - 0.5)) < 1e-9 and abs(b[1] - (f(2.87) / P - 0.5)) < 1e-9
    assert abs(b[4] - f(1.3) / P) < 1e-9 and abs(b[5] - f(1.3) / P) < 1e-9
    assert abs(math.hypot(b[2], b[3]) - 1.0) < 1e-12
    # axis-aligned ellipsoid a > b (c plays no part), then rotated about z by alpha: the box turns with it
    for alpha in (0.0, 0.4, -1.1, 1.5):
        cols = dict(cx=[3.0], cy=[3.0], d0=[2.5], d1=[0.75], d2=[1.6], n_p=[1.4], **_qz(alpha))
        b = o.particle_obbs(_scene(cols))[0]
        ux, uy = math.cos(alpha), math.sin(alpha)
        if ux < 0:
            ux, uy = -ux, -uy
        assert abs(b[2] - ux) < 1e-6 and abs(b[3] - uy) < 1e-6          # the quaternion is stored in float32
        assert abs(b[4] - 25.0) < 1e-5 and abs(b[5] - 7.5) < 1e-5
    # prism, identity rotation: the long axis points at the viewer, the shadow is the s x s square, u = (1, 0)
    cols = dict(cx=[3.0], cy=[3.0], d0=[1.2], d1=[3.0], d2=[0.5], n_p=[1.4], kind=np.array([1], np.uint8))
    b = o.particle_obbs(_scene(cols))[0]
    assert np.allclose(b[2:], (1.0, 0.0, 6.0, 6.0), atol=1e-5)
    # prism with the long axis along x (90 degrees about y): half lengths L/2 + hc and s/2
    r = math.sqrt(0.5)
    cols.update(qw=[r], qx=[0.0], qy=[r], qz=[0.0])
    b = o.particle_obbs(_scene(cols))[0]
    assert np.allclose(b[2:], (1.0, 0.0, (1.5 + 0.5) / P, 0.6 / P), atol=1e-4)
    # invalid particle: NaN
    cols["d0"] = [-1.0]
    assert np.all(np.isnan(o.particle_obbs(_scene(cols))[0]))


def test_box_contains_the_body_and_is_tight_on_sampled_surface_points():
    rng = np.random.default_rng(3)
    sc = make_config(4, n_override=60)
    B = o.particle_obbs(sc)
    for n in range(sc.N):
        q = np.array([sc.cols[k][n] for k in ("qw", "qx", "qy", "qz")], dtype=np.float64)
        R = o.rot_from_quat(q)
        d = np.array([sc.cols[k][n] for k in ("d0", "d1", "d2")], dtype=np.float64)
        if sc.cols["kind"][n] == 0:
            v = rng.standard_normal((20000, 3))
            v /= np.linalg.norm(v, axis=1, keepdims=True)
            pts = v * d                                              # points of the ellipsoid's surface
            tight = 2e-3
        else:
            s, L, hc = d
            pts = np.array([(sx * s / 2, sy * s / 2, sz * L / 2) for sx in (1, -1) for sy in (1, -1) for sz in (1, -1)]
                           + [(0, 0, L / 2 + hc), (0, 0, -(L / 2 + hc))])   # a polytope's extremes are vertices
            tight = 1e-9
        xy = (pts @ R.T)[:, :2] / P
        u = B[n, 2:4]
        along, across = xy @ u, xy @ np.array([-u[1], u[0]])
        assert np.abs(along).max() <= B[n, 4] * (1 + 1e-9) and np.abs(across).max() <= B[n, 5] * (1 + 1e-9)
        assert np.abs(along).max() >= B[n, 4] * (1 - tight) and np.abs(across).max() >= B[n, 5] * (1 - tight)


def test_covered_pixels_lie_inside_the_box_and_reach_its_sides():
    sc = make_config(4, n_override=24)
    B = o.particle_obbs(sc)
    jj, ii = np.meshgrid(np.arange(sc.W, dtype=np.float64), np.arange(sc.H, dtype=np.float64))
    for n in range(sc.N):
        one = subset(sc, [n])
        cov = o.render_opd(one)[0] != 0.0
        if not cov.any():
            continue
        dx, dy = jj[cov] - B[n, 0], ii[cov] - B[n, 1]
        u = B[n, 2:4]
        along, across = dx * u[0] + dy * u[1], -dx * u[1] + dy * u[0]
        assert np.abs(along).max() <= B[n, 4] + 1e-9 and np.abs(across).max() <= B[n, 5] + 1e-9
        inside = (0 <= B[n, 0] - B[n, 4] - B[n, 5]) and (B[n, 0] + B[n, 4] + B[n, 5] <= sc.W - 1) and \
                 (0 <= B[n, 1] - B[n, 4] - B[n, 5]) and (B[n, 1] + B[n, 4] + B[n, 5] <= sc.H - 1)
        if inside:                                                   # whole shadow on the canvas: the box is tight to ~1 px
            assert np.abs(along).max() >= B[n, 4] - 1.5 and np.abs(across).max() >= B[n, 5] - 1.5
