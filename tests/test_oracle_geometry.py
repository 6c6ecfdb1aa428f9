"""Pins for the oracle's thickness functions (pins P1-P7, P13).

Nothing here re-types the oracle's formulae: each test compares it with a closed form, an invariant,
a library routine (scipy Rotation / Delaunay / linprog) or brute force by inside-test only.
"""
import math

import numpy as np
import pytest
from scipy.spatial import Delaunay
from scipy.spatial.transform import Rotation

from oracle import oracle as o


def rand_quat(rng, f32=True):
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    return q.astype(np.float32).astype(np.float64) if f32 else q      # the scene stores float32


def scipy_R(q):
    """Library rotation matrix for a (w, x, y, z) quaternion (scipy is scalar-last)."""
    qn = q / np.linalg.norm(q)
    return Rotation.from_quat([qn[1], qn[2], qn[3], qn[0]]).as_matrix()


def quat_mul(a, b):
    w1, x1, y1, z1 = a
    w2, x2, y2, z2 = b
    return np.array([w1 * w2 - x1 * x2 - y1 * y2 - z1 * z2,
                     w1 * x2 + x1 * w2 + y1 * z2 - z1 * y2,
                     w1 * y2 - x1 * z2 + y1 * w2 + z1 * x2,
                     w1 * z2 + x1 * y2 - y1 * x2 + z1 * w2])


def prism_vertices(s, L, hc):
    v = [(sx * s / 2, sy * s / 2, sz * L / 2) for sx in (1, -1) for sy in (1, -1) for sz in (1, -1)]
    v += [(0, 0, L / 2 + hc), (0, 0, -(L / 2 + hc))]
    return np.array(v, dtype=np.float64)


def test_rot_from_quat_matches_scipy():
    rng = np.random.default_rng(10)
    for _ in range(50):
        q = rand_quat(rng)
        R = o.rot_from_quat(q)
        # float32-rounded q is unit only to ~1e-7, and the oracle does not renormalise (reading A4)
        np.testing.assert_allclose(R, scipy_R(q), atol=5e-7)
    # exact cases: 90 degrees about z maps body x to world y
    R = o.rot_from_quat([math.sqrt(0.5), 0, 0, math.sqrt(0.5)])
    np.testing.assert_allclose(R @ [1, 0, 0], [0, 1, 0], atol=1e-15)
    R = o.rot_from_quat([math.sqrt(0.5), math.sqrt(0.5), 0, 0])       # 90 degrees about x: y -> z
    np.testing.assert_allclose(R @ [0, 1, 0], [0, 0, 1], atol=1e-15)


def test_P1_sphere_closed_form_any_quaternion():
    rng = np.random.default_rng(11)
    for _ in range(200):
        Rr = np.float32(rng.uniform(0.3, 5.0))
        q = rand_quat(rng)
        dx, dy = rng.uniform(-1.2, 1.2, size=2) * float(Rr)
        r2 = dx * dx + dy * dy
        want = 2.0 * math.sqrt(float(Rr) ** 2 - r2) if r2 < float(Rr) ** 2 else 0.0
        got = o.thickness(0, q, (Rr, Rr, Rr), dx, dy)
        # q is unit to 1e-7 only, so R R^T = (1 + O(1e-7)) I: the "sphere" is exact to that order
        assert got == pytest.approx(want, abs=2e-6 * float(Rr) / max(math.sqrt(max(1 - r2 / float(Rr) ** 2, 1e-12)), 1e-3))
    # identity quaternion: exact to rounding
    for _ in range(200):
        Rr = np.float32(rng.uniform(0.3, 5.0))
        dx, dy = rng.uniform(-0.99, 0.99, size=2) * float(Rr) / math.sqrt(2)
        want = 2.0 * math.sqrt(float(Rr) ** 2 - dx * dx - dy * dy)
        assert o.thickness(0, (1, 0, 0, 0), (Rr, Rr, Rr), dx, dy) == pytest.approx(want, rel=1e-12)
    assert o.thickness(0, (1, 0, 0, 0), (2, 2, 2), 2.0001, 0.0) == 0.0
    assert o.thickness(0, (1, 0, 0, 0), (2, 2, 2), 0.0, 0.0) == pytest.approx(4.0, rel=1e-15)


def test_P2_axis_aligned_ellipsoid_and_axis_permutations():
    rng = np.random.default_rng(12)
    h = math.sqrt(0.5)
    # (quaternion, which body axis ends up along world x, y, z)
    cases = [((1, 0, 0, 0), (0, 1, 2)),
             ((h, 0, 0, h), (1, 0, 2)),      # 90 about z: world x <- body y, world y <- body x
             ((h, h, 0, 0), (0, 2, 1)),      # 90 about x: world y <- body z, world z <- body y
             ((h, 0, h, 0), (2, 1, 0))]      # 90 about y: world x <- body z, world z <- body x
    for q, perm in cases:
        for _ in range(100):
            ax = rng.uniform(0.5, 4.0, size=3).astype(np.float32)
            a, b, c = (float(ax[perm[0]]), float(ax[perm[1]]), float(ax[perm[2]]))   # world-axis semi-axes
            dx = rng.uniform(-1.1, 1.1) * a
            dy = rng.uniform(-1.1, 1.1) * b
            u = (dx / a) ** 2 + (dy / b) ** 2
            want = 2.0 * c * math.sqrt(1.0 - u) if u < 1.0 else 0.0
            got = o.thickness(0, q, ax, dx, dy)
            tol = 1e-9 if abs(1.0 - u) > 1e-6 else 1e-5
            assert got == pytest.approx(want, abs=tol)


def test_P3_schur_complement_projection_and_central_thickness():
    rng = np.random.default_rng(13)
    for _ in range(100):
        q = rand_quat(rng)
        ax = rng.uniform(0.5, 4.0, size=3).astype(np.float32).astype(np.float64)
        R = scipy_R(q)
        # shadow of an ellipsoid: d^T S d <= 1 with S^-1 = (R diag(a^2) R^T)_xy ; chord = T0 sqrt(1 - d^T S d)
        Cov = R @ np.diag(ax ** 2) @ R.T
        S = np.linalg.inv(Cov[:2, :2])
        M = R @ np.diag(1.0 / ax ** 2) @ R.T
        T0 = 2.0 / math.sqrt(M[2, 2])
        assert o.thickness(0, q, ax, 0.0, 0.0) == pytest.approx(T0, rel=1e-6)
        for _ in range(20):
            d = rng.uniform(-4, 4, size=2)
            u = d @ S @ d
            want = T0 * math.sqrt(1.0 - u) if u < 1.0 else 0.0
            got = o.thickness(0, q, ax, d[0], d[1])
            if abs(1.0 - u) > 1e-3:
                assert got == pytest.approx(want, rel=2e-5, abs=1e-9)


def test_P4_rotation_about_z_rotates_the_shadow():
    rng = np.random.default_rng(14)
    for kind in (0, 1):
        for _ in range(60):
            q = rand_quat(rng, f32=False)        # exactly unit: R(qz q) = Rz R(q) holds for unit quaternions
            dims = rng.uniform(0.8, 3.0, size=3).astype(np.float32)
            al = rng.uniform(0, 2 * math.pi)
            qz = np.array([math.cos(al / 2), 0, 0, math.sin(al / 2)])
            q2 = quat_mul(qz, q)
            d = rng.uniform(-2.5, 2.5, size=2)
            d2 = np.array([math.cos(al) * d[0] - math.sin(al) * d[1], math.sin(al) * d[0] + math.cos(al) * d[1]])
            t1 = o.thickness(kind, q, dims, d[0], d[1])
            t2 = o.thickness(kind, q2, dims, d2[0], d2[1])
            assert t2 == pytest.approx(t1, abs=1e-9)


def test_P5_prism_closed_forms():
    s, L, hc = np.float32(2.0), np.float32(5.0), np.float32(1.0)
    s_, L_, hc_ = float(s), float(L), float(hc)
    rng = np.random.default_rng(15)
    # identity: long axis along z, looking down the axis: t = L + 2 hc (1 - max(|dx|,|dy|)/(s/2))
    for _ in range(200):
        dx, dy = rng.uniform(-0.999, 0.999, size=2) * s_ / 2
        want = L_ + 2 * hc_ * (1 - max(abs(dx), abs(dy)) / (s_ / 2))
        assert o.thickness(1, (1, 0, 0, 0), (s, L, hc), dx, dy) == pytest.approx(want, rel=1e-12)
    assert o.thickness(1, (1, 0, 0, 0), (s, L, hc), s_ / 2 + 1e-3, 0.0) == 0.0
    # 90 degrees about x: body z -> world -y ... long axis along world y
    h = math.sqrt(0.5)
    q = (h, h, 0, 0)
    for _ in range(300):
        dx = rng.uniform(-0.6, 0.6) * s_
        dy = rng.uniform(-0.55, 0.55) * (L_ + 2 * hc_)
        if abs(dy) <= L_ / 2:
            want = s_ if abs(dx) < s_ / 2 else 0.0
            if abs(abs(dx) - s_ / 2) < 1e-6:
                continue
        else:
            w = (s_ / 2) * (1 - (abs(dy) - L_ / 2) / hc_)
            want = 2 * w if (w > 0 and abs(dx) < w) else 0.0
            if abs(abs(dx) - w) < 1e-6:
                continue
        assert o.thickness(1, q, (s, L, hc), dx, dy) == pytest.approx(want, abs=1e-12)


def test_P6_volume_invariant_under_rotation():
    rng = np.random.default_rng(16)
    p = 0.01
    g = (np.arange(-700, 700) + 0.5) * p
    for kind in (0, 1):
        for _ in range(3):
            q = rand_quat(rng)
            if kind == 0:
                dims = rng.uniform(1.0, 3.0, size=3).astype(np.float32)
                vol = 4.0 / 3.0 * math.pi * float(dims[0]) * float(dims[1]) * float(dims[2])
            else:
                s = rng.uniform(1.0, 2.5); L = s * rng.uniform(1.0, 2.0); hc = 0.5 * s
                dims = np.array([s, L, hc], dtype=np.float32)
                s, L, hc = map(float, dims)
                vol = s * s * L + 2.0 / 3.0 * s * s * hc
            cols = dict(cx=[0.0], cy=[0.0], qw=[q[0]], qx=[q[1]], qy=[q[2]], qz=[q[3]],
                        d0=[dims[0]], d1=[dims[1]], d2=[dims[2]], n_p=[2.0], kind=[kind])
            cols = {k: np.asarray(v, dtype=np.uint8 if k == "kind" else np.float32) for k, v in cols.items()}
            # frame centred on the particle: shift the centre to the middle of a 1400 x 1400 frame
            cols["cx"][:] = 7.0; cols["cy"][:] = 7.0
            opd = o.render_opd_frame(cols, 0, 1, 1400, 1400, p, 1.0, "full")      # (n_p - n_m) = 1 -> thickness
            assert opd.sum() * p * p == pytest.approx(vol, rel=2e-4)


def test_P7_vertices_satisfy_planes_with_three_equalities_and_symmetry():
    rng = np.random.default_rng(17)
    for _ in range(20):
        s = rng.uniform(1, 5); L = s * rng.uniform(1, 3); hc = 0.5 * s
        A, b = o.prism_planes(s, L, hc)
        assert A.shape == (12, 3)
        V = prism_vertices(s, L, hc)
        slack = b[None, :] - V @ A.T                       # [10, 12] >= 0
        assert slack.min() > -1e-12
        tight = (np.abs(slack) < 1e-12).sum(axis=1)
        assert (tight >= 3).all()
        # every plane holds at least 3 vertices (it is a face, not a redundant constraint)
        assert ((np.abs(slack) < 1e-12).sum(axis=0) >= 3).all()
        # centrally symmetric: the plane set is closed under n -> -n with the same offset
        for k in range(12):
            assert any(np.allclose(A[m], -A[k]) and b[m] == pytest.approx(b[k]) for m in range(12))
        q = rand_quat(rng)
        for _ in range(20):
            d = rng.uniform(-3, 3, size=2)
            for kind in (0, 1):
                t1 = o.thickness(kind, q, (s, L, hc), d[0], d[1])
                t2 = o.thickness(kind, q, (s, L, hc), -d[0], -d[1])
                assert t1 == pytest.approx(t2, abs=1e-12)


@pytest.mark.parametrize("kind", [0, 1])
def test_P13_brute_force_ray_marching_inside_test_only(kind):
    """8 x 8 frame, coarse pitch so the particle spans it; march z in steps of 1e-3 um and count points that
    pass the INSIDE TEST (ellipsoid: |D^-1/2 R^T q| <= 1 with scipy's rotation; prism: inside the convex hull
    of its 10 rotated vertices, scipy Delaunay) - no intersection algebra."""
    rng = np.random.default_rng(18 + kind)
    dz = 1e-3
    for trial in range(3):
        q = rand_quat(rng)
        R = scipy_R(q)
        if kind == 0:
            dims = rng.uniform(1.0, 3.0, size=3).astype(np.float32)
        else:
            s = rng.uniform(1.5, 3.0)
            dims = np.array([s, s * rng.uniform(1.0, 2.0), 0.5 * s], dtype=np.float32)
        rmax = o.circumradius(kind, dims)
        pitch = 2.2 * rmax / 8
        c = 4 * pitch + rng.uniform(-0.5, 0.5, size=2) * pitch          # sub-pixel shifted centre
        cols = dict(cx=[c[0]], cy=[c[1]], qw=[q[0]], qx=[q[1]], qy=[q[2]], qz=[q[3]],
                    d0=[dims[0]], d1=[dims[1]], d2=[dims[2]], n_p=[2.0], kind=[kind])
        cols = {k: np.asarray(v, dtype=np.uint8 if k == "kind" else np.float32) for k, v in cols.items()}
        got = o.render_opd_frame(cols, 0, 1, 8, 8, pitch, 1.0, "full")
        z = (np.arange(int(2 * rmax / dz) + 2) + 0.5) * dz - rmax - dz
        d64 = dims.astype(np.float64)
        if kind == 1:
            hull = Delaunay(prism_vertices(*d64) @ R.T)
        covered = 0
        for i in range(8):
            for j in range(8):
                dx = (j + 0.5) * pitch - float(cols["cx"][0])
                dy = (i + 0.5) * pitch - float(cols["cy"][0])
                P = np.stack([np.full_like(z, dx), np.full_like(z, dy), z], axis=1)
                if kind == 0:
                    body = P @ R                                                   # R^T q per row
                    inside = ((body / d64) ** 2).sum(axis=1) <= 1.0
                else:
                    inside = hull.find_simplex(P) >= 0
                t_march = inside.sum() * dz
                covered += t_march > 0
                assert got[i, j] == pytest.approx(t_march, abs=2 * dz + 1e-6 * rmax)
        assert covered >= 12         # the test really exercises covered pixels and the silhouette


# ---- workload statistic: covered (particle, pixel) pairs (bench.py's ALU roofline units) -------------------------------
def test_count_covered_sphere_is_the_gauss_circle_count_and_golden_file_matches():
    from workloads import make_scene, make_config, CONFIG_NAMES
    import os
    # two spheres + one prism with identity rotation: pixel centres strictly inside the disc r < R, or inside the square
    # |dx|, |dy| < s/2 (pin P5: the identity prism's shadow is the square), counted directly with numpy
    H = W = 96
    p = 0.1
    cols = dict(cx=[3.07, 6.51, 4.83], cy=[4.12, 2.93, 7.0], d0=[1.7, 0.93, 1.24], d1=[1.7, 0.93, 2.0], d2=[1.7, 0.93, 0.6],
                n_p=[1.4, 1.4, 1.4], kind=np.array([0, 0, 1], np.uint8))
    sc = make_scene("count", H, W, cols)
    x = (np.arange(W) + 0.5) * p
    X, Y = np.meshgrid(x, x)
    f = lambda v: float(np.float32(v))
    want_e = sum(int(np.count_nonzero((X - f(cx)) ** 2 + (Y - f(cy)) ** 2 < f(r) ** 2))
                 for cx, cy, r in zip(cols["cx"][:2], cols["cy"][:2], cols["d0"][:2]))
    want_p = int(np.count_nonzero((np.abs(X - f(4.83)) < f(1.24) / 2) & (np.abs(Y - f(7.0)) < f(1.24) / 2)))
    for mode in ("full", "bcircle"):
        assert o.count_covered(sc, mode) == (want_e, want_p)
    # the stored counts are what the oracle gives today for ALL five workloads (config 4's pair is the numerator of
    # bench.py's headline ALU roofline fraction; config 1: also = non-zero thickness pixels summed over single-particle renders)
    stored = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "covered_pairs.txt")) as fh:
        for ln in fh:
            q = ln.split()
            if len(q) == 3 and not ln.startswith("#"):
                stored[q[0]] = (int(q[1]), int(q[2]))
    assert set(stored) == set(CONFIG_NAMES.values())
    for cfg in (1, 2, 3, 4, 5):
        assert o.count_covered(make_config(cfg)) == stored[CONFIG_NAMES[cfg]]
    sc1 = make_config(1)
    from workloads import subset
    tot = sum(int(np.count_nonzero(o.render_opd(subset(sc1, [n]))[0])) for n in range(sc1.N))
    assert tot == stored[CONFIG_NAMES[1]][0]
