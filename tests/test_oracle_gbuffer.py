"""Pins for the oracle's G-buffer extras (depth map and instance-id map, reading A24): closed forms,
consistency with the pinned thickness function, a library rotation for the chord's midpoint, brute-force marching with
the inside test only, tie and permutation behaviour."""
import math

import numpy as np
from scipy.spatial.transform import Rotation

from oracle import oracle as o
from workloads import make_scene, subset

P = 0.1


def rand_quat(rng):
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    return q.astype(np.float32).astype(np.float64)


def scipy_R(q):
    qn = q / np.linalg.norm(q)
    return Rotation.from_quat([qn[1], qn[2], qn[3], qn[0]]).as_matrix()


def test_G1_sphere_depth_and_id():
    H = W = 64
    R, cz = 1.7, 0.35
    sc = make_scene("g", H, W, dict(cx=[3.23], cy=[3.11], cz=[cz], d0=[R], d1=[R], d2=[R], n_p=[1.4]))
    tid, dep = o.render_gbuffer(sc)
    f = lambda v: float(np.float32(v))
    x = (np.arange(W) + 0.5) * P
    X, Y = np.meshgrid(x, x)
    r2 = (X - f(3.23)) ** 2 + (Y - f(3.11)) ** 2
    inside = r2 < f(R) ** 2
    assert np.array_equal(tid[0] >= 0, inside) and np.all(tid[0][inside] == 0) and np.all(tid[0][~inside] == -1)
    assert np.allclose(dep[0][inside], f(cz) + np.sqrt(f(R) ** 2 - r2[inside]), atol=1e-12) and np.all(dep[0][~inside] == 0.0)
    assert o.chord(0, [1, 0, 0, 0], [1.0, 1.0, 1.0], 0.6, 0.0) == (-0.8, 0.8)
    assert o.chord(0, [1, 0, 0, 0], [1.0, 1.0, 1.0], 1.0, 0.2) is None


def test_G2_chord_is_consistent_with_the_pinned_thickness_and_centrally_symmetric():
    rng = np.random.default_rng(8)
    for kind in (0, 1):
        for _ in range(200):
            q = rand_quat(rng)
            dims = rng.uniform(0.5, 3.0, 3)
            dx, dy = rng.uniform(-2.5, 2.5, 2)
            c = o.chord(kind, q, dims, dx, dy)
            t = o.thickness(kind, q, dims, dx, dy)
            if c is None:
                assert t == 0.0
                continue
            assert abs((c[1] - c[0]) - t) <= 1e-12 * max(1.0, t) and t > 0.0
            m = o.chord(kind, q, dims, -dx, -dy)
            assert abs(m[0] + c[1]) < 1e-12 and abs(m[1] + c[0]) < 1e-12


def test_G3_prism_identity_and_ellipsoid_midpoint_closed_forms():
    s, L, hc = 1.2, 3.0, 0.5
    for dx, dy in ((0.0, 0.0), (0.31, -0.12), (-0.55, 0.2), (0.1, 0.59)):
        ze, zx = o.chord(1, [1, 0, 0, 0], [s, L, hc], dx, dy)
        want = L / 2 + hc * (1 - max(abs(dx), abs(dy)) / (s / 2))
        assert abs(zx - want) < 1e-12 and abs(ze + want) < 1e-12
    # ellipsoid: the chord's midpoint is z = -(M_xz dx + M_yz dy) / M_zz, M from a library rotation matrix
    rng = np.random.default_rng(2)
    for _ in range(50):
        q, dims = rand_quat(rng), rng.uniform(0.5, 3.0, 3)
        Rm = scipy_R(q)
        M = Rm @ np.diag(1.0 / dims ** 2) @ Rm.T
        dx, dy = rng.uniform(-0.3, 0.3, 2)
        ze, zx = o.chord(0, q, dims, dx, dy)
        assert abs(0.5 * (ze + zx) + (M[0, 2] * dx + M[1, 2] * dy) / M[2, 2]) < 1e-6      # float32 quaternion: |q| = 1 +- 6e-8


def test_G4_marching_with_the_inside_test_finds_the_same_top():
    """Walk down the vertical line in steps of 1e-3 um and take the first point inside the body (inside test only:
    q^T D q <= 1 in body coordinates / A x <= b): it lies within one step below the oracle's z_exit."""
    rng = np.random.default_rng(4)
    dz = 1e-3
    zs = np.arange(6.0, -6.0, -dz)
    for kind in (0, 1):
        for _ in range(12):
            q, dims = rand_quat(rng), rng.uniform(0.6, 2.5, 3)
            Rm = scipy_R(q)
            dx, dy = rng.uniform(-0.4, 0.4, 2)
            pts = np.stack([np.full_like(zs, dx), np.full_like(zs, dy), zs], axis=1) @ Rm          # body coordinates R^T x
            if kind == 0:
                inside = ((pts / dims) ** 2).sum(axis=1) <= 1.0
            else:
                A, b = o.prism_planes(*dims)
                inside = np.all(pts @ np.asarray(A).T <= np.asarray(b)[None, :], axis=1)
            c = o.chord(kind, q, dims, dx, dy)
            assert c is not None and inside.any()
            top = zs[np.argmax(inside)]
            assert -1e-5 <= c[1] - top <= dz + 1e-5, (kind, c, top)      # 1e-5: the marching uses a renormalised rotation


def test_G5_overlap_ties_permutation_and_modes():
    H = W = 64
    # a small sphere floating above a big one with the same axis: it owns the pixels of its disc, the big one the ring
    cols = dict(cx=[3.2, 3.2], cy=[3.2, 3.2], cz=[0.0, 1.5], d0=[2.0, 1.0], d1=[2.0, 1.0], d2=[2.0, 1.0], n_p=[1.4, 1.4])
    sc = make_scene("two", H, W, cols)
    tid, dep = o.render_gbuffer(sc)
    x = (np.arange(W) + 0.5) * P
    X, Y = np.meshgrid(x, x)
    r2 = (X - float(np.float32(3.2))) ** 2 + (Y - float(np.float32(3.2))) ** 2
    small_top = 1.5 + np.sqrt(np.maximum(1.0 - r2, 0.0))
    big_top = np.sqrt(np.maximum(4.0 - r2, 0.0))
    owns = (r2 < 1.0) & (small_top > big_top)                 # near its rim the small sphere dips below the big one's top
    assert owns.sum() > 100 and ((r2 < 1.0) & ~owns).sum() > 10
    assert np.all(tid[0][owns] == 1) and np.all(tid[0][(r2 < 4.0) & ~owns] == 0) and np.all(tid[0][r2 > 4.0] == -1)
    assert np.allclose(dep[0][owns], small_top[owns], atol=1e-12)
    assert np.allclose(dep[0][(r2 < 4.0) & ~owns], big_top[(r2 < 4.0) & ~owns], atol=1e-12)
    # below the big sphere's top the small one loses everywhere
    sc2 = make_scene("two", H, W, dict(cols, cz=[0.0, -0.5]))
    assert np.all(o.render_gbuffer(sc2)[0][0][r2 < 4.0] == 0)
    # exact tie (two identical particles): the smaller index wins
    sc3 = make_scene("tie", H, W, dict(cx=[3.2, 3.2], cy=[3.2, 3.2], cz=[0.2, 0.2], d0=[1.5] * 2, d1=[1.5] * 2, d2=[1.5] * 2,
                                         n_p=[1.4] * 2))
    t3 = o.render_gbuffer(sc3)[0][0]
    assert set(np.unique(t3)) == {-1, 0}
    # random mixed scene with random heights: the depth map does not depend on the particle order, the id map follows the
    # permutation; bcircle == full bit for bit
    rng = np.random.default_rng(6)
    n = 40
    qn = rng.standard_normal((n, 4)); qn /= np.linalg.norm(qn, axis=1, keepdims=True)
    kind = (np.arange(n) % 2).astype(np.uint8)
    cols = dict(cx=rng.uniform(0, 6.4, n), cy=rng.uniform(0, 6.4, n), cz=rng.uniform(-3, 3, n), d0=rng.uniform(0.4, 1.5, n),
                d1=rng.uniform(0.4, 2.5, n), d2=rng.uniform(0.3, 1.2, n), n_p=rng.uniform(1.36, 1.5, n),
                qw=qn[:, 0], qx=qn[:, 1], qy=qn[:, 2], qz=qn[:, 3], kind=kind)
    sc4 = make_scene("mix", H, W, cols)
    tid, dep = o.render_gbuffer(sc4)
    tid_f, dep_f = o.render_gbuffer(sc4, mode="full")
    assert np.array_equal(tid, tid_f) and np.array_equal(dep, dep_f)
    perm = rng.permutation(n)
    tid_p, dep_p = o.render_gbuffer(subset(sc4, perm))
    assert np.array_equal(dep_p, dep)
    back = np.where(tid_p >= 0, perm[np.maximum(tid_p, 0)], -1)
    assert np.array_equal(back, tid)
    # coverage agrees with the OPD frame: a pixel has an owner iff some particle has positive thickness there
    assert np.array_equal(tid[0] >= 0, o.render_opd(sc4)[0] != 0.0)
    assert len(np.unique(tid)) > 10


# ---- analytic slope of the visible surface ("the analytic height gradient / normal that falls out of the
# same ray test") ---------------------------------------------------------------------------------------------
def test_G6_top_slope_closed_forms_and_differenced_chord():
    # sphere: top z = sqrt(R^2 - r^2), dz/dx = -dx / z
    R, dx, dy = 2.0, 0.9, -0.5
    z = np.sqrt(R * R - dx * dx - dy * dy)
    sx, sy = o.top_slope(0, [1, 0, 0, 0], [R, R, R], dx, dy)
    assert abs(sx + dx / z) < 1e-13 and abs(sy + dy / z) < 1e-13
    assert o.top_slope(0, [1, 0, 0, 0], [R, R, R], 2.5, 0.0) is None
    # prism, identity rotation: top = cap faces z = L/2 + hc (1 - |x| / (s/2)) on the side where |x| > |y|: slope -+ 2 hc / s
    s_, L, hc = 2.0, 3.0, 0.8
    sx, sy = o.top_slope(1, [1, 0, 0, 0], [s_, L, hc], 0.6, 0.2)
    assert abs(sx + 2 * hc / s_) < 1e-13 and abs(sy) < 1e-13
    sx, sy = o.top_slope(1, [1, 0, 0, 0], [s_, L, hc], 0.1, -0.7)
    assert abs(sx) < 1e-13 and abs(sy - 2 * hc / s_) < 1e-13
    # any rotation, both kinds: central differences of the pinned chord's z_exit (G1-G4) at interior points
    rng = np.random.default_rng(6)
    h = 1e-6
    checked = 0
    for trial in range(80):
        kind = trial % 2
        q = rng.standard_normal(4); q /= np.linalg.norm(q)
        dims = rng.uniform(0.8, 3.0, 3)
        dx, dy = rng.uniform(-1.0, 1.0, 2)
        c0 = o.chord(kind, q, dims, dx, dy)
        if c0 is None or c0[1] - c0[0] < 0.3:
            continue
        zs = [o.chord(kind, q, dims, dx + a, dy + b)[1] for a, b in ((h, 0), (-h, 0), (0, h), (0, -h))]
        if abs(zs[0] + zs[1] - 2 * c0[1]) > 1e-9 or abs(zs[2] + zs[3] - 2 * c0[1]) > 1e-9:      # a face edge inside the stencil (prism)
            if kind == 1:
                continue
        sx, sy = o.top_slope(kind, q, dims, dx, dy)
        assert abs(sx - (zs[0] - zs[1]) / (2 * h)) < 2e-6 * max(1, abs(sx)) and abs(sy - (zs[2] - zs[3]) / (2 * h)) < 2e-6 * max(1, abs(sy))
        checked += 1
    assert checked > 40


def test_G7_normal_map_belongs_to_the_owner():
    from workloads import make_config
    sc = make_config(4, n_override=60)
    from dataclasses import replace
    for k in ("cx", "cy"):
        sc.cols[k][:] = (sc.cols[k] / 16.0).astype(np.float32)
    sc = replace(sc, H=128, W=128)
    tid, dep, nrm = o.render_gbuffer(sc, normals=True)
    t2, d2 = o.render_gbuffer(sc)
    assert np.array_equal(tid, t2) and np.array_equal(dep, d2)
    assert np.all(nrm[tid < 0] == 0.0)
    c = sc.cols
    for (i, j) in np.argwhere(tid[0] >= 0)[::97]:
        n = int(tid[0, i, j])
        want = o.top_slope(int(c["kind"][n]), [float(c[k][n]) for k in ("qw", "qx", "qy", "qz")], [float(c[k][n]) for k in ("d0", "d1", "d2")],
                           (j + 0.5) * sc.pitch_um - float(c["cx"][n]), (i + 0.5) * sc.pitch_um - float(c["cy"][n]))
        assert np.allclose(nrm[0, i, j], want, rtol=0, atol=0)
