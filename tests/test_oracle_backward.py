"""Pins for the oracle's first backward step (dL/dn_p, the adjoint of the OPD sum in the refractive indices; PAPER.md:124,
SURVEY 8(f) NEXT-3): closed form, the forward model differenced, linearity."""
from dataclasses import replace

import numpy as np

from oracle import oracle as o
from workloads import make_config, make_scene, subset

P = 0.1


def test_B1_unit_gradient_gives_the_discrete_volume():
    # G == 1: dL/dn_p[n] = sum of the particle's thickness over the pixels = its height map summed (and ~ volume / p^2)
    sc = make_config(4, n_override=20)
    g = o.backward_np(sc, np.ones((1, sc.H, sc.W), np.float32))
    for n in range(sc.N):
        assert abs(g[n] - o.render_height(subset(sc, [n]))[0].sum()) <= 1e-9 * max(1.0, g[n])
    R = 2.0
    one = make_scene("s", 96, 96, dict(cx=[4.8], cy=[4.8], d0=[R], d1=[R], d2=[R], n_p=[1.4]))
    vol = o.backward_np(one, np.ones((1, 96, 96), np.float32))[0] * P * P
    assert abs(vol - 4.0 / 3.0 * np.pi * R ** 3) < 2e-3 * vol


def test_B2_equals_the_forward_model_differenced_in_n_p():
    """L = sum_px G OPD is linear in every n_p: (L(n_p + d e_n) - L(n_p)) / d is the gradient, whatever d."""
    rng = np.random.default_rng(0)
    sc = make_config(4, n_override=16)
    G = rng.standard_normal((1, sc.H, sc.W)).astype(np.float32)
    g = o.backward_np(sc, G)
    L0 = float((G.astype(np.float64) * o.render_opd(sc)).sum())
    for n in (0, 5, 11):
        cols = dict(sc.cols)
        npn = cols["n_p"].copy()
        d = np.float32(0.25)
        npn[n] = npn[n] + d
        cols["n_p"] = npn
        L1 = float((G.astype(np.float64) * o.render_opd(replace(sc, cols=cols))).sum())
        step = float(npn[n]) - float(sc.cols["n_p"][n])           # the float32 step actually taken
        assert abs((L1 - L0) / step - g[n]) <= 1e-8 * max(1.0, abs(g[n]))
    # invalid particle: gradient 0; mode full == bcircle bit for bit
    assert np.array_equal(g, o.backward_np(sc, G, mode="full"))
    cols = dict(sc.cols); bad = cols["d0"].copy(); bad[3] = -1.0; cols["d0"] = bad
    assert o.backward_np(replace(sc, cols=cols), G)[3] == 0.0


def test_B3_linear_in_the_upstream_gradient_and_per_frame():
    rng = np.random.default_rng(1)
    sc = make_config(5, n_override=12)
    G1 = rng.standard_normal((sc.B, sc.H, sc.W)).astype(np.float32)
    G2 = rng.standard_normal((sc.B, sc.H, sc.W)).astype(np.float32)
    a, b = o.backward_np(sc, G1), o.backward_np(sc, G2)
    assert np.allclose(o.backward_np(sc, (G1 + G2).astype(np.float32)), a + b, rtol=1e-5, atol=1e-4)
    G3 = G1.copy(); G3[1:] = 0.0                                   # only frame 0 carries a gradient
    g3 = o.backward_np(sc, G3)
    fs = sc.frame_start
    assert np.all(g3[fs[1]:] == 0.0) and np.array_equal(g3[:fs[1]], a[:fs[1]])


# ---- gradient of the thickness in the lateral position, and dL/d(centre) -----------------------------------------------------
def _rq(rng):
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    return q.astype(np.float32).astype(np.float64)


def test_B4_thickness_gradient_closed_forms():
    # sphere: t = 2 sqrt(R^2 - r^2)  =>  grad t = -2 d / sqrt(R^2 - r^2); outside: 0
    R = 1.7
    for dx, dy in ((0.0, 0.0), (0.4, -0.9), (-1.2, 0.7)):
        gx, gy = o.thickness_grad(0, [1, 0, 0, 0], [R, R, R], dx, dy)
        s = np.sqrt(R * R - dx * dx - dy * dy)
        assert abs(gx + 2 * dx / s) < 1e-12 and abs(gy + 2 * dy / s) < 1e-12
    assert o.thickness_grad(0, [1, 0, 0, 0], [R, R, R], 1.5, 1.0) == (0.0, 0.0)
    # prism, identity rotation: t = L + 2 hc (1 - max(|dx|, |dy|) / (s/2))  =>  slope -+ 2 hc / (s/2) along the dominant axis
    s, L, hc = 1.2, 3.0, 0.5
    k = 2 * hc / (s / 2)
    assert np.allclose(o.thickness_grad(1, [1, 0, 0, 0], [s, L, hc], 0.3, 0.1), (-k, 0.0), atol=1e-12)
    assert np.allclose(o.thickness_grad(1, [1, 0, 0, 0], [s, L, hc], -0.3, 0.1), (k, 0.0), atol=1e-12)
    assert np.allclose(o.thickness_grad(1, [1, 0, 0, 0], [s, L, hc], 0.1, -0.4), (0.0, k), atol=1e-12)
    assert o.thickness_grad(1, [1, 0, 0, 0], [s, L, hc], 0.7, 0.0) == (0.0, 0.0)


def test_B5_thickness_gradient_is_the_pinned_thickness_differenced():
    """Central differences of the (pinned) thickness function, away from the silhouette and from face edges: the prism is
    piecewise linear (exact up to rounding), the ellipsoid smooth (O(h^2))."""
    rng = np.random.default_rng(12)
    h = 1e-5
    checked = 0
    for kind in (0, 1):
        for _ in range(300):
            q, dims = _rq(rng), rng.uniform(0.6, 3.0, 3)
            dx, dy = rng.uniform(-1.5, 1.5, 2)
            t0 = o.thickness(kind, q, dims, dx, dy)
            if t0 < 0.2:
                continue
            fx = (o.thickness(kind, q, dims, dx + h, dy) - o.thickness(kind, q, dims, dx - h, dy)) / (2 * h)
            fy = (o.thickness(kind, q, dims, dx, dy + h) - o.thickness(kind, q, dims, dx, dy - h)) / (2 * h)
            # skip points within h of a face edge of the prism (the slope jumps there): detected by a second difference
            if kind == 1:
                sx = o.thickness(kind, q, dims, dx + h, dy) + o.thickness(kind, q, dims, dx - h, dy) - 2 * t0
                sy = o.thickness(kind, q, dims, dx, dy + h) + o.thickness(kind, q, dims, dx, dy - h) - 2 * t0
                if abs(sx) > 1e-9 or abs(sy) > 1e-9:
                    continue
            gx, gy = o.thickness_grad(kind, q, dims, dx, dy)
            assert abs(gx - fx) <= 1e-6 * max(1.0, abs(gx)) and abs(gy - fy) <= 1e-6 * max(1.0, abs(gy)), (kind, gx, fx, gy, fy)
            checked += 1
    assert checked > 300


def test_B6_backward_centre_sums_the_pixel_gradients_and_matches_a_shifted_render():
    rng = np.random.default_rng(3)
    sc = make_config(4, n_override=12)
    G = rng.standard_normal((1, sc.H, sc.W)).astype(np.float32)
    gc = o.backward_centre(sc, G)
    assert np.array_equal(gc, o.backward_centre(sc, G, mode="full"))
    # one prism (piecewise linear thickness): L(cx + d) - L(cx - d) over 2 d with the oracle's own forward render; the
    # silhouette and the face edges sweep over a few pixel centres during the shift, so the agreement is to ~1e-3 only
    n = int(np.nonzero(sc.cols["kind"] == 1)[0][0])
    one = subset(sc, [n])
    g1 = o.backward_centre(one, G)[0]
    assert np.allclose(g1, gc[n], rtol=1e-12, atol=1e-12)
    d = 2.0 ** -12                                                # exactly representable shift of the float32 centre
    for axis, key in ((0, "cx"), (1, "cy")):
        Ls = []
        for sgn in (+1, -1):
            cols = dict(one.cols); c = cols[key].copy(); c[0] = np.float32(c[0] + sgn * d); cols[key] = c
            Ls.append(float((G.astype(np.float64) * o.render_opd(replace(one, cols=cols))).sum()))
        fd = (Ls[0] - Ls[1]) / (2 * d)
        scale = float(np.abs(G).max()) * 50.0
        assert abs(fd - g1[axis]) <= 2e-2 * max(abs(g1[axis]), scale), (fd, g1[axis])


def test_B7_adjoint_of_the_optics_stage_is_the_forward_model_differenced():
    """L = sum W I with random weights W: dL/dOPD[px] from backward_intensity equals (L(OPD + d e_px) - L(OPD - d e_px)) / 2d
    computed with the oracle's own forward functions (field, pupil, intensity), with and without defocus and ramp."""
    rng = np.random.default_rng(21)
    H, W_ = 24, 32
    lam, p = 0.55, 0.1
    for dz, tilt, NA in ((0.0, 0.0, 1.2), (1.3, 0.08, 1.0)):
        opd = rng.uniform(0.0, 0.8, (H, W_))
        Wt = rng.standard_normal((H, W_))
        P = o.pupil_function(H, W_, NA, p, lam, 1.33, dz)
        assert 10 < (np.abs(P) > 0).sum() < H * W_

        def L(opd_):
            return float((Wt * o.intensity(o.field(opd_, lam, p, tilt, 0.0), P)).sum())

        sc = make_scene("adj", H, W_, dict(cx=[], cy=[], d0=[], d1=[], d2=[], n_p=[]), lam=lam, NA=NA, tilt_x_rad=tilt,
                        defocus_um=dz)
        U = o.field(opd, lam, p, tilt, 0.0)[None]
        g = o.backward_intensity(sc, Wt[None], U=U)[0]
        d = 1e-6
        for (i, j) in ((0, 0), (5, 7), (23, 31), (11, 16), (2, 30)):
            e = np.zeros_like(opd); e[i, j] = d
            fd = (L(opd + e) - L(opd - e)) / (2 * d)
            assert abs(fd - g[i, j]) <= 1e-6 * max(1.0, abs(g[i, j])), (dz, i, j, fd, g[i, j])
    # all-pass pupil: I == 1 whatever the OPD, so every gradient vanishes
    sc0 = replace(sc, defocus_um=0.0)
    assert np.abs(o.backward_intensity(sc0, Wt[None], U=U, pupil_enabled=False)).max() < 1e-12
