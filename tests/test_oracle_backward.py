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


# ---- third step: shape parameters (dimensions, rotation) and the spectral loss of Eq. 8 -------------------------------------
def _interior_points(kind, q, dims, rng, n):
    """Offsets with a comfortably positive chord (not within a few 1e-3 of an outline or of a face change)."""
    pts = []
    r = o.circumradius(kind, dims)
    while len(pts) < n:
        dx, dy = rng.uniform(-r, r, 2)
        if o.thickness(kind, q, dims, dx, dy) > 0.05 * r:
            pts.append((dx, dy))
    return pts


def test_B8_shape_gradient_equals_the_differenced_thickness():
    """dt/d(d0, d1, d2, qw, qx, qy, qz) against central differences of the pinned thickness (P1-P7, P13) at interior points,
    both kinds, random rotations (the quaternion is NOT re-normalised after the step: the components are independent)."""
    rng = np.random.default_rng(8)
    h = 1e-6
    checked = 0
    for trial in range(60):
        kind = trial % 2
        q = rng.standard_normal(4); q /= np.linalg.norm(q)
        dims = rng.uniform(0.8, 3.0, 3) if kind == 0 else np.array([rng.uniform(1, 3), rng.uniform(2, 6), rng.uniform(0.5, 1.5)])
        for dx, dy in _interior_points(kind, q, dims, rng, 5):
            g = o.thickness_param_grad(kind, q, dims, dx, dy)
            par = np.concatenate([dims, q])
            fd = np.zeros(7)
            kink = False
            for p in range(7):
                up, dn_ = par.copy(), par.copy()
                up[p] += h; dn_[p] -= h
                tp, tm = o.thickness(kind, up[3:], up[:3], dx, dy), o.thickness(kind, dn_[3:], dn_[:3], dx, dy)
                t0 = o.thickness(kind, q, dims, dx, dy)
                fd[p] = (tp - tm) / (2 * h)
                kink = kink or abs(tp - 2 * t0 + tm) > 1e-9              # a face change inside the stencil: skip the point
            if kink:
                continue
            assert np.allclose(g, fd, rtol=2e-6, atol=2e-7), (kind, g, fd)
            checked += 1
    assert checked > 200


def test_B9_shape_gradient_closed_forms():
    # sphere a = b = c = R: t = 2 sqrt(R^2 - r^2); growing all three semi-axes together gives dt/dR = 2 R / sqrt(R^2 - r^2)
    R, dx, dy = 2.0, 0.7, -0.4
    g = o.thickness_param_grad(0, [1, 0, 0, 0], [R, R, R], dx, dy)
    assert abs(g[:3].sum() - 2 * R / np.sqrt(R * R - dx * dx - dy * dy)) < 1e-12
    # axis-aligned ellipsoid t = 2 c sqrt(1 - (dx/a)^2 - (dy/b)^2)
    a, b, c = 2.0, 1.5, 0.8
    w = 1 - (dx / a) ** 2 - (dy / b) ** 2
    g = o.thickness_param_grad(0, [1, 0, 0, 0], [a, b, c], dx, dy)
    assert np.allclose(g[:3], [2 * c * dx * dx / a ** 3 / np.sqrt(w), 2 * c * dy * dy / b ** 3 / np.sqrt(w), 2 * np.sqrt(w)], atol=1e-12)
    # a sphere does not care about its rotation
    q = np.array([0.3, -0.5, 0.4, 0.7]); q /= np.linalg.norm(q)
    g = o.thickness_param_grad(0, q, [R, R, R], dx, dy)
    tangent = g[3:] - (g[3:] @ q) * q                               # (the radial component rescales R(q): not a rotation)
    assert np.abs(tangent).max() < 1e-12
    # prism, identity rotation (P5): t = L + 2 hc (1 - m / (s/2)), m = max(|dx|, |dy|)
    s, L, hc = 2.0, 3.0, 0.9
    m = 0.61
    g = o.thickness_param_grad(1, [1, 0, 0, 0], [s, L, hc], m, 0.2)
    assert np.allclose(g[:3], [4 * hc * m / s ** 2, 1.0, 2 * (1 - m / (s / 2))], atol=1e-12)


def test_B10_backward_params_sums_the_pixel_gradients_and_matches_the_differenced_forward_model():
    sc = make_config(4, n_override=24)
    for k in ("cx", "cy"):
        sc.cols[k][:] = (sc.cols[k] / 16.0).astype(np.float32)
    sc = replace(sc, H=128, W=128)
    rng = np.random.default_rng(5)
    G = rng.standard_normal((1, 128, 128)).astype(np.float32)
    g = o.backward_params(sc, G)
    assert np.array_equal(g, o.backward_params(sc, G, mode="full"))
    # (a) the sum itself: dn * sum_px G * dt/dtheta with the pinned per-pixel gradient (B8, B9), written as a plain loop
    for n in (2, 7):
        c = sc.cols
        q = [float(c[k][n]) for k in ("qw", "qx", "qy", "qz")]; d = [float(c[k][n]) for k in ("d0", "d1", "d2")]
        acc = np.zeros(7)
        for i in range(128):
            for j in range(128):
                dx, dy = (j + 0.5) * sc.pitch_um - float(c["cx"][n]), (i + 0.5) * sc.pitch_um - float(c["cy"][n])
                if dx * dx + dy * dy < 200.0:
                    acc += float(G[0, i, j]) * o.thickness_param_grad(int(c["kind"][n]), q, d, dx, dy)
        assert np.allclose(g[n], (float(c["n_p"][n]) - sc.n_medium) * acc, rtol=1e-10, atol=1e-12)
    # (b) against the forward model differenced in the parameter, for the PRISMS (piecewise linear thickness) with a smooth
    # upstream gradient.  (For ellipsoids dt/dtheta grows like 1 / sqrt(w) towards the outline, the sum
    # over pixel centres is dominated by the outline pixels and the pixel-sampled loss has sqrt-type kinks: its difference
    # quotient scatters by up to 20 % around the almost-everywhere derivative; B8, B9 and (a) pin that case.)
    jj, ii = np.meshgrid(np.arange(128), np.arange(128))
    Gs = (np.cos(0.05 * jj + 0.3) * np.sin(0.04 * ii + 1.0)).astype(np.float32)[None]
    gs = o.backward_params(sc, Gs)
    names = ("d0", "d1", "d2", "qw", "qx", "qy", "qz")
    h = 2.0 ** -11                                                  # exactly representable steps on the float32 scene
    dev = []
    for n in np.flatnonzero(sc.cols["kind"] == 1):
        for p, name in enumerate(names):
            vals = []
            for sgn in (+1, -1):
                cols = {k: v.copy() for k, v in sc.cols.items()}
                cols[name][n] = np.float32(cols[name][n] + sgn * h)
                step = float(cols[name][n]) - float(sc.cols[name][n])
                vals.append((float((Gs[0].astype(np.float64) * o.render_opd(replace(sc, cols=cols))[0]).sum()), step))
            fd = (vals[0][0] - vals[1][0]) / (vals[0][1] - vals[1][1])
            dev.append(abs(gs[n, p] - fd) / max(abs(fd), np.abs(gs[n]).max()))
    dev = np.array(dev)
    # most of the 84 (prism, parameter) pairs agree to 1e-4; where a steep face sweeps over pixel centres within the step the
    # difference quotient itself is off by up to a few per cent
    assert len(dev) >= 70 and np.median(dev) < 1e-3 and np.percentile(dev, 90) < 1e-2 and dev.max() < 5e-2, \
        (np.median(dev), np.percentile(dev, 90), dev.max())


def test_B11_spectral_loss_and_its_gradient():
    rng = np.random.default_rng(3)
    I = 1.0 + 0.2 * rng.standard_normal((12, 10))
    T = 1.0 + 0.2 * rng.standard_normal((12, 10))
    eps = 1e-3
    assert o.spectral_loss(T, T, eps) == 0.0
    assert abs(o.spectral_loss(I, np.roll(T, (3, -2), (0, 1)), eps) - o.spectral_loss(I, T, eps)) < 1e-9   # |F| ignores circular shifts
    # eps -> 0: scaling the image shifts every log|F| by log c: loss = n_bins log(c)^2 against itself
    assert abs(o.spectral_loss(3.0 * T, T, 1e-300) - T.size * np.log(3.0) ** 2) < 1e-9
    # brute-force DFT instead of the library FFT
    ky, kx = np.meshgrid(np.arange(12), np.arange(10), indexing="ij")
    def dft(A):
        out = np.zeros((12, 10), complex)
        for y in range(12):
            for x in range(10):
                out += A[y, x] * np.exp(-2j * np.pi * (ky * y / 12 + kx * x / 10))
        return out
    brute = ((np.log(np.abs(dft(I)) + eps) - np.log(np.abs(dft(T)) + eps)) ** 2).sum()
    assert abs(brute - o.spectral_loss(I, T, eps)) < 1e-9
    # gradient against central differences of the loss, pixel by pixel
    g = o.spectral_loss_grad(I, T, eps)
    h = 1e-6
    for (y, x) in ((0, 0), (3, 7), (11, 9), (6, 2)):
        up, dn_ = I.copy(), I.copy()
        up[y, x] += h; dn_[y, x] -= h
        fd = (o.spectral_loss(up, T, eps) - o.spectral_loss(dn_, T, eps)) / (2 * h)
        assert abs(g[y, x] - fd) < 1e-5 * max(1.0, abs(fd))
