"""Pins for the oracle's height map and its finite-difference gradient / Laplacian (reading A25)."""
import numpy as np
from scipy import ndimage

from oracle import oracle as o
from workloads import make_config, make_scene, subset

P = 0.1


def test_H1_height_is_the_thickness_sum():
    # one sphere: h = 2 sqrt(R^2 - r^2); a scene: h = sum of the single-particle heights = OPD with unit index contrast
    sc = make_scene("h", 64, 64, dict(cx=[3.23], cy=[3.11], d0=[1.7], d1=[1.7], d2=[1.7], n_p=[1.4]))
    h = o.render_height(sc)[0]
    f = lambda v: float(np.float32(v))
    x = (np.arange(64) + 0.5) * P
    X, Y = np.meshgrid(x, x)
    r2 = (X - f(3.23)) ** 2 + (Y - f(3.11)) ** 2
    want = np.where(r2 < f(1.7) ** 2, 2 * np.sqrt(np.maximum(f(1.7) ** 2 - r2, 0)), 0.0)
    assert np.allclose(h, want, atol=1e-12)
    sc = make_config(4, n_override=30)
    tot = o.render_height(sc)[0]
    parts = sum(o.render_height(subset(sc, [n]))[0] for n in range(sc.N))
    assert np.allclose(tot, parts, atol=1e-11)
    # the same pixels as the OPD frame are non-zero, and h * dn = OPD for a single particle
    one = subset(sc, [3])
    dn = float(one.cols["n_p"][0]) - one.n_medium
    assert np.allclose(o.render_height(one)[0] * dn, o.render_opd(one)[0], atol=1e-12)


def test_H2_gradient_is_numpy_gradient_and_exact_on_planes():
    rng = np.random.default_rng(1)
    h = rng.standard_normal((37, 53))
    gx, gy = o.height_gradient(h, P)
    ny, nx = np.gradient(h, P)                                   # library routine: central inside, one-sided at the edges
    assert np.allclose(gx, nx, atol=1e-12) and np.allclose(gy, ny, atol=1e-12)
    jj, ii = np.meshgrid(np.arange(53) * P, np.arange(37) * P)
    gx, gy = o.height_gradient(3.0 + 0.7 * jj - 1.9 * ii, P)     # a plane: exact everywhere, borders included
    assert np.allclose(gx, 0.7, atol=1e-12) and np.allclose(gy, -1.9, atol=1e-12)
    # a sphere's height 2 sqrt(R^2 - r^2) has gradient -2 d / sqrt(R^2 - r^2): central differences agree to O(p^2) inside
    sc = make_scene("h", 96, 96, dict(cx=[4.8], cy=[4.8], d0=[4.0], d1=[4.0], d2=[4.0], n_p=[1.4]))
    hh = o.render_height(sc)[0]
    gx, gy = o.height_gradient(hh, P)
    x = (np.arange(96) + 0.5) * P
    X, Y = np.meshgrid(x, x)
    dx, dy = X - float(np.float32(4.8)), Y - float(np.float32(4.8))
    r2 = dx * dx + dy * dy
    core = r2 < 2.0 ** 2
    s = np.sqrt(16.0 - r2[core])
    assert np.allclose(gx[core], -2 * dx[core] / s, atol=2e-3) and np.allclose(gy[core], -2 * dy[core] / s, atol=2e-3)


def test_H3_laplacian_is_the_library_five_point_stencil_and_exact_on_quadratics():
    rng = np.random.default_rng(2)
    h = rng.standard_normal((29, 41))
    lap = o.height_laplacian(h, P)
    assert np.allclose(lap, ndimage.laplace(h, mode="nearest") / (P * P), atol=1e-9)
    jj, ii = np.meshgrid(np.arange(41) * P, np.arange(29) * P)
    q = 1.5 * jj ** 2 - 0.4 * ii ** 2 + 0.3 * jj * ii + 2.0 * jj
    assert np.allclose(o.height_laplacian(q, P)[1:-1, 1:-1], 2 * 1.5 - 2 * 0.4, atol=1e-9)
