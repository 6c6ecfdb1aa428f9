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
