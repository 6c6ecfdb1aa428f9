"""Pins of the oracle's brightfield amplitude, Eq. 4 (reading A27): the Fresnel
transmittance against the textbook sine / tangent forms and its closed-form special cases, the amplitude map against
the cases where height, gradient and curvature are known exactly."""
import numpy as np

from oracle import oracle as o
from workloads import make_config

P = 0.1


def test_F1_fresnel_special_cases():
    n1, n2 = 1.33, 1.47
    assert abs(o.fresnel_transmittance(1.0, n1, n2) - 4 * n1 * n2 / (n1 + n2) ** 2) < 1e-15      # normal incidence
    assert np.all(o.fresnel_transmittance(np.linspace(0, 1, 11), 1.4, 1.4) == 1.0)               # no interface
    assert abs(o.fresnel_transmittance(0.0, n1, n2)) < 1e-15                                     # grazing: all reflected
    # Brewster's angle tan(theta_B) = n2 / n1: R_p = 0, so T = 1 - R_s / 2 with R_s = cos^2(2 theta_B)
    tb = np.arctan(n2 / n1)
    assert abs(o.fresnel_transmittance(np.cos(tb), n1, n2) - (1.0 - 0.5 * np.cos(2 * tb) ** 2)) < 1e-14
    # total internal reflection beyond the critical angle (dense -> thin only)
    tc = np.arcsin(n1 / n2)
    assert o.fresnel_transmittance(np.cos(tc + 1e-6), n2, n1) == 0.0 and o.fresnel_transmittance(np.cos(tc - 1e-3), n2, n1) > 0.0


def test_F2_fresnel_equals_the_sine_tangent_forms_and_is_reciprocal():
    n1, n2 = 1.33, 1.52
    ti = np.linspace(0.01, 1.55, 400)
    tt = np.arcsin(n1 / n2 * np.sin(ti))
    rs = np.sin(ti - tt) ** 2 / np.sin(ti + tt) ** 2                                             # textbook alternative forms
    rp = np.tan(ti - tt) ** 2 / np.tan(ti + tt) ** 2
    T = o.fresnel_transmittance(np.cos(ti), n1, n2)
    assert np.allclose(T, 1.0 - 0.5 * (rs + rp), atol=1e-12)
    assert np.all(np.diff(T) < 0)                                                                # falls monotonically with the angle
    assert np.allclose(T, o.fresnel_transmittance(np.cos(tt), n2, n1), atol=1e-12)               # the reverse path transmits the same


def test_A1_flat_tilted_and_curved_height_maps():
    n1, n2, dmu, gain = 1.33, 1.45, 0.08, 0.3
    T0 = 4 * n1 * n2 / (n1 + n2) ** 2
    z = np.zeros((20, 30))
    assert np.allclose(o.brightfield_amplitude(z, P, n1, n2, dmu, gain), T0, atol=1e-15)         # h = 0: A = T_F(0) + 0
    assert np.allclose(o.brightfield_amplitude(z + 2.5, P, n1, n2, dmu, gain), T0 * np.exp(-2.5 * dmu), atol=1e-15)   # slab: C = 0
    jj, ii = np.meshgrid((np.arange(30) + 0.5) * P, (np.arange(20) + 0.5) * P)
    a, b = 0.7, -1.2                                                                             # a plane: gradient exact, no curvature
    h = 1.0 + a * jj + b * ii
    want = o.fresnel_transmittance(1.0 / np.sqrt(1 + a * a + b * b), n1, n2) * np.exp(-h * dmu)
    got = o.brightfield_amplitude(h, P, n1, n2, dmu, gain)
    assert np.allclose(got[1:-1, 1:-1], want[1:-1, 1:-1], atol=1e-12)
    # a paraboloid cap h = c - k r^2 (convex): laplacian -4k, so the caustic term ADDS 4 k gain (light concentrated)
    k = 0.35
    x0, y0 = 1.5, 1.0
    h = 3.0 - k * ((jj - x0) ** 2 + (ii - y0) ** 2)
    got = o.brightfield_amplitude(h, P, n1, n2, 0.0, gain)[1:-1, 1:-1]
    cos_i = 1.0 / np.sqrt(1 + (2 * k) ** 2 * ((jj - x0) ** 2 + (ii - y0) ** 2))
    assert np.allclose(got, (o.fresnel_transmittance(cos_i, n1, n2) + 4 * k * gain)[1:-1, 1:-1], atol=1e-9)


def test_A2_neutral_parameters_give_the_plain_coherent_image():
    sc = make_config(2, n_override=40)
    sc.cols["cx"][:] = sc.cols["cx"] / 8; sc.cols["cy"][:] = sc.cols["cy"] / 8
    from dataclasses import replace
    sc = replace(sc, H=128, W=128)
    plain = o.render_intensity(sc)
    assert np.allclose(o.render_brightfield(sc, sc.n_medium, 0.0, 0.0), plain, atol=1e-13)       # T_F = 1, no absorption, no caustic
    dark = o.render_brightfield(sc, 1.45, 0.2, 0.0)
    assert dark.mean() < plain.mean()                                                            # absorption and reflection only remove light
    lens = o.render_brightfield(sc, sc.n_medium, 0.0, 0.05)
    h = o.render_height(sc)[0]
    assert lens[0][h > 2.0].mean() > plain[0][h > 2.0].mean()                                    # convex bodies: hotspots
