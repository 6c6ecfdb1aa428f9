"""Pins for the oracle's defocus factor (Eq. 3) and DIC image (Eq. 5), SURVEY 8(f) NEXT-1.

Nothing here re-types the oracle's formulae on arrays: each test compares with a scalar closed form, a physical
law with a textbook solution (Gaussian beam, focusing wave), an invariant, or brute-force DFT sums written as loops.
"""
import cmath
import math

import numpy as np

from oracle import oracle as o
from workloads import make_config

P_UM, LAM, N_M = 0.1, 0.55, 1.33


# ---- defocus -------------------------------------------------------------------------------------------------------
def test_D1_zero_defocus_is_the_identity():
    assert np.all(o.defocus_factor(32, 48, P_UM, LAM, N_M, 0.0) == 1.0)
    P = o.pupil_function(32, 48, 0.4, P_UM, LAM, N_M, 0.0)
    assert np.array_equal(P, o.pupil_mask(32, 48, 0.4, P_UM, LAM).astype(np.complex128))
    sc = make_config(1)
    U = o.render_field(sc)
    I0 = o.render_intensity(sc, U=U)
    from dataclasses import replace
    assert np.array_equal(o.render_intensity(replace(sc, defocus_um=0.0), U=U), I0)
    assert not np.allclose(o.render_intensity(replace(sc, defocus_um=3.0), U=U), I0, atol=1e-3)


def test_D2_plane_wave_on_a_bin_gets_the_scalar_phase():
    """U = exp(2 pi i (mx j / W + my i / H)) is the single FFT bin (my, mx): the image is U times
    exp(2 pi i dz sqrt((n/lambda)^2 - (mx/(W p))^2 - (my/(H p))^2)); intensity stays 1."""
    H, W, dz = 40, 64, 7.3
    jj, ii = np.meshgrid(np.arange(W), np.arange(H))
    for mx, my in ((0, 0), (5, 0), (0, -7), (-9, 4), (9, 5)):
        U = np.exp(2j * np.pi * (mx * jj / W + my * ii / H))
        V = o.coherent_image(U, o.defocus_factor(H, W, P_UM, LAM, N_M, dz))
        rad = (N_M / LAM) ** 2 - (mx / (W * P_UM)) ** 2 - (my / (H * P_UM)) ** 2
        assert rad > 0
        want = cmath.exp(2j * math.pi * dz * math.sqrt(rad))
        assert np.allclose(V / U, want, atol=1e-11)
    # an evanescent bin is removed: (n/lambda) = 2.418 cycles/um < 16 / (40 * 0.1) = 4 cycles/um
    U = np.exp(2j * np.pi * (16 * ii / H))
    assert np.abs(o.coherent_image(U, o.defocus_factor(H, W, P_UM, LAM, N_M, dz))).max() < 1e-12


def test_D3_semigroup_conjugate_and_unit_modulus():
    H, W = 48, 32
    a, b = o.defocus_factor(H, W, P_UM, LAM, N_M, 2.5), o.defocus_factor(H, W, P_UM, LAM, N_M, -6.0)
    c = o.defocus_factor(H, W, P_UM, LAM, N_M, -3.5)
    assert np.allclose(a * b, c, atol=1e-12)
    assert np.allclose(o.defocus_factor(H, W, P_UM, LAM, N_M, -2.5), np.conj(a), atol=1e-15)
    mod = np.abs(a)
    assert np.all((np.abs(mod - 1.0) < 1e-15) | (mod == 0.0))
    # number of propagating bins = lattice points inside the ellipse (mx/(W p))^2 + (my/(H p))^2 <= (n/lambda)^2
    mx = np.fft.fftfreq(W, 1.0 / W)[None, :] / (W * P_UM)
    my = np.fft.fftfreq(H, 1.0 / H)[:, None] / (H * P_UM)
    assert int((mod > 0).sum()) == int(((mx ** 2 + my ** 2) <= (N_M / LAM) ** 2).sum())


def _gauss(H, W, w0, curvature_R=None):
    x = (np.arange(W) - W // 2) * P_UM
    y = (np.arange(H) - H // 2) * P_UM
    X, Y = np.meshgrid(x, y)
    r2 = X * X + Y * Y
    U = np.exp(-r2 / (w0 * w0)).astype(np.complex128)
    if curvature_R is not None:                      # converging towards a focus at distance R: phase -k r^2 / (2 R)
        U = U * np.exp(-1j * (2 * np.pi * N_M / LAM) * r2 / (2.0 * curvature_R))
    return U, X, Y


def test_D4_gaussian_beam_spreads_as_the_textbook_says():
    """A Gaussian beam of waist w0 in a medium of index n has w(z) = w0 sqrt(1 + (z / zR)^2), zR = pi w0^2 n / lambda
    (Siegman, Lasers, ch. 17).  Pins k0 = 2 pi n_medium / lambda and the frequency grid m / (W p)."""
    H = W = 512
    w0, dz = 2.5, 40.0
    U, X, Y = _gauss(H, W, w0)
    V = o.coherent_image(U, o.defocus_factor(H, W, P_UM, LAM, N_M, dz))
    I = np.abs(V) ** 2
    w_meas = 2.0 * math.sqrt(float((I * X * X).sum() / I.sum()))          # <x^2> = w^2 / 4 for exp(-2 r^2 / w^2)
    zR = math.pi * w0 * w0 * N_M / LAM
    w_want = w0 * math.sqrt(1.0 + (dz / zR) ** 2)
    assert abs(w_meas - w_want) < 5e-3 * w_want
    # with the vacuum wavenumber instead (k0 = 2 pi / lambda) the beam would be 10 % wider: the pin can tell
    w_vac = w0 * math.sqrt(1.0 + (dz / (math.pi * w0 * w0 / LAM)) ** 2)
    assert abs(w_vac - w_want) > 0.08 * w_want
    assert abs(I.sum() - (np.abs(U) ** 2).sum()) < 1e-9 * I.sum()         # propagation is unitary


def test_D5_sign_a_converging_wave_focuses_at_positive_dz():
    """With the phase sign +i of Eq. 2 (A12) a forward wave is exp(+i k z): exp(-i k r^2 / (2R)) converges to a focus a
    distance R downstream.  Its peak intensity must grow for dz = +R and shrink for dz = -R."""
    H = W = 256
    R = 30.0
    U, _, _ = _gauss(H, W, 4.0, curvature_R=R)
    peak0 = (np.abs(U) ** 2).max()
    up = (np.abs(o.coherent_image(U, o.defocus_factor(H, W, P_UM, LAM, N_M, +R))) ** 2).max()
    dn = (np.abs(o.coherent_image(U, o.defocus_factor(H, W, P_UM, LAM, N_M, -R))) ** 2).max()
    assert up > 10.0 * peak0 and dn < 0.5 * peak0      # focal spot lambda R / (pi n w0) = 0.99 um: (4 / 0.99)^2 = 16


# ---- DIC -----------------------------------------------------------------------------------------------------------
def _n_pass(P):
    return float((np.abs(P) ** 2).sum())


def test_C1_zero_shear_gives_a_flat_image_of_known_level():
    """ds = 0: U e^{i theta} - U e^{-i theta} = 2 i sin(theta) U, |U| = 1, so D = 4 sin^2(theta) everywhere and the
    convolution with |h|^2 multiplies by sum |h|^2 = sum |P|^2 / (H W) (Parseval)."""
    sc = make_config(1)
    U = o.render_field(sc)[0]
    H, W = U.shape
    for dz in (0.0, 2.0):
        P = o.pupil_function(H, W, 0.4, P_UM, LAM, N_M, dz)
        I = o.dic_image(U, P, (0, 0), 0.7)
        assert np.allclose(I, 4.0 * math.sin(0.7) ** 2 * _n_pass(P) / (H * W), rtol=0, atol=1e-13)


def test_C2_uniform_phase_gradient_reads_as_sin2_of_half_the_phase_step_plus_bias():
    """U = exp(2 pi i m j / W): U(r + ds) = U e^{i phi}, U(r - ds) = U e^{-i phi}, phi = 2 pi m sx / W, hence
    D = 4 sin^2(phi + theta): DIC measures the phase gradient along the shear, offset by the bias."""
    H, W, m = 32, 64, 3
    jj, ii = np.meshgrid(np.arange(W), np.arange(H))
    U = np.exp(2j * np.pi * m * jj / W)
    P = o.pupil_function(H, W, 0.5, P_UM, LAM, N_M)
    for sx, sy, th in ((2, 0, 0.3), (-1, 5, -0.9), (0, 3, 0.4)):
        phi = 2 * math.pi * m * sx / W
        want = 4.0 * math.sin(phi + th) ** 2 * _n_pass(P) / (H * W)
        assert np.allclose(o.dic_image(U, P, (sx, sy), th), want, rtol=0, atol=1e-13)
    # the same along y
    U = np.exp(2j * np.pi * 2 * ii / H)
    want = 4.0 * math.sin(2 * math.pi * 2 * 3 / H + 0.25) ** 2 * _n_pass(P) / (H * W)
    assert np.allclose(o.dic_image(U, P, (4, 3), 0.25), want, rtol=0, atol=1e-13)


def test_C3_brute_force_sums_on_a_tiny_frame():
    """Eq. 5 by definition with explicit loops: h[r] = (1/HW) sum_k P[k] e^{+2 pi i k.r / N} (inverse DFT as a sum),
    I[r] = sum_r' D[r'] |h[r - r']|^2 with indices taken modulo the frame (circular, A22)."""
    rng = np.random.default_rng(5)
    H, W = 6, 8
    U = np.exp(2j * np.pi * rng.random((H, W)))
    P = o.pupil_function(H, W, 1.0, 0.3, LAM, N_M, dz=1.7)              # coarse pitch: NA p / lambda = 0.545
    assert 20 < int((np.abs(P) > 0).sum()) < H * W
    sx, sy, th = 1, -2, 0.6
    h = np.zeros((H, W), dtype=np.complex128)
    for i in range(H):
        for j in range(W):
            acc = 0.0
            for ky in range(H):
                for kx in range(W):
                    acc += P[ky, kx] * cmath.exp(2j * math.pi * (ky * i / H + kx * j / W))
            h[i, j] = acc / (H * W)
    D = np.zeros((H, W))
    for i in range(H):
        for j in range(W):
            d = U[(i + sy) % H, (j + sx) % W] * cmath.exp(1j * th) - U[(i - sy) % H, (j - sx) % W] * cmath.exp(-1j * th)
            D[i, j] = abs(d) ** 2
    want = np.zeros((H, W))
    for i in range(H):
        for j in range(W):
            acc = 0.0
            for i2 in range(H):
                for j2 in range(W):
                    acc += D[i2, j2] * abs(h[(i - i2) % H, (j - j2) % W]) ** 2
            want[i, j] = acc
    assert np.allclose(o.dic_image(U, P, (sx, sy), th), want, rtol=0, atol=1e-13)


def test_C4_symmetries_and_energy():
    sc = make_config(1)
    U = o.render_field(sc)[0]
    H, W = U.shape
    P = o.pupil_function(H, W, 0.4, P_UM, LAM, N_M, 1.0)
    I = o.dic_image(U, P, (3, 1), 0.5)
    assert np.allclose(o.dic_image(U, P, (-3, -1), -0.5), I, atol=1e-13)              # swapping the two copies
    assert np.allclose(o.dic_image(U, P, (3, 1), 0.5 + math.pi), I, atol=1e-13)       # bias is defined modulo pi
    assert I.min() > -1e-13
    # energy: sum I = sum D * sum |h|^2
    Up, Um = np.roll(U, (-1, -3), (0, 1)), np.roll(U, (1, 3), (0, 1))
    D = np.abs(Up * cmath.exp(0.5j) - Um * cmath.exp(-0.5j)) ** 2
    assert abs(I.sum() - D.sum() * _n_pass(P) / (H * W)) < 1e-9 * I.sum()
    # an all-pass pupil has h = delta: the image is D itself
    assert np.allclose(o.dic_image(U, None, (3, 1), 0.5), D, atol=1e-12)
    # a particle-free frame with no bias is dark; the spheres of config 1 are not
    assert np.abs(o.dic_image(np.ones((H, W), complex), P, (3, 1), 0.0)).max() < 1e-15
    assert o.dic_image(U, P, (3, 1), 0.0).max() > 1e-3


def test_render_dic_wires_scene_optics_and_noise():
    from dataclasses import replace
    sc = replace(make_config(1), defocus_um=1.5, read_noise_sigma=0.02)
    U = o.render_field(sc)
    I = o.render_dic(sc, (2, 0), 0.4, U=U)
    P = o.pupil_function(sc.H, sc.W, float(sc.NA[0]), sc.pitch_um, float(sc.lambda_um[0]), sc.n_medium, 1.5)
    want = o.dic_image(U[0], P, (2, 0), 0.4) + 0.02 * o.read_noise(sc.seed, 0, sc.H, sc.W)
    assert np.array_equal(I[0], want)
