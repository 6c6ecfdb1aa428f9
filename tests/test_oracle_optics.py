"""Pins for the oracle's frame-level pieces (pins P8-P12, P14-P16):
OPD accumulation, exit wave, pupil, coherent intensity, Philox read noise.

Nothing here re-types the oracle's formulae or re-calls its library routine as the expected value: expected
values come from invariants, special cases, a brute-force O(n^4) DFT, and cuRAND's host Philox generator.
"""
import ctypes
import math
import os

import numpy as np
import pytest

from oracle import oracle as o
from workloads import make_config, make_scene, subset


def small_mixed_scene(n=24, H=96, W=80, seed=5, **kw):
    rng = np.random.default_rng(seed)
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    kind = (np.arange(n) % 2).astype(np.uint8)
    s = rng.uniform(0.8, 2.5, n)
    d = np.where(kind[:, None] == 1, np.stack([s, s * rng.uniform(1, 2.5, n), 0.5 * s], 1),
                 rng.uniform(0.5, 2.5, (n, 3)))
    cols = dict(cx=rng.uniform(-0.5, W * 0.1 + 0.5, n), cy=rng.uniform(-0.5, H * 0.1 + 0.5, n),
                qw=q[:, 0], qx=q[:, 1], qy=q[:, 2], qz=q[:, 3], d0=d[:, 0], d1=d[:, 1], d2=d[:, 2],
                n_p=rng.uniform(1.36, 1.5, n), kind=kind)
    return make_scene("small_mixed", H, W, cols, **kw)


# ----------------------------------------------------------------------------- P8, P14, P15
def test_P8_permutation_invariance_and_additivity():
    sc = small_mixed_scene()
    full = o.render_opd(sc, "full")[0]
    rng = np.random.default_rng(0)
    perm = rng.permutation(sc.N)
    np.testing.assert_allclose(o.render_opd(subset(sc, perm), "full")[0], full, atol=1e-12)
    a = o.render_opd(subset(sc, np.arange(0, sc.N, 2)), "full")[0]
    b = o.render_opd(subset(sc, np.arange(1, sc.N, 2)), "full")[0]
    np.testing.assert_allclose(a + b, full, atol=1e-12)
    # a single particle's frame is (n_p - n_m) * thickness at each pixel centre
    k = 3
    one = o.render_opd(subset(sc, [k]), "full")[0]
    i, j = np.unravel_index(np.argmax(one), one.shape)
    qd = [float(sc.cols[c][k]) for c in ("qw", "qx", "qy", "qz")]
    dm = [float(sc.cols[c][k]) for c in ("d0", "d1", "d2")]
    t = o.thickness(int(sc.kind[k]), qd, dm, (j + 0.5) * 0.1 - float(sc.cx[k]), (i + 0.5) * 0.1 - float(sc.cy[k]))
    assert one[i, j] == pytest.approx((float(sc.n_p[k]) - 1.33) * t, rel=1e-13)
    assert one[i, j] > 0


def test_P14_integer_pixel_translation_shifts_the_patch():
    rng = np.random.default_rng(3)
    H = W = 64
    for kind in (0, 1):
        q = rng.standard_normal(4); q /= np.linalg.norm(q)
        # centres on a dyadic grid so that cx + k * 0.1 (float32) keeps the same sub-pixel offset to ~1e-7 um
        base = dict(qw=[q[0]], qx=[q[1]], qy=[q[2]], qz=[q[3]], d0=[1.1], d1=[1.7], d2=[0.6], n_p=[1.45], kind=[kind])
        a = o.render_opd(make_scene("a", H, W, dict(cx=[2.03], cy=[2.51], **base)), "full")[0]
        b = o.render_opd(make_scene("b", H, W, dict(cx=[2.03 + 1.3], cy=[2.51 + 0.9], **base)), "full")[0]
        shifted = np.zeros_like(a)
        shifted[9:, 13:] = a[:-9, :-13]
        # float32 centres: 2.03f + 1.3 is not exactly (2.03 + 1.3)f; the residual sub-pixel shift is < 3e-7 um
        assert np.abs(b - shifted).max() < 2e-5          # silhouette pixels move by slope * 3e-7
        assert np.abs(b - shifted).mean() < 1e-7
        assert (shifted > 0).sum() > 200


def test_P15_bcircle_equals_full_bit_for_bit():
    sc = small_mixed_scene(n=40, H=128, W=112, seed=8)
    assert np.array_equal(o.render_opd(sc, "full"), o.render_opd(sc, "bcircle"))
    c1 = make_config(1)
    assert np.array_equal(o.render_opd(c1, "full"), o.render_opd(c1, "bcircle"))


def test_offcanvas_particles_are_clipped_not_wrapped():
    """PAPER.md:119 'strict boolean masking': a particle straddling the border contributes only inside."""
    H = W = 32
    base = dict(d0=[1.0], d1=[1.0], d2=[1.0], n_p=[1.43])
    inside = o.render_opd(make_scene("i", H, W, dict(cx=[0.2], cy=[1.6], **base)), "full")[0]
    assert inside[:, :12].max() > 0 and inside[:, 20:].max() == 0.0          # nothing wraps to the right edge
    far = o.render_opd(make_scene("f", H, W, dict(cx=[-5.0], cy=[40.0], **base)), "full")[0]
    assert far.max() == 0.0


def test_invalid_particles_are_skipped():
    H = W = 32
    cols = dict(cx=[1.6, 1.6, 1.6, 1.6], cy=[1.6, 1.6, 1.6, 1.6], d0=[1.0, -1.0, np.nan, 1.0], d1=[1.0, 1.0, 1.0, 0.0],
                d2=[1.0, 1.0, 1.0, 1.0], n_p=[1.43, 1.43, 1.43, 1.43])
    got = o.render_opd(make_scene("v", H, W, cols), "full")[0]
    ref = o.render_opd(make_scene("r", H, W, {k: v[:1] for k, v in cols.items()}), "full")[0]
    assert np.array_equal(got, ref)
    assert list(o.particle_valid(make_scene("v", H, W, cols).cols)) == [True, False, False, False]


# ----------------------------------------------------------------------------- P9, field
def test_P9_zero_particles_uniform_field_and_intensity():
    sc = make_scene("empty", 32, 48, dict(cx=[], cy=[], d0=[], d1=[], d2=[], n_p=[]))
    opd = o.render_opd(sc)
    assert opd.shape == (1, 32, 48) and not opd.any()
    U = o.render_field(sc, opd)
    assert np.array_equal(U, np.ones_like(U))
    I = o.render_intensity(sc, U)
    np.testing.assert_allclose(I, 1.0, atol=1e-13)
    # a pupil that passes DC only: I = |mean U|^2 everywhere
    sc2 = small_mixed_scene(n=10, H=32, W=32, NA=1e-4)
    U2 = o.render_field(sc2)[0]
    I2 = o.render_intensity(sc2, U2[None])[0]
    np.testing.assert_allclose(I2, abs(U2.mean()) ** 2, rtol=1e-12)


def test_field_phase_values_at_known_opd():
    """Eq. 2 with A == 1, sign +i: OPD = lambda/4 -> U = i; lambda/2 -> -1; the ramp adds 2 pi sin(theta)/lambda * x."""
    lam, p = 0.5, 0.1
    opd = np.array([[0.0, lam / 4, lam / 2, lam]])
    U = o.field(opd, lam, p)
    np.testing.assert_allclose(U[0], [1, 1j, -1, 1], atol=1e-15)
    th = math.asin(0.25)                                   # fx0 = 0.5 cycles/um: x = 0.05, 0.15 ... -> phase pi (j + 1/2)/10
    U = o.field(np.zeros((2, 8)), lam, p, tilt_x=th)
    want = np.exp(1j * math.pi * (np.arange(8) + 0.5) / 10)
    np.testing.assert_allclose(U[0], want, atol=1e-14)
    np.testing.assert_allclose(U[1], want, atol=1e-14)
    U = o.field(np.zeros((8, 2)), lam, p, tilt_y=th)
    np.testing.assert_allclose(U[:, 1], want, atol=1e-14)


# ----------------------------------------------------------------------------- pupil, P10-P12
def test_pupil_mask_against_float_definition_and_printed_thresholds():
    # DESIGN.md / SURVEY 8(c) A10 worked values: cfg 1 rho^2 = 346.64 -> 346, cfg 4 rho^2 = 58581.6 -> 58581
    assert o.pupil_threshold(256, 256, 0.4, 0.1, 0.55) // (256 * 256) == 346
    assert o.pupil_threshold(2048, 2048, 0.65, 0.1, 0.55) // (2048 * 2048) == 58581
    for (H, W, NA, lam) in [(64, 64, 0.4, 0.55), (48, 80, 0.65, 0.47), (33, 20, 0.8, 0.61)]:
        m = o.pupil_mask(H, W, NA, 0.1, lam)
        fx = np.fft.fftfreq(W, d=0.1)                     # cycles / um
        fy = np.fft.fftfreq(H, d=0.1)
        f2 = fx[None, :] ** 2 + fy[:, None] ** 2
        fc2 = (NA / lam) ** 2
        sure = np.abs(f2 - fc2) > 1e-9 * fc2
        assert np.array_equal(m[sure], (f2 <= fc2)[sure])
        assert m[0, 0] and m.sum() == pytest.approx(math.pi * fc2 * (H * 0.1) * (W * 0.1), rel=0.15)
        # symmetric under k -> -k
        assert np.array_equal(m, np.roll(m[::-1, ::-1], (1, 1), (0, 1)))


def _dft2_brute(U):
    H, W = U.shape
    Fy = np.exp(-2j * np.pi * np.outer(np.arange(H), np.arange(H)) / H)
    Fx = np.exp(-2j * np.pi * np.outer(np.arange(W), np.arange(W)) / W)
    out = np.zeros((H, W), dtype=np.complex128)
    for ky in range(H):
        for kx in range(W):
            out[ky, kx] = (Fy[ky][:, None] * Fx[kx][None, :] * U).sum()
    return out


def test_P12_coherent_image_against_brute_force_dft():
    sc = small_mixed_scene(n=6, H=12, W=16, seed=2, NA=0.5, tilt_x_rad=0.1)
    U = o.render_field(sc)[0]
    mask = o.pupil_mask(12, 16, 0.5, 0.1, 0.55)
    F = _dft2_brute(U) * mask
    V = np.conj(_dft2_brute(np.conj(F))) / (12 * 16)       # inverse DFT by conjugation
    np.testing.assert_allclose(o.coherent_image(U, mask), V, atol=1e-11)
    np.testing.assert_allclose(o.intensity(U, mask), np.abs(V) ** 2, atol=1e-11)
    np.testing.assert_allclose(o.coherent_image(U, None), U, atol=1e-13)    # all-pass returns U


def test_P11_parseval():
    sc = small_mixed_scene(n=20, H=64, W=64, seed=4, NA=0.5)
    U = o.render_field(sc)[0]
    I_all = o.render_intensity(sc, U[None], pupil_enabled=False)[0]
    np.testing.assert_allclose(I_all, 1.0, atol=1e-12)                     # |U| = 1 everywhere
    assert I_all.sum() == pytest.approx(64 * 64, rel=1e-13)
    mask = o.pupil_mask(64, 64, 0.5, 0.1, 0.55)
    I = o.intensity(U, mask)
    F = _dft2_brute(U[:8, :8])                                              # tiny brute-force Parseval too
    assert (np.abs(F) ** 2).sum() / 64 == pytest.approx((np.abs(U[:8, :8]) ** 2).sum(), rel=1e-12)
    Fm = np.fft.fft2(U) * mask
    assert I.sum() == pytest.approx((np.abs(Fm) ** 2).sum() / (64 * 64), rel=1e-12)
    assert I.sum() < 64 * 64                                                # a low-pass loses energy


def test_P10_ramp_on_an_fft_bin_is_a_pupil_shift():
    """Shift theorem: tilt with fx0 = m0 / (W p) == the un-tilted field seen through a pupil centred at -m0 bins
    (the paper's 'asymmetric Fourier pupil')."""
    H = W = 64
    lam, p, m0 = 0.55, 0.1, 5
    th = math.asin(m0 / (W * p) * lam)
    sc = small_mixed_scene(n=20, H=H, W=W, seed=6, NA=0.5)
    opd = o.render_opd(sc)[0]
    mask = o.pupil_mask(H, W, 0.5, p, lam)
    I_tilt = o.intensity(o.field(opd, lam, p, tilt_x=th), mask)
    U0 = o.field(opd, lam, p)
    V = np.fft.ifft2(np.fft.fft2(U0) * np.roll(mask, -m0, axis=1))
    np.testing.assert_allclose(I_tilt, np.abs(V) ** 2, atol=1e-10)
    assert np.abs(I_tilt - o.intensity(U0, mask)).max() > 1e-3             # and the tilt does change the image


# ----------------------------------------------------------------------------- P16 Philox / noise
def _curand_host_philox(seed, offset, n_quads):
    lib = ctypes.CDLL(os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "lib64", "libcurand.so"))
    gen = ctypes.c_void_p()
    assert lib.curandCreateGeneratorHost(ctypes.byref(gen), 161) == 0      # CURAND_RNG_PSEUDO_PHILOX4_32_10
    assert lib.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
    assert lib.curandSetGeneratorOffset(gen, ctypes.c_ulonglong(offset)) == 0
    out = np.zeros(4 * n_quads, dtype=np.uint32)
    assert lib.curandGenerate(gen, out.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(out.size)) == 0
    lib.curandDestroyGenerator(gen)
    return out.reshape(n_quads, 4)


def test_P16_philox_block_function_against_curand_host_generator():
    """cuRAND's host Philox4x32-10 generator (default ordering, probed on this image): output quadruple m of
    the stream is the Philox block for counter (0, 0, m, 0) under key (seed lo, seed hi); an offset of 4 k
    skips k quadruples.  After the first round every word of the state is generic, so rounds 2-10 exercise
    every data path of the round function (both multipliers, both key words, all four lanes); only the naming
    of the input words (which one carries the pixel index) is left to reading A13."""
    seed = 0x0123456789ABCDEF
    try:
        ref = _curand_host_philox(seed, 0, 6000)
    except OSError:
        pytest.skip("libcurand not found")
    key = (seed & 0xFFFFFFFF, seed >> 32)
    ctr = np.zeros((6000, 4), dtype=np.uint64); ctr[:, 2] = np.arange(6000)
    assert np.array_equal(o.philox4x32_10(ctr, key), ref)
    ref = _curand_host_philox(seed, 4 * 77, 8)
    ctr = np.zeros((8, 4), dtype=np.uint64); ctr[:, 2] = 77 + np.arange(8)
    assert np.array_equal(o.philox4x32_10(ctr, key), ref)
    for sd in (0, 42, 2 ** 64 - 1, 0xDEADBEEF00000001):
        ref = _curand_host_philox(sd, 0, 16)
        ctr = np.zeros((16, 4), dtype=np.uint64); ctr[:, 2] = np.arange(16)
        assert np.array_equal(o.philox4x32_10(ctr, (sd & 0xFFFFFFFF, sd >> 32)), ref)
    # the four input words are distinct inputs: moving the index to another word changes the block
    blocks = set()
    for w in range(4):
        c = np.zeros((1, 4), dtype=np.uint64); c[0, w] = 5
        blocks.add(tuple(o.philox4x32_10(c, key)[0]))
    assert len(blocks) == 4


def test_P16_read_noise_statistics_and_keying():
    z = o.read_noise(1234, 0, 512, 512).ravel()
    n = z.size
    assert abs(z.mean()) < 4 / math.sqrt(n)
    assert abs(z.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs((z ** 4).mean() - 3) < 0.1
    from scipy import stats
    assert stats.kstest(z, "norm").pvalue > 1e-3
    assert abs(np.corrcoef(z[:-1], z[1:])[0, 1]) < 4 / math.sqrt(n)
    # keyed on (seed, frame, pixel): frames and seeds give different, reproducible streams
    assert np.array_equal(o.read_noise(1234, 0, 16, 16), o.read_noise(1234, 0, 16, 16))
    assert not np.array_equal(o.read_noise(1234, 0, 16, 16), o.read_noise(1234, 1, 16, 16))
    assert not np.array_equal(o.read_noise(1234, 0, 16, 16), o.read_noise(1235, 0, 16, 16))
    # pixel index is i W + j: a wider frame's first row starts with the narrower frame's first row
    assert np.array_equal(o.read_noise(7, 2, 4, 8).ravel()[:16], o.read_noise(7, 2, 2, 8).ravel())


def test_intensity_with_noise_is_additive():
    sc = small_mixed_scene(n=8, H=32, W=32, seed=9, NA=0.5, read_noise_sigma=0.01)
    sc0 = small_mixed_scene(n=8, H=32, W=32, seed=9, NA=0.5)
    sc.seed = sc0.seed = 99
    d = o.render_intensity(sc)[0] - o.render_intensity(sc0)[0]
    np.testing.assert_allclose(d, 0.01 * o.read_noise(99, 0, 32, 32), atol=1e-14)
