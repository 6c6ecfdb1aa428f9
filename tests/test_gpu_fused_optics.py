"""GPU parity of the fused, pruned library stage (L1-L3 on power-of-two frames: row FFT -> [column FFT, pupil, inverse column
FFT] of the columns the pupil keeps -> inverse row FFT + sensor; csrc/optics.cu) against the oracle's numpy.fft pipeline, on
the shapes the five workloads do not cover: non-square frames, the smallest and the largest row, every first-stage radix
(2, 4, 8), an all-pass pupil, per-frame pupils of different width, defocus, noise, and frames that keep the cuFFT path."""
from dataclasses import replace

import numpy as np
import pytest

from workloads import make_scene

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def og():
    import torch
    assert torch.cuda.is_available()
    import paper_2606_21381_b200 as m
    m.lib()
    return m


@pytest.fixture(scope="module")
def o():
    from oracle import oracle
    return oracle


def _scene(H, W, seed, B=1, **kw):
    rng = np.random.default_rng(seed)
    n = 30 * B
    kind = (rng.uniform(size=n) < 0.5).astype(np.uint8)
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    cols = dict(cx=rng.uniform(0.0, W * 0.1, n), cy=rng.uniform(0.0, H * 0.1, n), qw=q[:, 0], qx=q[:, 1], qy=q[:, 2],
                qz=q[:, 3], d0=rng.uniform(0.4, 2.0, n), d1=rng.uniform(0.4, 2.5, n), d2=rng.uniform(0.3, 1.5, n),
                n_p=rng.uniform(1.36, 1.5, n), kind=kind)
    return make_scene(f"fo{H}x{W}", H, W, cols, frame_start=[30 * b for b in range(B + 1)], **kw)


def _check(og, o, sc, pupil_enabled=True):
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc, pupil_enabled=pupil_enabled)
    I = ctx.render_intensity(P, opt).clone()
    I2 = ctx.render_intensity(P, opt)
    assert bool((I == I2).all())                                 # no atomics anywhere in the stage: same bits
    assert ctx.check_guards() == 0
    ctx.close()
    I = I.cpu().numpy().astype(np.float64)
    ref = o.render_intensity(sc, pupil_enabled=pupil_enabled)
    tol = 1e-4 * ref.mean()
    err = np.abs(I - ref).max()
    assert err <= tol, f"{sc.H}x{sc.W}: intensity max abs err {err:.3e} > {tol:.3e}"
    return I


# lg(n) mod 3 picks the first-stage radix: 64 -> 8, 128 -> 2, 256 -> 4, 512 -> 8, 1024 -> 2, 4096 -> 8
@pytest.mark.parametrize("H,W", [(64, 64), (128, 512), (512, 128), (256, 1024), (64, 4096), (4096, 64)])
def test_fused_stage_on_power_of_two_shapes(og, o, H, W):
    _check(og, o, _scene(H, W, seed=H + W, NA=0.55, lam=0.52, tilt_x_rad=0.03))


def test_fused_stage_all_pass_and_narrow_pupils(og, o):
    sc = _scene(128, 256, seed=5, NA=0.5)
    a = _check(og, o, sc, pupil_enabled=False)                   # every column kept
    assert np.abs(a - 1.0).max() < 1e-4                          # |U| = 1 without a pupil
    _check(og, o, replace(sc, NA=np.array([1.0e-3])))            # only the zero-frequency bin passes
    _check(og, o, replace(sc, NA=np.array([5.0])))               # wider than the grid: all-pass through the threshold


def test_fused_stage_batch_with_different_pupils_defocus_and_noise(og, o):
    sc = _scene(256, 128, seed=9, B=3, NA=[0.2, 0.9, 0.45], lam=[0.45, 0.65, 0.55], read_noise_sigma=0.01)
    _check(og, o, sc)
    _check(og, o, replace(sc, defocus_um=2.5))
    # Poisson counts are integers decided by the float32 image: the oracle's sensor is applied to the GPU's own noise-free
    # image (as tests/test_gpu_shot_noise.py does), which the line above has tied to the oracle's
    noisy = replace(sc, defocus_um=2.5, shot_noise_photons=500.0)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P = og.Particles.from_scene(sc)
    I0 = ctx.render_intensity(P, og.optics_from_scene(replace(noisy, shot_noise_photons=0.0, read_noise_sigma=0.0))).cpu().numpy()
    I1 = ctx.render_intensity(P, og.optics_from_scene(noisy)).cpu().numpy().astype(np.float64)
    ctx.close()
    for b in range(sc.B):
        want = o.shot_noise(I0[b].astype(np.float64), 500.0, sc.seed, b) + 0.01 * o.read_noise(sc.seed, b, sc.H, sc.W)
        assert np.abs(I1[b] - want).max() <= 2e-6 * max(1.0, want.max())


def test_other_frame_sizes_keep_the_cufft_path(og, o):
    _check(og, o, _scene(96, 160, seed=3, NA=0.6))               # not powers of two
    _check(og, o, _scene(32, 64, seed=4, NA=0.6))                # below the smallest fused row


@pytest.mark.parametrize("H,W,B,dz", [(256, 128, 3, 0.0), (128, 512, 1, 2.0), (64, 4096, 1, 0.0), (96, 160, 1, 1.0)])
def test_adjoint_of_the_stage_fused_and_cufft_paths(og, o, H, W, B, dz):
    """osog_backward_intensity runs the same three kernels twice on power-of-two frames (epilogues g_V = G V and
    dL/dOPD = (4 pi / lambda) Im(g_U conj U), conjugated pupil) and keeps cuFFT elsewhere (96 x 160): the bar of
    tests/test_gpu_backward.py."""
    import torch
    kw = dict(NA=[0.3, 0.8, 0.5][:B], lam=[0.45, 0.6, 0.55][:B]) if B > 1 else dict(NA=0.6, lam=0.5)
    sc = replace(_scene(H, W, seed=7 * H + W, B=B, tilt_y_rad=-0.02, **kw), defocus_um=dz)
    rng = np.random.default_rng(H + W)
    GI = rng.standard_normal((sc.B, sc.H, sc.W)).astype(np.float32)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    g = ctx.backward_intensity(P, opt, torch.from_numpy(GI).cuda())
    assert torch.equal(g, ctx.backward_intensity(P, opt, torch.from_numpy(GI).cuda()))
    assert ctx.check_guards() == 0
    ctx.close()
    ref = o.backward_intensity(sc, GI)
    err = np.abs(g.cpu().numpy().astype(np.float64) - ref).max()
    assert err <= 2e-4 * np.abs(ref).max(), (err, np.abs(ref).max())


@pytest.mark.parametrize("H,W,B,shear,dz,pupil", [(128, 512, 1, (3, -2), 1.0, True), (256, 64, 2, (-30, 100), 0.0, True),
                                                  (64, 128, 1, (1, 1), 0.0, False)])
def test_dic_stage_fused_path(og, o, H, W, B, shear, dz, pupil):
    """The DIC image on power-of-two frames: K1 forms the interference image on the fly, K2 multiplies the kept columns (twice the
    pupil's radius: the support of the transfer function) by the cached OTF.  Bar of tests/test_gpu_defocus_dic.py."""
    kw = dict(NA=[0.35, 0.8][:B], lam=[0.5, 0.62][:B]) if B > 1 else dict(NA=0.6, lam=0.5)
    sc = replace(_scene(H, W, seed=11 * H + W, B=B, tilt_x_rad=0.02, **kw), defocus_um=dz)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc, pupil_enabled=pupil)
    dic = og.make_dic(shear[0], shear[1], 0.4)
    g = ctx.render_dic(P, opt, dic).clone()
    assert bool((g == ctx.render_dic(P, opt, dic)).all()) and ctx.check_guards() == 0
    ctx.close()
    ref = o.render_dic(sc, shear, 0.4, pupil_enabled=pupil)
    tol = 1e-4 * max(ref.mean(), 1e-3)
    err = np.abs(g.cpu().numpy().astype(np.float64) - ref).max()
    assert err <= tol, (err, tol)
