"""GPU parity of the widened library stage: defocus factor of Eq. 3 in
osog_render_intensity and the DIC image of Eq. 5 (osog_render_dic / osog_field_to_dic) against the
float64 oracle.  Bar (reading A15, as for the intensity): max abs error <= 1e-4 * mean(oracle image)."""
import math
from dataclasses import replace

import numpy as np
import pytest

from workloads import make_config, make_scene

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


@pytest.fixture(scope="module")
def fields(o):
    """Oracle exit waves of the workloads used below (computed once)."""
    cache = {}

    def get(k, n=None):
        if (k, n) not in cache:
            sc = make_config(k, n_override=n)
            cache[(k, n)] = (sc, o.render_field(sc))
        return cache[(k, n)]
    return get


def gpu_intensity(og, sc, pupil=True):
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    out = ctx.render_intensity(og.Particles.from_scene(sc), og.optics_from_scene(sc, pupil_enabled=pupil))
    out = out.cpu().numpy().astype(np.float64)
    ctx.close()
    return out


def gpu_dic(og, sc, shear, theta, pupil=True, repeat=1):
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P = og.Particles.from_scene(sc)
    opt = og.optics_from_scene(sc, pupil_enabled=pupil)
    for _ in range(repeat):
        out = ctx.render_dic(P, opt, og.make_dic(shear[0], shear[1], theta))
    out = out.cpu().numpy().astype(np.float64)
    assert ctx.status()[0] == 0
    ctx.close()
    return out


@pytest.mark.parametrize("k,dz", [(1, 2.0), (1, -7.5), (2, 4.0), (4, 1.5), (5, -3.0)])
def test_defocused_intensity_matches_oracle(og, o, fields, k, dz):
    sc0, U = fields(k)
    sc = replace(sc0, defocus_um=dz)
    ref = o.render_intensity(sc, U=U)
    g = gpu_intensity(og, sc)
    tol = 1e-4 * ref.mean()
    e = np.abs(g - ref).max()
    assert e <= tol, f"defocused intensity max abs err {e:.3e} > {tol:.3e}"
    # and defocus does something: it differs from the in-focus image by far more than the bar
    assert np.abs(ref - o.render_intensity(sc0, U=U)).max() > 100 * tol


def test_defocus_all_pass_pupil_drops_only_evanescent_bins(og, o, fields):
    sc0, U = fields(1)
    sc = replace(sc0, defocus_um=3.0)
    ref = o.render_intensity(sc, U=U, pupil_enabled=False)
    g = gpu_intensity(og, sc, pupil=False)
    assert np.abs(g - ref).max() <= 1e-4 * ref.mean()


def test_zero_defocus_is_bitwise_the_in_focus_path(og):
    import torch
    sc = make_config(2)
    a = gpu_intensity(og, sc)
    b = gpu_intensity(og, replace(sc, defocus_um=0.0))
    assert np.array_equal(a, b)


@pytest.mark.parametrize("k,shear,theta,dz", [(1, (2, 0), 0.5, 0.0), (1, (0, -3), -0.3, 2.0), (2, (3, 3), math.pi / 4, 0.0),
                                             (3, (1, 0), 0.2, 0.0), (4, (2, 1), 0.7, 1.0), (5, (-2, 4), 0.4, -2.0)])
def test_dic_matches_oracle(og, o, fields, k, shear, theta, dz):
    """All five BASELINE workloads at full size (config 5: 16 frames, per-frame lambda / NA, read noise)."""
    sc0, U = fields(k)
    sc = replace(sc0, defocus_um=dz)
    ref = o.render_dic(sc, shear, theta, U=U)
    g = gpu_dic(og, sc, shear, theta)
    tol = 1e-4 * ref.mean()
    e = np.abs(g - ref).max()
    assert e <= tol, f"DIC max abs err {e:.3e} > {tol:.3e}"


def test_dic_closed_forms_on_the_gpu(og):
    """No particles: U = ramp only.  On-bin ramp exp(2 pi i m j / W) => flat image 4 sin^2(2 pi m sx / W + theta) sum|P|^2/HW
    (pin C2 of the oracle, here straight against the closed form); zero shear => 4 sin^2(theta) sum|P|^2 / HW."""
    H = W = 128
    lam, p, m = 0.55, 0.1, 5
    tilt = math.asin(m * lam / (W * p))                           # ramp frequency sin(tilt) / lambda = m / (W p): bin m
    sc = make_scene("ramp", H, W, dict(cx=[], cy=[], d0=[], d1=[], d2=[], n_p=[]), lam=lam, NA=0.5, tilt_x_rad=tilt)
    ctx = og.Context(H, W, 0)
    P = og.Particles.from_scene(sc)
    opt = og.optics_from_scene(sc)
    mx = np.fft.fftfreq(W, 1.0 / W)
    npass = int(((mx[None, :] ** 2 + mx[:, None] ** 2) * (lam / (W * p)) ** 2 <= 0.5 ** 2).sum())
    for sx, sy, th in ((3, 0, 0.4), (0, 7, 0.4), (-2, 1, -1.1)):
        g = ctx.render_dic(P, opt, og.make_dic(sx, sy, th)).cpu().numpy().astype(np.float64)
        want = 4.0 * math.sin(2 * math.pi * m * sx / W + th) ** 2 * npass / (H * W)
        assert np.abs(g - want).max() <= 1e-4 * max(want, 1e-3), (sx, sy, th)
    ctx.close()


def test_dic_ragged_frame_wrap_and_repeat_calls(og, o):
    """Frame that is no tile multiple, shear large enough to wrap around the border, second call reuses the scratch."""
    rng = np.random.default_rng(11)
    H, W, n = 100, 150, 30
    cols = dict(cx=rng.uniform(0, W * 0.1, n), cy=rng.uniform(0, H * 0.1, n), d0=rng.uniform(0.5, 2, n),
                d1=rng.uniform(0.5, 2, n), d2=rng.uniform(0.5, 2, n), n_p=rng.uniform(1.36, 1.5, n))
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    cols.update(qw=q[:, 0], qx=q[:, 1], qy=q[:, 2], qz=q[:, 3], kind=(np.arange(n) % 2).astype(np.uint8))
    sc = make_scene("ragged_dic", H, W, cols, NA=0.6, defocus_um=1.0)
    ref = o.render_dic(sc, (140, -97), 0.3)
    g = gpu_dic(og, sc, (140, -97), 0.3, repeat=2)
    assert np.abs(g - ref).max() <= 1e-4 * ref.mean()


def test_field_to_dic_equals_render_dic_and_leaves_the_field_untouched(og):
    import torch
    sc = make_config(2)
    ctx = og.Context(sc.H, sc.W, sc.N)
    P = og.Particles.from_scene(sc)
    opt = og.optics_from_scene(sc)
    dic = og.make_dic(2, -1, 0.6)
    a = ctx.render_dic(P, opt, dic).clone()
    U = ctx.render_field(P, opt).clone()
    U0 = U.clone()
    b = ctx.field_to_dic(opt, dic, U)
    assert torch.equal(a, b) and torch.equal(torch.view_as_real(U), torch.view_as_real(U0))
    # the coherent path still works after the DIC path used the context's buffers
    c = ctx.render_intensity(P, opt)
    d = ctx.field_to_intensity(opt, U)
    assert torch.equal(c, d)
    ctx.close()


def test_dic_argument_errors(og):
    ctx = og.Context(64, 64, 4)
    sc = make_scene("e", 64, 64, dict(cx=[3.0], cy=[3.0], d0=[1.0], d1=[1.0], d2=[1.0], n_p=[1.4]))
    P = og.Particles.from_scene(sc)
    opt = og.optics_from_scene(sc)
    for bad in (og.make_dic(64, 0, 0.1), og.make_dic(0, -64, 0.1), og.make_dic(1, 1, float("nan"))):
        with pytest.raises(og.OsogError) as ei:
            ctx.render_dic(P, opt, bad)
        assert ei.value.code == og.OSOG_EINVAL
    d = og.make_dic(1, 1, 0.1)
    d.struct_size = 4
    with pytest.raises(og.OsogError):
        ctx.render_dic(P, opt, d)
    bad_opt = og.optics_from_scene(replace(sc, defocus_um=float("inf")))
    with pytest.raises(og.OsogError):
        ctx.render_intensity(P, bad_opt)
    ctx.render_dic(P, opt, og.make_dic(63, -63, 0.1))             # the largest allowed shear is fine
    assert ctx.status()[0] == 0
    ctx.close()


def test_cached_transfer_function_follows_the_optics(og, o, fields):
    """The OTF is kept between DIC calls and rebuilt only when the optics change: same optics twice -> same bits; a new
    NA, wavelength-independent defocus or pupil switch on the same context -> still the oracle's image."""
    import torch
    sc0, U = fields(1)
    ctx = og.Context(sc0.H, sc0.W, sc0.N)
    P = og.Particles.from_scene(sc0)
    dic = og.make_dic(2, 1, 0.5)
    first = ctx.render_dic(P, og.optics_from_scene(sc0), dic).clone()
    assert torch.equal(ctx.render_dic(P, og.optics_from_scene(sc0), dic), first)
    for change in (dict(NA=np.array([0.7])), dict(defocus_um=2.5), dict(lambda_um=np.array([0.48])), dict()):
        sc = replace(sc0, **change)
        Uc = o.render_field(sc) if "lambda_um" in change else U
        ref = o.render_dic(sc, (2, 1), 0.5, U=Uc)
        g = ctx.render_dic(P, og.optics_from_scene(sc), dic).cpu().numpy().astype(np.float64)
        assert np.abs(g - ref).max() <= 1e-4 * ref.mean(), change
    ref = o.render_dic(sc0, (2, 1), 0.5, U=U, pupil_enabled=False)
    g = ctx.render_dic(P, og.optics_from_scene(sc0, pupil_enabled=False), dic).cpu().numpy().astype(np.float64)
    assert np.abs(g - ref).max() <= 1e-4 * ref.mean()
    ctx.close()
