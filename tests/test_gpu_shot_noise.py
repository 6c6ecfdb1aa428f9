"""GPU parity of the Poisson shot noise (reading A26) against the oracle.
The integer draw is index-like work decided by float64 comparisons: on the same rates both sides must give the same
counts; a difference is accepted only where the oracle's own decision is within rounding (a uniform within 1e-12 of a CDF
step for the inversion branch; none was ever seen).  The noisy intensity / DIC image is compared with the oracle's sensor
model applied to the GPU's OWN noise-free image (both then decide the draw on the same float32 rates), at float32 rounding."""
from dataclasses import replace

import numpy as np
import pytest

from workloads import make_config

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


def test_poisson_draws_equal_the_oracle_bit_for_bit(og, o):
    import torch
    rng = np.random.default_rng(3)
    n = 400_000
    lam = np.concatenate([rng.uniform(0.0, 10.0, n // 4), rng.uniform(10.0, 60.0, n // 4), 10.0 ** rng.uniform(1.0, 5.5, n // 4),
                          np.array([0.0, 9.999999, 10.0, 10.000001, 1e-30, 3e5]), rng.uniform(9.9, 10.1, n // 4 - 6)]).astype(np.float32)
    ctx = og.Context(64, 64, 0)
    for seed, frame in ((0, 0), (0xDEADBEEFCAFE1234, 7)):
        got = ctx.poisson(torch.from_numpy(lam), seed, frame).cpu().numpy().astype(np.int64)
        want = o.poisson_counts(lam.astype(np.float64), seed, frame)
        differ = np.flatnonzero(got != want)
        print(f"poisson: {differ.size} of {lam.size} draws differ")
        assert differ.size == 0, (lam[differ][:5], got[differ][:5], want[differ][:5])
    ctx.close()


@pytest.mark.parametrize("k,photons,sigma", [(2, 200.0, 0.0), (4, 5000.0, 0.01), (5, 40.0, 0.01)])
def test_intensity_with_shot_noise_is_the_oracles_sensor_on_the_same_image(og, o, k, photons, sigma):
    sc = replace(make_config(k), shot_noise_photons=photons, read_noise_sigma=sigma)
    clean = replace(sc, shot_noise_photons=0.0, read_noise_sigma=0.0)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P = og.Particles.from_scene(sc)
    I0 = ctx.render_intensity(P, og.optics_from_scene(clean)).cpu().numpy()            # float32, noise-free
    I1 = ctx.render_intensity(P, og.optics_from_scene(sc)).cpu().numpy().astype(np.float64)
    ctx.close()
    want = np.empty_like(I1)
    for b in range(sc.B):
        J = o.shot_noise(I0[b].astype(np.float64), photons, sc.seed, b)
        want[b] = J + (sigma * o.read_noise(sc.seed, b, sc.H, sc.W) if sigma else 0.0)
    err = np.abs(I1 - want)
    assert err.max() <= 2e-6 * max(1.0, want.max()), err.max()
    # and it is shot noise: whole photons, variance I / photons
    if sigma == 0.0:
        assert np.abs(I1 * photons - np.round(I1 * photons)).max() < 1e-3
    d = I1 - I0
    assert abs(d.mean()) < 6 * np.sqrt((I0.mean() / photons + sigma * sigma) / d.size)
    assert abs(d.var() / (I0.mean() / photons + sigma * sigma) - 1.0) < 0.05


def test_dic_with_shot_noise_and_argument_check(og, o):
    sc = replace(make_config(2, n_override=300), shot_noise_photons=800.0)
    ctx = og.Context(sc.H, sc.W, sc.N)
    P = og.Particles.from_scene(sc)
    dic = og.make_dic(2, 1, 0.6)
    D0 = ctx.render_dic(P, og.optics_from_scene(replace(sc, shot_noise_photons=0.0)), dic).cpu().numpy()
    D1 = ctx.render_dic(P, og.optics_from_scene(sc), dic).cpu().numpy().astype(np.float64)
    want = o.shot_noise(D0[0].astype(np.float64), 800.0, sc.seed, 0)
    assert np.abs(D1[0] - want).max() <= 2e-6 * max(1.0, want.max())
    bad = og.make_optics(1, 0.1, 1.33, 0.55, 0.4, shot_noise_photons=-1.0)
    with pytest.raises(og.OsogError) as e:
        ctx.render_intensity(P, bad)
    assert e.value.code == og.OSOG_EINVAL
    ctx.close()


@pytest.mark.parametrize("k,amp", [(2, 0.05), (4, 0.02), (5, 0.03)])
def test_micro_topography_matches_oracle(og, o, k, amp):
    """Micro-topography of the height map (reading A29): OPD, field, intensity and height with
    topography_amplitude > 0 against the oracle.  Bars: the hot path's own (OPD 1e-5 + 1e-5 |o|, field / intensity 1e-4 mean I),
    widened by what the float32 Box-Muller normal of the kernel allows: |d eta| <= 2e-6, so OPD gets + amp * 2e-6 * |o| and
    the field + 2 pi / lambda times that."""
    sc = replace(make_config(k), topography_amplitude=amp)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    opd = ctx.render_opd(P, opt).cpu().numpy().astype(np.float64)
    U = ctx.render_field(P, opt).cpu().numpy().astype(np.complex128)
    I = ctx.render_intensity(P, opt).cpu().numpy().astype(np.float64)
    h = ctx.render_height(P, opt, grad=False, lap=False)[0].cpu().numpy().astype(np.float64)
    smooth = ctx.render_opd(P, og.optics_from_scene(replace(sc, topography_amplitude=0.0))).cpu().numpy()
    assert ctx.status()[0] == 0 and ctx.check_guards() == 0
    ctx.close()
    ref = o.render_opd(sc)
    assert np.all(np.abs(opd - ref) <= 1e-5 + (1e-5 + 2e-6 * amp) * np.abs(ref)), float(np.abs(opd - ref).max())
    assert not np.allclose(opd, smooth, atol=1e-4)                  # it really is a different surface
    href = o.render_height(sc)
    assert np.all(np.abs(h - href) <= 1e-5 + (1e-5 + 2e-6 * amp) * np.abs(href))
    Uref = o.render_field(sc, opd=ref)
    Iref = o.render_intensity(sc, U=Uref)
    lam_min = float(np.min(sc.lambda_um))
    tol = 1e-4 * Iref.mean() + 2 * np.pi / lam_min * 2e-6 * amp * float(np.abs(ref).max())
    assert np.abs(U - Uref).max() <= tol, (np.abs(U - Uref).max(), tol)
    assert np.abs(I - Iref).max() <= 2 * tol, (np.abs(I - Iref).max(), tol)
