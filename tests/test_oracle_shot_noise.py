"""Pins of the oracle's Poisson shot noise (reading A26; "P(lambda) + G(0, sigma^2)").
The paper gives no constants, so the pins are what the mathematics fixes: the inversion branch against the library's
quantile function (the definition of inversion), both branches against the Poisson law (moments and a chi-square test
against scipy.stats.poisson.pmf), keying and stream separation, and the special cases."""
import numpy as np
import pytest
from scipy import stats

from oracle import oracle as o


def test_S1_inversion_branch_is_the_quantile_function():
    """lam < 10: the draw is F^-1(u) = the smallest k with CDF(k) >= u, for the very uniform the stream gives."""
    n = 20000
    rng = np.random.default_rng(0)
    lam = rng.uniform(0.01, 9.99, n)
    k = o.poisson_counts(lam, seed=123, frame=2)
    u = o.shot_uniforms(123, 2, np.arange(n), 0)[:, 0]
    want = stats.poisson.ppf(u, lam)
    edge = np.abs(stats.poisson.cdf(np.minimum(k, want), lam) - u) < 1e-12     # u on a CDF step to rounding: either is right
    assert np.all((k == want) | edge) and edge.sum() <= 1


@pytest.mark.parametrize("lam", [0.3, 4.0, 9.99, 10.0, 37.0, 1000.0, 2.5e5])
def test_S2_mean_and_variance_equal_lambda(lam):
    n = 1_000_000
    k = o.poisson_counts(np.full(n, lam), seed=7, frame=0).astype(np.float64)
    se_mean = np.sqrt(lam / n)
    assert abs(k.mean() - lam) < 5 * se_mean
    # var of the sample variance of a Poisson: (lam + 2 lam^2 ... ) / n ~ (lam + 2 lam^2) / n
    assert abs(k.var() - lam) < 5 * np.sqrt((lam + 2 * lam * lam) / n)


@pytest.mark.parametrize("lam", [3.7, 12.0, 25.0, 300.0])
def test_S3_chi_square_against_the_poisson_pmf(lam):
    n = 400_000
    k = o.poisson_counts(np.full(n, lam), seed=99, frame=1)
    lo, hi = int(stats.poisson.ppf(1e-4, lam)), int(stats.poisson.ppf(1 - 1e-4, lam))
    edges = np.arange(lo, hi + 2)
    obs = np.histogram(np.clip(k, lo, hi), bins=edges)[0].astype(np.float64)
    pm = stats.poisson.pmf(np.arange(lo, hi + 1), lam)
    pm[0] += stats.poisson.cdf(lo - 1, lam)
    pm[-1] += stats.poisson.sf(hi, lam)
    chi2 = ((obs - n * pm) ** 2 / (n * pm)).sum()
    assert chi2 < stats.chi2.ppf(1 - 1e-6, df=len(pm) - 1), chi2


def test_S4_special_cases_and_keying():
    assert np.all(o.poisson_counts(np.zeros(100), 1, 0) == 0)
    lam = np.full(5000, 20.0)
    a = o.poisson_counts(lam, seed=5, frame=3)
    assert np.array_equal(a, o.poisson_counts(lam, seed=5, frame=3))                   # a pure function of the key
    for other in (o.poisson_counts(lam, seed=6, frame=3), o.poisson_counts(lam, seed=5, frame=4),
                  o.poisson_counts(lam, seed=5, frame=3, pixels=np.arange(5000) + 5000)):
        assert (a != other).mean() > 0.8 and abs(np.corrcoef(a, other)[0, 1]) < 0.06
    # a draw depends on its own pixel only: a permutation of the pixels permutes the draws
    perm = np.random.default_rng(1).permutation(5000)
    assert np.array_equal(o.poisson_counts(lam, 5, 3, pixels=perm), a[perm])
    # the shot-noise stream (counter word 2 = 1) is not the read-noise stream (word 2 = 0)
    z = o.read_noise(5, 3, 50, 100).ravel()
    assert abs(np.corrcoef(a.astype(float), z)[0, 1]) < 0.06
    u = o.shot_uniforms(5, 3, np.arange(200000), 0)
    assert u.min() >= 0.0 and u.max() < 1.0 and abs(u.mean() - 0.5) < 0.003 and abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.01


def test_S5_shot_noise_of_an_image():
    I = np.linspace(0.0, 2.0, 64 * 64).reshape(64, 64)
    assert np.array_equal(o.shot_noise(I, 0.0, 1, 0), I)                              # photons = 0: off
    J = o.shot_noise(I, 500.0, 1, 0)
    assert np.abs(J * 500.0 - np.round(J * 500.0)).max() < 1e-9 and J.min() >= 0.0      # whole photons
    assert abs((J - I).mean()) < 5 * np.sqrt(I.mean() / 500.0 / I.size)
    assert abs(((J - I) ** 2).mean() - I.mean() / 500.0) < 0.1 * I.mean() / 500.0      # variance = I / photons
    neg = o.shot_noise(np.full((4, 4), -0.2), 100.0, 1, 0)
    assert np.all(neg == 0.0)                                                          # max(I, 0)


# ---- micro-topography of the height map (reading A29) ------------------------------------------------------------
def test_T1_topography_factor_statistics_keying_and_effect():
    from dataclasses import replace
    from workloads import make_config
    sc = make_config(2, n_override=60)
    sc.cols["cx"][:] = sc.cols["cx"] / 4; sc.cols["cy"][:] = sc.cols["cy"] / 4
    sc = replace(sc, H=256, W=256)
    smooth = o.render_opd(sc)
    assert np.all(o.topography_factor(sc, 0) == 1.0)                                   # amplitude 0: off
    a = 0.03
    rough = replace(sc, topography_amplitude=a)
    f = o.topography_factor(rough, 0)
    eta = (f - 1.0) / a
    n = eta.size
    assert abs(eta.mean()) < 5 / np.sqrt(n) and abs(eta.var() - 1.0) < 5 * np.sqrt(2.0 / n)      # N(0, 1)
    assert abs(stats.kstest(eta.ravel(), "norm").statistic) < 0.01
    # white: neighbouring pixels uncorrelated; its own stream: uncorrelated with the read noise of the same key
    assert abs(np.corrcoef(eta[:, :-1].ravel(), eta[:, 1:].ravel())[0, 1]) < 0.02
    assert abs(np.corrcoef(eta[:-1].ravel(), eta[1:].ravel())[0, 1]) < 0.02
    assert abs(np.corrcoef(eta.ravel(), o.read_noise(sc.seed, 0, 256, 256).ravel())[0, 1]) < 0.02
    assert not np.array_equal(f, o.topography_factor(replace(rough, seed=sc.seed + 1), 0))
    # every thickness at a pixel is scaled by the same factor: OPD and height scale with it, empty pixels stay empty
    assert np.array_equal(o.render_opd(rough)[0], smooth[0] * f)
    assert np.array_equal(o.render_height(rough)[0], o.render_height(sc)[0] * f)
    assert np.all(o.render_opd(rough)[smooth == 0.0] == 0.0)
    # and the images change accordingly: rougher bodies scatter more light out of the pupil
    assert not np.allclose(o.render_intensity(rough), o.render_intensity(sc), atol=1e-6)
