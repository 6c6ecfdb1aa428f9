"""GPU parity of the brightfield amplitude of Eq. 4 (osog_render_brightfield, reading A27;
PAPER.md:94-99) against the oracle.  Bar: the intensity bar of the hot path, max |dI| <= 1e-4 mean(I), plus what the
float32 height map allows in the curvature term: the Laplacian divides second differences of a float32 map of heights up
to h_max by p^2, so the caustic term carries up to gain * 4 * 2^-24 h_max / p^2 of rounding that no kernel can avoid."""
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


@pytest.mark.parametrize("k,npart,dmu,gain", [(1, 1.42, 0.05, 0.02), (2, 1.45, 0.03, 0.01), (3, 1.41, 0.02, 0.01),
                                              (4, 1.43, 0.01, 0.005), (5, 1.44, 0.04, 0.01)])
def test_brightfield_matches_oracle_on_the_baseline_workloads(og, o, k, npart, dmu, gain):
    sc = make_config(k)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P = og.Particles.from_scene(sc)
    got = ctx.render_brightfield(P, og.optics_from_scene(sc), og.make_brightfield(npart, dmu, gain)).cpu().numpy().astype(np.float64)
    assert ctx.status()[0] == 0 and ctx.check_guards() == 0
    ctx.close()
    want = o.render_brightfield(sc, npart, dmu, gain)
    hmax = float(o.render_height(sc).max())
    amp = np.sqrt(want.max())
    tol = 1e-4 * want.mean() + 2.0 * amp * gain * 4.0 * 2.0 ** -24 * hmax / sc.pitch_um ** 2
    err = np.abs(got - want).max()
    print(f"cfg {k}: brightfield max err {err:.3e}, tol {tol:.3e} (hot-path part {1e-4 * want.mean():.3e})")
    assert err <= tol


def test_brightfield_neutral_parameters_and_argument_checks(og, o):
    import torch
    sc = make_config(2, n_override=300)
    ctx = og.Context(sc.H, sc.W, sc.N)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    plain = ctx.render_intensity(P, opt).clone()
    same = ctx.render_brightfield(P, opt, og.make_brightfield(sc.n_medium, 0.0, 0.0))
    assert torch.equal(plain, same)                       # T_F = 1, no absorption, no caustic: A == 1 exactly
    dark = ctx.render_brightfield(P, opt, og.make_brightfield(1.45, 0.2, 0.0))
    assert float(dark.mean()) < float(plain.mean())
    for bad in (og.make_brightfield(0.0), og.make_brightfield(float("nan")), og.make_brightfield(1.4, float("inf"))):
        with pytest.raises(og.OsogError) as e:
            ctx.render_brightfield(P, opt, bad)
        assert e.value.code == og.OSOG_EINVAL
    # the hot path is untouched by a brightfield call in between
    assert torch.equal(ctx.render_intensity(P, opt), plain)
    ctx.close()
