"""GPU parity of the rest of the backward pass: osog_backward_params
(dL/d(dimensions, quaternion)) and osog_spectral_loss (Eq. 8 and its gradient) against the oracle, and an end-to-end fit
that drives the whole chain: render -> Eq. 8 -> adjoint of the optics -> gradients in n_p, centre, dimensions, rotation."""
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


@pytest.mark.parametrize("k,n", [(1, None), (2, None), (3, 1500), (4, 3000), (5, 240)])
def test_backward_params_matches_oracle(og, o, k, n):
    import torch
    sc = make_config(k, n_override=n)
    rng = np.random.default_rng(50 + k)
    G = rng.standard_normal((sc.B, sc.H, sc.W)).astype(np.float32)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    Gd = torch.from_numpy(G).cuda()
    g = ctx.backward_params(P, opt, Gd)
    assert torch.equal(g, ctx.backward_params(P, opt, Gd))      # fixed summation order: same bits
    assert ctx.check_guards() == 0
    g = g.cpu().numpy().astype(np.float64)
    ref = o.backward_params(sc, G)
    # both sides sum analytic float64 terms; left: the float32 rounding of the result and, near an ellipsoid's outline
    # where dt/dtheta ~ 1 / sqrt(w), the ~1e-9 relative difference between two evaluation orders of the discriminant
    scale = np.abs(o.backward_params(sc, np.abs(G))) + np.abs(ref)
    big = np.maximum(scale.max(axis=1, keepdims=True), 1.0)
    err = np.abs(g - ref)
    print(f"cfg {k}: max rel err {(err / big).max():.2e}")
    assert np.all(err <= 5e-7 * big), float((err / big).max())
    ctx.close()


def test_backward_params_skips_invalid_and_off_canvas_particles(og, o):
    import torch
    # (the prism has identity rotation: vertical faces, thickness discontinuous there; its centre and side are chosen so
    # that no pixel centre lies within 1e-3 um of a vertical face, as in the forward tests)
    cols = dict(cx=[3.0, 500.0, 4.013, 5.0], cy=[3.0, 3.0, 4.021, float("nan")], d0=[1.0, 1.0, 1.57, 1.0], d1=[1.0, 1.0, 2.5, 1.0],
                d2=[1.0, 1.0, 0.6, 1.0], n_p=[1.4] * 4, kind=np.array([0, 0, 1, 0], np.uint8))
    sc = make_scene("edge", 80, 96, cols)
    G = np.ones((1, 80, 96), np.float32)
    ctx = og.Context(sc.H, sc.W, sc.N, check=False)
    g = ctx.backward_params(og.Particles.from_scene(sc), og.optics_from_scene(sc), torch.from_numpy(G).cuda()).cpu().numpy()
    ref = o.backward_params(sc, G)
    assert np.all(g[1] == 0.0) and np.all(g[3] == 0.0) and np.abs(g[0]).max() > 0 and np.abs(g[2]).max() > 0
    assert np.allclose(g, ref, rtol=1e-5, atol=1e-5)
    ctx.close()


@pytest.mark.parametrize("H,W,B", [(64, 96, 1), (256, 256, 3), (1024, 1024, 1)])
def test_spectral_loss_matches_oracle(og, o, H, W, B):
    import torch
    rng = np.random.default_rng(H + B)
    I = (1.0 + 0.3 * rng.standard_normal((B, H, W))).astype(np.float32)
    T = (1.0 + 0.3 * rng.standard_normal((B, H, W))).astype(np.float32)
    eps = 1e-3
    ctx = og.Context(H, W, 0, max_frames=B)
    loss, g = ctx.spectral_loss(torch.from_numpy(I).cuda(), torch.from_numpy(T).cuda(), eps)
    loss2, none = ctx.spectral_loss(torch.from_numpy(I).cuda(), torch.from_numpy(T).cuda(), eps, grad=False)
    assert none is None and torch.equal(loss, loss2) and ctx.check_guards() == 0
    loss, g = loss.cpu().numpy(), g.cpu().numpy().astype(np.float64)
    for b in range(B):
        want = o.spectral_loss(I[b], T[b], eps)
        gw = o.spectral_loss_grad(I[b], T[b], eps)
        # float32 FFT of H W samples: |F| good to ~1e-6 relative of the typical magnitude; the loss sums H W squared log differences
        assert abs(loss[b] - want) <= 2e-4 * want, (loss[b], want)
        assert np.abs(g[b] - gw).max() <= 2e-3 * np.abs(gw).max(), (np.abs(g[b] - gw).max(), np.abs(gw).max())
    zero, gz = ctx.spectral_loss(torch.from_numpy(T).cuda(), torch.from_numpy(T).cuda(), eps)
    assert float(zero.abs().max()) == 0.0 and float(gz.abs().max()) == 0.0
    with pytest.raises(og.OsogError):
        ctx.spectral_loss(torch.from_numpy(I).cuda(), torch.from_numpy(T).cuda(), 0.0)
    ctx.close()


def test_end_to_end_fit_with_the_spectral_loss(og, o):
    """DiffOSOG in miniature: a target image is rendered from known parameters; starting from perturbed
    refractive indices and dimensions, gradient descent on Eq. 8 through the whole chain (osog_render_intensity ->
    osog_spectral_loss -> osog_backward_intensity -> osog_backward_np / _params) brings the loss down and the parameters
    back towards the truth.  (Prisms: their thickness is piecewise linear, so the chain gradient is the derivative of the
    pixel-sampled loss almost everywhere.)"""
    import torch
    rng = np.random.default_rng(11)
    n = 12
    q = rng.standard_normal((n, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    s = rng.uniform(1.5, 3.0, n)
    cols = dict(cx=rng.uniform(3.0, 22.0, n), cy=rng.uniform(3.0, 22.0, n), qw=q[:, 0], qx=q[:, 1], qy=q[:, 2], qz=q[:, 3],
                d0=s, d1=s * rng.uniform(1.2, 2.5, n), d2=0.5 * s, n_p=rng.uniform(1.38, 1.45, n), kind=np.ones(n, np.uint8))
    truth = make_scene("fit", 256, 256, cols, NA=0.5)
    ctx = og.Context(truth.H, truth.W, n)
    opt = og.optics_from_scene(truth)
    target = ctx.render_intensity(og.Particles.from_scene(truth), opt).clone()
    cur = {k: v.copy() for k, v in truth.cols.items()}
    cur["n_p"] = (cur["n_p"] + rng.uniform(-0.02, 0.02, n)).astype(np.float32)
    cur["d1"] = (cur["d1"] * rng.uniform(0.93, 1.07, n)).astype(np.float32)
    eps = 1e-2
    err0 = (np.abs(cur["n_p"] - truth.cols["n_p"]).mean(), np.abs(cur["d1"] - truth.cols["d1"]).mean())
    losses = []
    lr_np, lr_d = 2e-8, 2e-5
    for it in range(120):
        P = og.Particles(cur, None)
        I = ctx.render_intensity(P, opt)
        loss, gI = ctx.spectral_loss(I, target, eps)
        gopd = ctx.backward_intensity(P, opt, gI)
        gnp = ctx.backward_np(P, opt, gopd).cpu().numpy()
        gpar = ctx.backward_params(P, opt, gopd).cpu().numpy()
        losses.append(float(loss[0]))
        cur["n_p"] = (cur["n_p"] - lr_np * gnp).astype(np.float32)
        cur["d1"] = (cur["d1"] - lr_d * gpar[:, 1]).astype(np.float32)
    err1 = (np.abs(cur["n_p"] - truth.cols["n_p"]).mean(), np.abs(cur["d1"] - truth.cols["d1"]).mean())
    print("loss", losses[0], "->", losses[-1], "| mean |n_p error|", err0[0], "->", err1[0], "| mean |L error|", err0[1], "->", err1[1])
    assert losses[-1] < 0.5 * losses[0]
    assert err1[0] < err0[0] and err1[1] < err0[1]
    ctx.close()


def test_gathers_refuse_micro_topography(og):
    """The gradient gathers differentiate the smooth bodies: with topography_amplitude != 0 they return OSOG_EINVAL."""
    import torch
    sc = replace(make_config(2, n_override=50), topography_amplitude=0.02)
    ctx = og.Context(sc.H, sc.W, sc.N)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    G = torch.ones((1, sc.H, sc.W), dtype=torch.float32, device="cuda")
    for call in (ctx.backward_np, ctx.backward_centre, ctx.backward_params):
        with pytest.raises(og.OsogError) as e:
            call(P, opt, G)
        assert e.value.code == og.OSOG_EINVAL
    ctx.close()


@pytest.mark.parametrize("k,n", [(2, None), (3, 1500), (4, 3000), (5, 240)])
def test_backward_particles_one_pass_equals_the_three_gathers(og, o, k, n):
    """osog_backward_particles forms dL/dn_p, dL/d(cx, cy) and dL/d(dims, q) from one set of moments: same numbers as the three
    separate gathers up to a different float64 summation order, and the same bars against the oracle."""
    import torch
    sc = make_config(k, n_override=n)
    rng = np.random.default_rng(70 + k)
    G = rng.standard_normal((sc.B, sc.H, sc.W)).astype(np.float32)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    Gd = torch.from_numpy(G).cuda()
    gnp, gc, gpar = ctx.backward_particles(P, opt, Gd)
    again = ctx.backward_particles(P, opt, Gd)
    assert all(torch.equal(a, b) for a, b in zip((gnp, gc, gpar), again))          # reproducible bits
    only_c = ctx.backward_particles(P, opt, Gd, np_=False, params=False)
    assert only_c[0] is None and only_c[2] is None and torch.equal(only_c[1], gc)
    assert ctx.check_guards() == 0
    absG = np.abs(G)
    f64 = lambda t: t.cpu().numpy().astype(np.float64)
    # dL/dn_p: the bar of test_backward_np_matches_oracle (relative to the sum of magnitudes)
    ref, scale = o.backward_np(sc, G), o.backward_np(sc, absG)
    assert np.all(np.abs(f64(gnp) - ref) <= 2e-7 * scale + 1e-6)
    assert np.all(np.abs(f64(gnp) - f64(ctx.backward_np(P, opt, Gd))) <= 2e-7 * scale + 1e-6)
    # dL/d(cx, cy) and dL/d(dims, q): the bars of their own parity tests (per particle, relative to the largest component's scale)
    for got, sep, fn in ((gc, ctx.backward_centre(P, opt, Gd), o.backward_centre), (gpar, ctx.backward_params(P, opt, Gd), o.backward_params)):
        ref = fn(sc, G)
        big = np.maximum((np.abs(fn(sc, absG)) + np.abs(ref)).max(axis=1, keepdims=True), 1.0)
        assert np.all(np.abs(f64(got) - ref) <= 5e-7 * big), float((np.abs(f64(got) - ref) / big).max())
        assert np.all(np.abs(f64(got) - f64(sep)) <= 5e-7 * big), float((np.abs(f64(got) - f64(sep)) / big).max())
    ctx.close()
