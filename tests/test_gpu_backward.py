"""GPU parity of the first backward step (osog_backward_np: dL/dn_p) against the oracle, and against
the GPU's own forward model differenced in n_p (the OPD sum is linear in it)."""
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


@pytest.mark.parametrize("k,n", [(1, None), (2, None), (3, 2000), (4, 4000), (5, 300)])
def test_backward_np_matches_oracle(og, o, k, n):
    import torch
    sc = make_config(k, n_override=n)
    rng = np.random.default_rng(k)
    G = rng.standard_normal((sc.B, sc.H, sc.W)).astype(np.float32)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    Gd = torch.from_numpy(G).cuda()
    g = ctx.backward_np(P, opt, Gd)
    g2 = ctx.backward_np(P, opt, Gd)
    assert torch.equal(g, g2)                                    # fixed summation order: same bits
    g = g.cpu().numpy().astype(np.float64)
    ref = o.backward_np(sc, G)
    # float32 result of a float64 sum of up to ~1e4 terms of either sign: bar relative to the sum of magnitudes
    scale = o.backward_np(sc, np.abs(G))
    assert np.all(np.abs(g - ref) <= 2e-7 * scale + 1e-6), float(np.abs(g - ref).max())
    # the context still renders the same bits afterwards
    a = ctx.render_opd(P, opt).clone()
    fresh = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    assert torch.equal(a, fresh.render_opd(P, opt))
    fresh.close()
    ctx.close()


def test_backward_np_is_the_forward_model_differenced(og):
    """L = sum G * OPD(n_p) rendered by the hot path (fp32 output): (L(n_p + d e_n) - L(n_p)) / d ~ dL/dn_p[n]."""
    import torch
    sc = make_config(4, n_override=200)
    rng = np.random.default_rng(9)
    G = torch.from_numpy(np.abs(rng.standard_normal((1, sc.H, sc.W))).astype(np.float32)).cuda()
    ctx = og.Context(sc.H, sc.W, sc.N)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    g = ctx.backward_np(P, opt, G).cpu().numpy().astype(np.float64)
    L0 = float((G.double() * ctx.render_opd(P, opt).double()).sum())
    assert ctx.status()[0] == 0 and L0 > 0.0
    for n in (3, 77, 150):
        cols = dict(sc.cols)
        npn = cols["n_p"].copy(); npn[n] += np.float32(0.5); cols["n_p"] = npn
        P1 = og.Particles(cols, None)
        L1 = float((G.double() * ctx.render_opd(P1, opt).double()).sum())
        step = float(npn[n]) - float(sc.cols["n_p"][n])
        assert abs((L1 - L0) / step - g[n]) <= 2e-4 * abs(g[n]) + 1e-3, (n, (L1 - L0) / step, g[n])
    ctx.close()


@pytest.mark.parametrize("k,n", [(1, None), (2, None), (3, 2000), (4, 4000), (5, 300)])
def test_backward_centre_matches_oracle(og, o, k, n):
    import torch
    sc = make_config(k, n_override=n)
    rng = np.random.default_rng(20 + k)
    G = rng.standard_normal((sc.B, sc.H, sc.W)).astype(np.float32)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    Gd = torch.from_numpy(G).cuda()
    g = ctx.backward_centre(P, opt, Gd)
    assert torch.equal(g, ctx.backward_centre(P, opt, Gd))      # fixed summation order: same bits
    g = g.cpu().numpy().astype(np.float64)
    ref = o.backward_centre(sc, G)
    # both sides sum in float64; what is left is the float32 rounding of the result (measured: 8e-8 of the scale below)
    # and, near an ellipsoid's outline where grad t ~ 1 / sqrt(w), the ~1e-9 relative difference of the two formulas for w
    scale = np.abs(o.backward_centre(sc, np.abs(G))) + np.abs(ref)
    big = np.maximum(scale.max(axis=1, keepdims=True), 1.0)
    err = np.abs(g - ref)
    assert np.all(err <= 5e-7 * big), float((err / big).max())
    ctx.close()


@pytest.mark.parametrize("k,n,dz", [(1, None, 0.0), (2, None, 1.5), (4, 4000, 0.0), (5, 300, -1.0)])
def test_backward_intensity_matches_oracle(og, o, k, n, dz):
    """Adjoint of the optics stage: dL/dOPD from dL/dI.  Bar: the field bar of north_star carried through the bilinear
    form Im(g_U conj(U)): max abs error <= 2e-4 of the largest gradient magnitude."""
    import torch
    from dataclasses import replace
    sc = replace(make_config(k, n_override=n), defocus_um=dz)
    rng = np.random.default_rng(30 + k)
    GI = rng.standard_normal((sc.B, sc.H, sc.W)).astype(np.float32)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    g = ctx.backward_intensity(P, opt, torch.from_numpy(GI).cuda()).cpu().numpy().astype(np.float64)
    ref = o.backward_intensity(sc, GI)
    err = np.abs(g - ref).max()
    assert err <= 2e-4 * np.abs(ref).max(), (err, np.abs(ref).max())
    assert np.abs(ref).max() > 1.0
    ctx.close()


def test_full_chain_gradient_of_an_intensity_loss(og, o):
    """L = sum W I(theta): backward_intensity -> backward_np / backward_centre give dL/dn_p and dL/dc.
    dL/dn_p is checked against central differences of the GPU's own forward intensity (L is smooth in n_p).  dL/dc is the
    almost-everywhere derivative of a pixel-sampled loss (outline pixels that cross a pixel centre during a shift add steps
    that no analytic gradient contains: see include/osog.h and pins B4-B6), so it is checked against the oracle's chain."""
    import torch
    sc = make_config(4, n_override=120)
    sc.cols["cx"][:] = (sc.cols["cx"] * 0.5).astype(np.float32)          # crowd them into a quarter of the frame
    sc.cols["cy"][:] = (sc.cols["cy"] * 0.5).astype(np.float32)
    rng = np.random.default_rng(5)
    W = rng.standard_normal((1, sc.H, sc.W)).astype(np.float32)
    Wt = torch.from_numpy(W).cuda()
    ctx = og.Context(sc.H, sc.W, sc.N)
    opt = og.optics_from_scene(sc)

    def L(cols):
        return float((Wt.double() * ctx.render_intensity(og.Particles(cols, None), opt).double()).sum())

    P = og.Particles.from_scene(sc)
    gopd = ctx.backward_intensity(P, opt, Wt)
    gnp = ctx.backward_np(P, opt, gopd).cpu().numpy().astype(np.float64)
    gc = ctx.backward_centre(P, opt, gopd).cpu().numpy().astype(np.float64)
    for n in (1, 17, 42, 77):
        d = 2.0 ** -9
        vals = []
        for sgn in (+1, -1):
            cols = dict(sc.cols); a = cols["n_p"].copy(); a[n] = np.float32(a[n] + sgn * d); cols["n_p"] = a
            vals.append(L(cols))
        fd = (vals[0] - vals[1]) / (2 * d)
        assert abs(fd - gnp[n]) <= 5e-2 * max(abs(gnp[n]), 0.05 * np.abs(gnp).max()), (n, fd, gnp[n])
    ref_gopd = o.backward_intensity(sc, W)
    ref_np, ref_c = o.backward_np(sc, ref_gopd), o.backward_centre(sc, ref_gopd)
    assert np.abs(gnp - ref_np).max() <= 1e-3 * np.abs(ref_np).max()
    assert np.abs(gc - ref_c).max() <= 1e-3 * np.abs(ref_c).max()
    ctx.close()
