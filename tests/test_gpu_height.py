"""GPU parity of the G-buffer height map and its finite-difference gradient / Laplacian (osog_render_height, SURVEY 8(f)
NEXT-2, reading A25) against the oracle.  Bars: h as the OPD frame (|g - o| <= 1e-5 um + 1e-5 |o|); the stencils amplify a
height error e to e / p (gradient) and 8 e / p^2 (Laplacian), so their bars are those of h scaled accordingly."""
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


def check(og, o, sc):
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P = og.Particles.from_scene(sc)
    opt = og.optics_from_scene(sc)
    h, g, l = ctx.render_height(P, opt)
    h, g, l = (t.cpu().numpy().astype(np.float64) for t in (h, g, l))
    h_only = ctx.render_height(P, opt, grad=False, lap=False)[0].cpu().numpy().astype(np.float64)
    assert np.array_equal(h_only, h)
    assert ctx.status()[0] == 0
    ctx.close()
    ref = o.render_height(sc)
    p = sc.pitch_um
    tol_h = 1e-5 + 1e-5 * np.abs(ref)
    assert np.all(np.abs(h - ref) <= tol_h), float(np.abs(h - ref).max())
    for b in range(sc.B):
        gx, gy = o.height_gradient(ref[b], p)
        th = float(tol_h[b].max())
        tol_g = 2 * th / p + 1e-5 * np.maximum(np.abs(gx), np.abs(gy))
        assert np.all(np.abs(g[b, :, :, 0] - gx) <= tol_g) and np.all(np.abs(g[b, :, :, 1] - gy) <= tol_g)
        # the stencils are exact functions of h: applied to the GPU's own h they reproduce its outputs to float rounding
        gx2, gy2 = o.height_gradient(h[b], p)
        assert np.all(np.abs(g[b, :, :, 0] - gx2) <= 2e-6 * (np.abs(gx2) + np.abs(h[b]).max() / p))
        assert np.all(np.abs(g[b, :, :, 1] - gy2) <= 2e-6 * (np.abs(gy2) + np.abs(h[b]).max() / p))
    lap = np.stack([o.height_laplacian(ref[b], p) for b in range(min(sc.B, 2))])
    tol_l = 8 * float(tol_h.max()) / (p * p) + 1e-5 * np.abs(lap)
    assert np.all(np.abs(l[:lap.shape[0]] - lap) <= tol_l)


@pytest.mark.parametrize("k,n", [(1, None), (2, None), (3, 4000), (4, 8000), (5, 600)])
def test_height_gradient_laplacian_match_oracle(og, o, k, n):
    check(og, o, make_config(k, n_override=n))


def test_height_on_a_ragged_frame_and_full_config4_height_only(og, o):
    rng = np.random.default_rng(5)
    n = 40
    q = rng.standard_normal((n, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    cols = dict(cx=rng.uniform(-1, 14, n), cy=rng.uniform(-1, 11, n), d0=rng.uniform(0.4, 2, n), d1=rng.uniform(0.4, 3, n),
                d2=rng.uniform(0.3, 1.5, n), n_p=rng.uniform(1.36, 1.5, n), qw=q[:, 0], qx=q[:, 1], qy=q[:, 2], qz=q[:, 3],
                kind=(np.arange(n) % 2).astype(np.uint8))
    check(og, o, make_scene("ragged_h", 100, 130, cols))
    sc = make_config(4)
    ctx = og.Context(sc.H, sc.W, sc.N)
    h = ctx.render_height(og.Particles.from_scene(sc), og.optics_from_scene(sc), grad=False, lap=False)[0]
    ref = o.render_height(sc)
    assert np.all(np.abs(h.cpu().numpy().astype(np.float64) - ref) <= 1e-5 + 1e-5 * np.abs(ref))
    ctx.close()
