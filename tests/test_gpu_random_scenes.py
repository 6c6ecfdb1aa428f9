"""Randomised parity: many small seeded scenes with adversarial parameter distributions (near-vertical prism faces,
needle / disc ellipsoids, sub-pixel and frame-filling particles, n_p below the medium, centres far off the frame),
each compared with the oracle in its plain `full` mode (no culling at all on the oracle side)."""
import numpy as np
import pytest

from workloads import make_scene
from test_gpu_parity import og, o  # noqa: F401  (fixtures)

pytestmark = pytest.mark.gpu

H, W = 96, 136


def _quat(rng, n, style):
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    if style == "near_axis":
        # rotations by almost exact multiples of 90 degrees about a coordinate axis: prism faces almost parallel to z
        base = np.array([[1, 0, 0, 0], [np.sqrt(.5), np.sqrt(.5), 0, 0], [np.sqrt(.5), 0, np.sqrt(.5), 0],
                         [np.sqrt(.5), 0, 0, np.sqrt(.5)], [0, 1, 0, 0], [.5, .5, .5, .5]], dtype=np.float64)
        q = base[rng.integers(0, len(base), n)] + rng.standard_normal((n, 4)) * 10.0 ** rng.uniform(-7, -2, (n, 1))
        q /= np.linalg.norm(q, axis=1, keepdims=True)
    return q


def _scene(seed):
    rng = np.random.default_rng(1000 + seed)
    style = ("uniform", "near_axis", "needles", "tiny_and_huge")[seed % 4]
    n = int(rng.integers(20, 90))
    kind = (rng.uniform(size=n) < 0.5).astype(np.uint8)
    q = _quat(rng, n, "near_axis" if style == "near_axis" else "uniform")
    if style == "needles":
        abc = np.stack([rng.uniform(0.05, 0.3, n), rng.uniform(0.05, 6.0, n), rng.uniform(2.0, 9.0, n)], 1)
        abc = np.take_along_axis(abc, rng.permuted(np.tile(np.arange(3), (n, 1)), axis=1), 1)
        s = rng.uniform(0.1, 0.6, n); L = s * rng.uniform(5, 30, n); hc = s * rng.uniform(0.05, 3.0, n)
    elif style == "tiny_and_huge":
        scale = 10.0 ** rng.uniform(-1.7, 1.3, n)                  # 0.02 um .. 20 um
        abc = scale[:, None] * rng.uniform(0.5, 1.5, (n, 3))
        s = scale; L = s * rng.uniform(0.2, 3.0, n); hc = s * rng.uniform(0.1, 1.0, n)
    else:
        abc = rng.uniform(0.3, 4.0, (n, 3))
        s = rng.uniform(0.5, 4.0, n); L = s * rng.uniform(0.3, 3.0, n); hc = s * rng.uniform(0.1, 1.5, n)
    d = np.where(kind[:, None] == 1, np.stack([s, L, hc], 1), abc)
    cols = dict(cx=rng.uniform(-4.0, W * 0.1 + 4.0, n), cy=rng.uniform(-4.0, H * 0.1 + 4.0, n),
                qw=q[:, 0], qx=q[:, 1], qy=q[:, 2], qz=q[:, 3], d0=d[:, 0], d1=d[:, 1], d2=d[:, 2],
                n_p=rng.uniform(1.25, 1.55, n), kind=kind)       # some particles are optically thinner than the medium
    return make_scene(f"random{seed}", H, W, cols, lam=float(rng.uniform(0.45, 0.65)), NA=float(rng.uniform(0.3, 0.9)),
                      tilt_x_rad=float(rng.uniform(-0.2, 0.2)), tilt_y_rad=float(rng.uniform(-0.2, 0.2)))


@pytest.mark.parametrize("seed", range(24))
def test_random_scene_matches_oracle_full_mode(og, o, seed):
    sc = _scene(seed)
    ctx = og.Context(sc.H, sc.W, sc.N)
    P = og.Particles.from_scene(sc)
    opt = og.optics_from_scene(sc)
    opd = ctx.render_opd(P, opt).cpu().numpy().astype(np.float64)[0]
    U = ctx.render_field(P, opt).cpu().numpy().astype(np.complex128)[0]
    assert ctx.status()[0] == 0
    cnt, off, lst = ctx.debug_bins()
    ctx.close()
    ref = o.render_opd(sc, "full")[0]
    err = np.abs(opd - ref)
    tol = 1e-5 + 1e-5 * np.abs(ref)
    assert np.all(err <= tol), f"seed {seed}: {np.count_nonzero(err > tol)} pixels out, max {err.max():.3e} at {np.unravel_index(err.argmax(), err.shape)}"
    Uref = o.field(ref, float(sc.lambda_um[0]), sc.pitch_um, sc.tilt_x_rad, sc.tilt_y_rad)
    assert np.abs(U - Uref).max() <= 1e-4, f"seed {seed}: field {np.abs(U - Uref).max():.3e}"
    oc, oo, ol = o.binning(sc, og.osog_tile_size())
    assert np.array_equal(off, oo) and np.array_equal(lst, ol)


@pytest.mark.parametrize("seed", range(0, 24, 3))
def test_random_scene_gbuffer_and_gradients(og, o, seed):
    """The same adversarial scenes through the widened calls: depth / instance-id maps (front-to-back ranking, explicit
    smallest-index rule) and all particle gradients from the one-pass gather, each at the bar of its own parity test."""
    import torch
    import test_gpu_gbuffer as G
    sc = G.with_heights(_scene(seed), seed=500 + seed)
    G.check(og, o, sc)
    rng = np.random.default_rng(seed)
    Gm = rng.standard_normal((sc.B, sc.H, sc.W)).astype(np.float32)
    ctx = og.Context(sc.H, sc.W, sc.N, max_frames=sc.B)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    gnp, gc, gpar = ctx.backward_particles(P, opt, torch.from_numpy(Gm).cuda())
    assert ctx.check_guards() == 0
    ctx.close()
    absG = np.abs(Gm)
    f64 = lambda t: t.cpu().numpy().astype(np.float64)
    ref, scale = o.backward_np(sc, Gm), o.backward_np(sc, absG)
    assert np.all(np.abs(f64(gnp) - ref) <= 2e-7 * scale + 1e-6)
    for got, fn in ((gc, o.backward_centre), (gpar, o.backward_params)):
        ref = fn(sc, Gm)
        big = np.maximum((np.abs(fn(sc, absG)) + np.abs(ref)).max(axis=1, keepdims=True), 1.0)
        assert np.all(np.abs(f64(got) - ref) <= 5e-7 * big), float((np.abs(f64(got) - ref) / big).max())
