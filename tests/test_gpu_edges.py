"""GPU edge cases through the C ABI: empty input, ragged frames, off-frame and invalid particles, tile lists
longer than their staging slice (ordered re-scan), one hot tile on a large frame, pair-list overflow, vertical prism faces (fp64 path), batches with
per-frame optics (more than one optics chunk), y tilt, all-pass pupil (Parseval), and argument errors."""
import ctypes as C

import numpy as np
import pytest

from workloads import make_config, make_scene
from test_gpu_parity import check_against_oracle, render_all, og, o  # noqa: F401  (fixtures)

pytestmark = pytest.mark.gpu


def _mixed(n, H, W, seed, spread=1.0, B=1):
    rng = np.random.default_rng(seed)
    q = rng.standard_normal((n, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    kind = (rng.uniform(size=n) < 0.5).astype(np.uint8)
    s = rng.uniform(0.4, 2.5, n)
    d = np.where(kind[:, None] == 1, np.stack([s, s * rng.uniform(1, 3, n), 0.5 * s], 1), rng.uniform(0.3, 3.0, (n, 3)))
    return dict(cx=rng.uniform(-1.0, W * 0.1 * spread + 1.0, n), cy=rng.uniform(-1.0, H * 0.1 * spread + 1.0, n),
                qw=q[:, 0], qx=q[:, 1], qy=q[:, 2], qz=q[:, 3], d0=d[:, 0], d1=d[:, 1], d2=d[:, 2],
                n_p=rng.uniform(1.36, 1.5, n), kind=kind)


def test_zero_particles_uniform_field_and_intensity(og, o):
    sc = make_scene("empty", 96, 128, dict(cx=[], cy=[], d0=[], d1=[], d2=[], n_p=[]))
    g = render_all(og, sc)
    assert np.all(g["opd"] == 0.0)
    assert np.all(g["field"] == 1.0 + 0.0j)
    assert np.abs(g["intensity"] - 1.0).max() <= 1e-6          # P9: N = 0, no ramp -> I == 1
    assert g["bins"][2].size == 0 and g["status"] == (0, 0, 0)


@pytest.mark.parametrize("H,W", [(70, 50), (33, 97), (1, 5), (130, 4)])
def test_ragged_frames_and_off_frame_particles(og, o, H, W):
    sc = make_scene("ragged", H, W, _mixed(40, H, W, seed=H * 1000 + W), tilt_x_rad=0.05, tilt_y_rad=-0.03)
    check_against_oracle(og, o, sc)


def test_invalid_particles_are_skipped_and_reported(og, o):
    cols = _mixed(30, 64, 64, seed=5)
    cols["d1"][3] = -1.0
    cols["cx"][7] = np.nan
    cols["qy"][11] = np.inf
    cols["kind"][13] = 7
    cols["d0"][17] = 0.0
    sc = make_scene("bad", 64, 64, cols)
    g, _ = check_against_oracle(og, o, sc)
    assert g["status"][1] & og.OSOG_WBADPARTICLE


@pytest.mark.parametrize("n,longest", [(2600, 2048), (900, 600), (1100, 1024)])
def test_list_longer_than_shared_sort_capacity(og, o, n, longest):
    """n small spheres inside one 32 x 32 tile: lists beyond the staging slice (1,024 entries here) are rebuilt in order
    from the particles' tile ranges; shorter crowded lists take many rank-sort passes per lane; all are composed in many batches."""
    rng = np.random.default_rng(11)
    cols = dict(cx=rng.uniform(3.3, 6.2, n), cy=rng.uniform(3.3, 6.2, n), d0=np.full(n, 0.12), d1=np.full(n, 0.12),
                d2=np.full(n, 0.12), n_p=rng.uniform(1.36, 1.5, n))
    sc = make_scene("crowd", 96, 96, cols)
    g, _ = check_against_oracle(og, o, sc)
    assert g["bins"][0].max() > longest


def test_pair_list_overflow_is_reported_and_frames_zeroed(og):
    """max_pairs is the TOTAL capacity of the tile lists (CSR list of the device scan): a call that needs more sets
    OSOG_WOVERFLOW, zero-fills its frames and reports the exact number of pairs that would have sufficed."""
    sc = make_config(2, n_override=300)
    ctx = og.Context(sc.H, sc.W, sc.N, max_pairs=50, check=False)
    P = og.Particles.from_scene(sc)
    opt = og.optics_from_scene(sc)
    opd = ctx.render_opd(P, opt)
    r, bits, pairs = ctx.status()
    assert r == og.OSOG_ECAPACITY and (bits & og.OSOG_WOVERFLOW) and pairs > 50
    assert float(opd.abs().max()) == 0.0
    ctx.close()
    ctx = og.Context(sc.H, sc.W, sc.N, max_pairs=pairs)      # the reported need is exactly enough
    ctx.render_opd(P, opt)
    assert ctx.status()[0] == 0
    cnt = ctx.debug_bins()[0]
    assert int(cnt.sum()) == pairs == ctx.status()[2]
    ctx.close()
    ctx = og.Context(sc.H, sc.W, sc.N, max_pairs=pairs - 1, check=False)   # one entry less is not
    ctx.render_opd(P, opt)
    assert ctx.status()[0] == og.OSOG_ECAPACITY
    assert ctx.check_guards() == 0                           # an overflowing call writes nothing past its (too small) list
    ctx.close()


def test_overflow_raises_through_the_binding(og):
    """The Python methods check the device status by default: an overflowing call raises instead of handing back zeros."""
    sc = make_config(2, n_override=300)
    ctx = og.Context(sc.H, sc.W, sc.N, max_pairs=50)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    for call in (ctx.render_opd, ctx.render_field, ctx.render_intensity):
        with pytest.raises(og.OsogError) as e:
            call(P, opt)
        assert e.value.code == og.OSOG_ECAPACITY and e.value.pairs_needed > 50
    ctx.close()
    ctx = og.Context(sc.H, sc.W, sc.N, max_pairs=e.value.pairs_needed)
    assert float(ctx.render_opd(P, opt).max()) > 0.0
    ctx.close()


def test_one_hot_tile_on_a_large_frame_with_default_sizing(og, o):
    """3,000 sub-pixel-to-small spheres inside one 32 x 32 tile of a 2048 x 2048 frame, context sized by default
    (max_pairs = 64 N + 1024 in total): one crowded tile must not fail the call although its list is far longer than a
    tile's staging slice.  Bins (offsets from the device scan) bit-exact, OPD / field / intensity at the bars."""
    n = 3000
    rng = np.random.default_rng(21)
    x0, y0 = 40 * 3.2 + 0.4, 17 * 3.2 + 0.4                   # inside tile (40, 17): 3.2 um = 32 pixels
    cols = dict(cx=rng.uniform(x0, x0 + 2.4, n), cy=rng.uniform(y0, y0 + 2.4, n), d0=np.full(n, 0.08), d1=np.full(n, 0.08),
                d2=np.full(n, 0.08), n_p=rng.uniform(1.36, 1.5, n))
    sc = make_scene("hot_tile", 2048, 2048, cols)
    g, _ = check_against_oracle(og, o, sc)
    cnt = g["bins"][0]
    assert cnt.max() == n and cnt.sum() == n and g["status"] == (0, 0, n)


def test_crowded_tiles_in_a_batch_take_the_ordered_rescan(og, o):
    """Lists longer than their staging slice in several tiles of several frames (frame-relative particle ranges of the
    re-scan, both warps of a tile meeting in the middle, odd list lengths)."""
    H = W = 96
    B, per = 3, 1500
    rng = np.random.default_rng(5)
    parts = []
    for b in range(B):
        parts.append(dict(cx=rng.uniform(2.0 + b, 5.5 + b, per), cy=rng.uniform(2.5, 7.0, per), d0=np.full(per, 0.1),
                          d1=np.full(per, 0.15), d2=np.full(per, 0.12), n_p=rng.uniform(1.36, 1.5, per)))
    cols = {k: np.concatenate([p[k] for p in parts]) for k in parts[0]}
    sc = make_scene("crowd_batch", H, W, cols, frame_start=np.arange(B + 1) * per, lam=np.full(B, 0.55), NA=np.full(B, 0.5))
    g = render_all(og, sc, max_pairs=3 * 4500)
    assert g["guards"] == 0                # staging slices of 500 entries per tile, the fullest lists are longer
    assert g["status"][0] == 0
    oc, oo, ol = o.binning(sc, og.osog_tile_size())
    cnt, off, lst = g["bins"]
    assert cnt.max() > 500 and np.array_equal(off, oo) and np.array_equal(lst, ol)
    ref = o.render_opd(sc)
    assert np.all(np.abs(g["opd"] - ref) <= 1e-5 + 1e-5 * np.abs(ref))


def test_recompose_refused_after_a_call_that_left_no_sorted_lists(og):
    """osog_debug_recompose_field composes from the sorted lists of the last field-capable call: after any other call
    (atomic variant, labels, gradients) it must refuse rather than compose from stale or unsorted lists."""
    import torch
    sc = make_config(2, n_override=200)
    ctx = og.Context(sc.H, sc.W, sc.N)
    P, opt = og.Particles.from_scene(sc), og.optics_from_scene(sc)
    buf = torch.empty((1, sc.H, sc.W, 2), dtype=torch.float32, device="cuda")
    ctx.render_field(P, opt)
    ctx.recompose_field(buf)
    for other in (ctx.render_opd_atomic, ctx.render_opd_smem_atomic, ctx.particle_obbs):
        ctx.render_field(P, opt)
        other(P, opt)
        with pytest.raises(og.OsogError) as e:
            ctx.recompose_field(buf)
        assert e.value.code == og.OSOG_EINVAL
    ctx.close()


def test_prisms_with_vertical_faces_take_the_fp64_path(og, o):
    """Identity and 90-degree rotations give face normals with n_z == 0 exactly (thickness is discontinuous at those
    faces); centres are placed so that no pixel centre lies within 1e-3 um of a vertical face."""
    r = np.sqrt(0.5)
    cols = dict(cx=[3.213, 9.047, 6.131], cy=[3.377, 4.021, 9.563], qw=[1.0, r, r], qx=[0.0, r, 0.0], qy=[0.0, 0.0, r],
                qz=[0.0, 0.0, 0.0], d0=[2.03, 1.57, 1.21], d1=[3.3, 4.1, 2.9], d2=[1.0, 0.8, 0.6], n_p=[1.45, 1.40, 1.42],
                kind=np.ones(3, np.uint8))
    check_against_oracle(og, o, make_scene("vertical", 128, 128, cols))


def test_batch_with_per_frame_optics_across_optics_chunks(og, o):
    B, n = 19, 60                                             # 19 frames > one 16-frame optics chunk
    rng = np.random.default_rng(3)
    parts = [_mixed(n, 64, 96, seed=100 + b) for b in range(B)]
    cols = {k: np.concatenate([p[k] for p in parts]) for k in parts[0]}
    sc = make_scene("batch", 64, 96, cols, lam=rng.uniform(0.45, 0.65, B), NA=rng.uniform(0.3, 0.8, B), seed=77,
                    frame_start=np.arange(B + 1) * n, tilt_x_rad=0.1, read_noise_sigma=0.01)
    check_against_oracle(og, o, sc)


def test_partial_batch_uses_the_single_frame_plan(og, o):
    sc = make_config(5, n_override=200)
    import paper_2606_21381_b200 as m
    ctx = m.Context(sc.H, sc.W, sc.N, max_frames=sc.B + 3)
    P = m.Particles.from_scene(sc)
    I = ctx.render_intensity(P, m.optics_from_scene(sc)).cpu().numpy().astype(np.float64)
    Iref = o.render_intensity(sc)
    assert np.abs(I - Iref).max() <= 1e-4 * Iref.mean()
    ctx.close()


def test_all_pass_pupil_conserves_energy(og, o):
    sc = make_config(2, n_override=200)
    g, _ = check_against_oracle(og, o, sc, pupil=False, what=("field", "intensity"))
    assert abs(g["intensity"].sum() / (sc.H * sc.W) - 1.0) < 1e-5      # P11: sum |U|^2 = H W for |U| = 1


def test_argument_errors(og):
    sc = make_config(1)
    ctx = og.Context(sc.H, sc.W, 10)                          # max_particles 10 < 64
    P = og.Particles.from_scene(sc)
    opt = og.optics_from_scene(sc)
    with pytest.raises(og.OsogError) as e:
        ctx.render_opd(P, opt)
    assert e.value.code == og.OSOG_EINVAL
    ctx.close()
    ctx = og.Context(sc.H, sc.W, sc.N)
    bad = og.make_optics(1, -0.1, 1.33, 0.55, 0.4)
    with pytest.raises(og.OsogError):
        ctx.render_opd(P, bad)
    two = og.make_optics(2, 0.1, 1.33, 0.55, 0.4)             # B > max_frames
    with pytest.raises(og.OsogError):
        ctx.render_opd(P, two)
    assert og.lib().osog_render_opd(ctx._ctx, C.byref(P.c), P.N, C.byref(opt), None) == og.OSOG_EINVAL
    ctx.close()


def test_context_reuse_keeps_scratch_invariants(og, o):
    """The tile counters and the status slot are kept clean by the kernels themselves (no memset per call): a context
    reused across different scenes, after the atomic variant and after an overflowing call, must give the same bits
    as a fresh context."""
    import torch
    big = make_config(2, n_override=400)
    small = make_scene("reuse", big.H, big.W, _mixed(50, big.H, big.W, seed=9))
    fresh = og.Context(big.H, big.W, 400)
    ref_small = fresh.render_opd(og.Particles.from_scene(small), og.optics_from_scene(small)).clone()
    ref_big = fresh.render_opd(og.Particles.from_scene(big), og.optics_from_scene(big)).clone()
    fresh.close()
    ctx = og.Context(big.H, big.W, 400, max_pairs=40 * 1024)     # 40 entries per tile
    Pb, Ps = og.Particles.from_scene(big), og.Particles.from_scene(small)
    ob, os_ = og.optics_from_scene(big), og.optics_from_scene(small)
    ctx.render_opd_atomic(Pb, ob)
    assert torch.equal(ctx.render_opd(Ps, os_), ref_small)
    assert ctx.status() == (0, 0, ctx.status()[2])
    tiny = og.Context(big.H, big.W, 400, max_pairs=10, check=False)
    tiny.render_opd(Pb, ob)
    assert tiny.status()[0] == og.OSOG_ECAPACITY
    out = tiny.render_opd(og.Particles.from_scene(make_scene("one", big.H, big.W, dict(cx=[5.0], cy=[5.0], d0=[1.0], d1=[1.0], d2=[1.0], n_p=[1.4]))),
                          os_)
    assert tiny.status()[0] == 0 and float(out.max()) > 0.0        # the overflow bit does not stick to the next call
    tiny.close()
    assert torch.equal(ctx.render_opd(Pb, ob), ref_big)
    cnt, off, lst = ctx.debug_bins()
    oc, oo, ol = o.binning(big, og.osog_tile_size())
    assert np.array_equal(off, oo) and np.array_equal(lst, ol)
    assert torch.equal(ctx.render_opd(Ps, os_), ref_small)
    assert ctx.check_guards() == 0
    ctx.close()


def test_context_reuse_with_changing_batch_size(og):
    """The per-tile counters are double-buffered and each call clears the other slot for the next one: a small batch
    between two large ones must not leave stale counts in the tiles it did not use (same bits as fresh contexts)."""
    import torch
    H = W = 160
    scenes = [make_scene(f"b{B}", H, W, _mixed(30 * B, H, W, seed=100 + B), frame_start=[30 * k for k in range(B + 1)],
                         lam=np.full(B, 0.55), NA=np.full(B, 0.5)) for B in (4, 1, 3, 4, 2, 4)]
    ctx = og.Context(H, W, 120, max_frames=4)
    for sc in scenes:
        fresh = og.Context(H, W, 120, max_frames=4)
        want = fresh.render_opd(og.Particles.from_scene(sc), og.optics_from_scene(sc)).clone()
        fresh.close()
        got = ctx.render_opd(og.Particles.from_scene(sc), og.optics_from_scene(sc))
        assert ctx.status()[0] == 0
        assert torch.equal(got, want), sc.name
    assert ctx.check_guards() == 0
    ctx.close()


def test_batch_with_unequal_and_empty_frames(og, o):
    """Frames of 0, 57, 5 and 130 particles in one call: every frame equals the single-frame render of its own particles
    (same bits), the empty frame is the particle-free frame, bins / OPD / field / intensity / depth maps match the oracle."""
    import torch
    from workloads import subset
    H = W = 128
    counts = [0, 57, 5, 130]
    fs = np.concatenate([[0], np.cumsum(counts)])
    cols = _mixed(int(fs[-1]), H, W, seed=77)
    B = len(counts)
    sc = make_scene("uneven", H, W, cols, frame_start=fs, lam=np.array([0.5, 0.55, 0.6, 0.45]), NA=np.array([0.4, 0.5, 0.6, 0.7]),
                    tilt_x_rad=0.07)
    g, _ = check_against_oracle(og, o, sc)
    assert np.all(g["opd"][0] == 0.0) and np.allclose(np.abs(g["field"][0]), 1.0, atol=1e-6)
    ctx = og.Context(H, W, sc.N, max_frames=B)
    tid, dep = ctx.render_gbuffer(og.Particles.from_scene(sc), og.optics_from_scene(sc))
    rid, rdep = o.render_gbuffer(sc)
    from test_gpu_gbuffer import ids_valid
    ids_valid(o, sc, tid.cpu().numpy(), rid)          # per-pixel validity of any differing owner, no rate
    assert np.all(tid.cpu().numpy()[0] == -1)
    assert np.all(np.abs(dep.cpu().numpy() - rdep) <= 1e-6 + 2e-7 * np.abs(rdep))
    batch = ctx.render_opd(og.Particles.from_scene(sc), og.optics_from_scene(sc)).clone()
    ctx.close()
    one = og.Context(H, W, sc.N)
    for b in range(1, B):
        sub = make_scene("one", H, W, {k: v[fs[b]:fs[b + 1]] for k, v in sc.cols.items()}, lam=sc.lambda_um[b], NA=sc.NA[b],
                         tilt_x_rad=0.07)
        assert torch.equal(one.render_opd(og.Particles.from_scene(sub), og.optics_from_scene(sub))[0], batch[b])
    one.close()
