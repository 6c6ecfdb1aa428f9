"""Seeded generators for the five BASELINE.json workloads.

Every draw is made in float64 from ``numpy.random.default_rng(seed)`` (PCG64) in the order
documented per config, then cast once to float32.  The float32 arrays ARE the scene: the
oracle promotes them to float64, the CUDA path reads them as they are.

Particle SoA ("Structure-of-Arrays ... dense tensor S in R^{N x D}"), one
array per column:
  cx, cy, cz          centre, um (cz is carried but unused: projection is along z)
  qw, qx, qy, qz      unit quaternion (Hamilton, body -> world)
  d0, d1, d2          kind 0 (ellipsoid): semi-axes a, b, c
                      kind 1 (capped tetragonal prism): side s, length L, cap height hc
  n_p                 refractive index of the particle
  kind                uint8, 0 or 1
  frame_start         int32 [B+1] CSR offsets of each frame's particles
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
import numpy as np

CONFIG_NAMES = {
    1: "cfg1_64_spheres_256",
    2: "cfg2_1k_ellipsoids_1024",
    3: "cfg3_10k_prisms_clumped_2048",
    4: "cfg4_40k_mixed_2048_oblique",
    5: "cfg5_16x5k_mixed_1024_noise",
}

_F32_COLS = ("cx", "cy", "cz", "qw", "qx", "qy", "qz", "d0", "d1", "d2", "n_p")


@dataclass
class Scene:
    name: str
    seed: int
    H: int
    W: int
    B: int
    pitch_um: float
    n_medium: float
    lambda_um: np.ndarray        # float64 [B]
    NA: np.ndarray               # float64 [B]
    tilt_x_rad: float = 0.0
    tilt_y_rad: float = 0.0
    read_noise_sigma: float = 0.0
    defocus_um: float = 0.0      # delta z of Eq. 3; 0 = in focus
    shot_noise_photons: float = 0.0   # photons at unit intensity for the Poisson term of PAPER.md:126; 0 = off
    topography_amplitude: float = 0.0   # relative amplitude of the micro-topography of PAPER.md:74; 0 = smooth bodies
    cols: dict = field(default_factory=dict)   # float32 [N] each + kind uint8 [N]
    frame_start: np.ndarray = None             # int32 [B+1]

    @property
    def N(self) -> int:
        return int(self.frame_start[-1])

    def __getattr__(self, key):
        cols = self.__dict__.get("cols", {})
        if key in cols:
            return cols[key]
        raise AttributeError(key)


def _quat(rng, n):
    """Uniform random rotation: 4 normals, normalised in float64 (order w, x, y, z)."""
    q = rng.standard_normal((n, 4))
    q /= np.sqrt((q * q).sum(axis=1, keepdims=True))
    return q


def _pack(name, seed, H, W, B, lam, NA, cols, frame_start, **kw):
    out = {}
    for k in _F32_COLS:
        out[k] = np.ascontiguousarray(np.asarray(cols[k], dtype=np.float64).astype(np.float32))
    out["kind"] = np.ascontiguousarray(np.asarray(cols["kind"], dtype=np.uint8))
    n = out["kind"].shape[0]
    for k in _F32_COLS:
        assert out[k].shape == (n,), (k, out[k].shape)
    return Scene(name=name, seed=seed, H=H, W=W, B=B, pitch_um=0.1, n_medium=1.33,
                 lambda_um=np.asarray(lam, dtype=np.float64).reshape(B),
                 NA=np.asarray(NA, dtype=np.float64).reshape(B),
                 cols=out, frame_start=np.asarray(frame_start, dtype=np.int32), **kw)


def _ellipsoid_cols(rng, n):
    """cfg 2 recipe: a, b, c ~ U[0.5, 4] i.i.d., q uniform, n_p ~ U[1.36, 1.50]."""
    abc = rng.uniform(0.5, 4.0, size=(n, 3))
    q = _quat(rng, n)
    n_p = rng.uniform(1.36, 1.50, size=n)
    return abc, q, n_p


def _prism_cols(rng, n):
    """cfg 3 recipe: s ~ U[1, 5], L = s * U[1, 3], hc = 0.5 s, q uniform, n_p ~ U[1.38, 1.45]."""
    s = rng.uniform(1.0, 5.0, size=n)
    L = s * rng.uniform(1.0, 3.0, size=n)
    hc = 0.5 * s
    q = _quat(rng, n)
    n_p = rng.uniform(1.38, 1.45, size=n)
    return np.stack([s, L, hc], axis=1), q, n_p


def _exact_half_kinds(rng, n):
    """Seeded random permutation of exactly n//2 ones (prisms) and n - n//2 zeros."""
    kind = np.zeros(n, dtype=np.uint8)
    kind[: n // 2] = 1
    return rng.permutation(kind)


def make_config(k: int, n_override: int | None = None) -> Scene:
    """Build BASELINE.json config k (1..5).  ``n_override`` shrinks N (per frame) for tests."""
    if k == 1:
        seed, n, H, W = 0, 64, 256, 256
        n = n_override or n
        rng = np.random.default_rng(seed)
        R = rng.uniform(1.0, 3.0, size=n)
        n_p = rng.uniform(1.38, 1.45, size=n)
        cx = rng.uniform(0.0, W * 0.1, size=n)
        cy = rng.uniform(0.0, H * 0.1, size=n)
        cols = dict(cx=cx, cy=cy, cz=np.zeros(n), qw=np.ones(n), qx=np.zeros(n), qy=np.zeros(n),
                    qz=np.zeros(n), d0=R, d1=R, d2=R, n_p=n_p, kind=np.zeros(n, np.uint8))
        return _pack(CONFIG_NAMES[1], seed, H, W, 1, [0.55], [0.4], cols, [0, n])
    if k == 2:
        seed, n, H, W = 1, 1000, 1024, 1024
        n = n_override or n
        rng = np.random.default_rng(seed)
        abc, q, n_p = _ellipsoid_cols(rng, n)
        cx = rng.uniform(0.0, W * 0.1, size=n)
        cy = rng.uniform(0.0, H * 0.1, size=n)
        cols = dict(cx=cx, cy=cy, cz=np.zeros(n), qw=q[:, 0], qx=q[:, 1], qy=q[:, 2], qz=q[:, 3],
                    d0=abc[:, 0], d1=abc[:, 1], d2=abc[:, 2], n_p=n_p, kind=np.zeros(n, np.uint8))
        return _pack(CONFIG_NAMES[2], seed, H, W, 1, [0.55], [0.4], cols, [0, n])
    if k == 3:
        seed, n, H, W = 2, 10000, 2048, 2048
        n = n_override or n
        rng = np.random.default_rng(seed)
        dims, q, n_p = _prism_cols(rng, n)
        clump_x = rng.uniform(0.0, W * 0.1, size=20)
        clump_y = rng.uniform(0.0, H * 0.1, size=20)
        which = rng.integers(0, 20, size=n)
        cx = clump_x[which] + rng.normal(0.0, 15.0, size=n)
        cy = clump_y[which] + rng.normal(0.0, 15.0, size=n)
        cols = dict(cx=cx, cy=cy, cz=np.zeros(n), qw=q[:, 0], qx=q[:, 1], qy=q[:, 2], qz=q[:, 3],
                    d0=dims[:, 0], d1=dims[:, 1], d2=dims[:, 2], n_p=n_p, kind=np.ones(n, np.uint8))
        return _pack(CONFIG_NAMES[3], seed, H, W, 1, [0.55], [0.4], cols, [0, n])
    if k == 4:
        seed, n, H, W = 3, 40000, 2048, 2048
        n = n_override or n
        rng = np.random.default_rng(seed)
        kind = _exact_half_kinds(rng, n)
        abc, qe, npe = _ellipsoid_cols(rng, n)          # drawn for all n, used where kind == 0
        dims, qp, npp = _prism_cols(rng, n)             # drawn for all n, used where kind == 1
        cx = rng.uniform(0.0, W * 0.1, size=n)
        cy = rng.uniform(0.0, H * 0.1, size=n)
        isp = kind.astype(bool)
        d = np.where(isp[:, None], dims, abc)
        q = np.where(isp[:, None], qp, qe)
        n_p = np.where(isp, npp, npe)
        cols = dict(cx=cx, cy=cy, cz=np.zeros(n), qw=q[:, 0], qx=q[:, 1], qy=q[:, 2], qz=q[:, 3],
                    d0=d[:, 0], d1=d[:, 1], d2=d[:, 2], n_p=n_p, kind=kind)
        return _pack(CONFIG_NAMES[4], seed, H, W, 1, [0.55], [0.65], cols, [0, n],
                     tilt_x_rad=float(np.deg2rad(10.0)))
    if k == 5:
        seed, n, H, W, B = 4, 5000, 1024, 1024, 16
        n = n_override or n
        rng = np.random.default_rng(seed)
        lam = rng.uniform(0.45, 0.65, size=B)
        NA = rng.uniform(0.3, 0.8, size=B)
        parts = []
        for _ in range(B):
            kind = _exact_half_kinds(rng, n)
            abc = np.clip(rng.lognormal(np.log(2.0), 0.5, size=(n, 3)), 0.25, 8.0)
            s = np.clip(rng.lognormal(np.log(2.0), 0.5, size=n), 0.25, 8.0)
            L = s * rng.uniform(1.0, 3.0, size=n)
            dims = np.stack([s, L, 0.5 * s], axis=1)
            q = _quat(rng, n)
            n_p = rng.uniform(1.36, 1.50, size=n)
            cx = rng.uniform(0.0, W * 0.1, size=n)
            cy = rng.uniform(0.0, H * 0.1, size=n)
            d = np.where(kind.astype(bool)[:, None], dims, abc)
            parts.append(dict(cx=cx, cy=cy, cz=np.zeros(n), qw=q[:, 0], qx=q[:, 1], qy=q[:, 2],
                              qz=q[:, 3], d0=d[:, 0], d1=d[:, 1], d2=d[:, 2], n_p=n_p, kind=kind))
        cols = {k2: np.concatenate([p[k2] for p in parts]) for k2 in parts[0]}
        return _pack(CONFIG_NAMES[5], seed, H, W, B, lam, NA, cols,
                     np.arange(B + 1, dtype=np.int64) * n, read_noise_sigma=0.01)
    raise ValueError(f"unknown config {k}")


def make_scene(name, H, W, cols, *, lam=0.55, NA=0.4, seed=0, frame_start=None, **kw) -> Scene:
    """Hand-built scene for closed-form / edge-case tests.  ``cols`` maps the SoA names above to
    sequences; missing quaternion defaults to identity, cz to 0, kind to 0."""
    n = len(cols["cx"])
    full = dict(cz=np.zeros(n), qw=np.ones(n), qx=np.zeros(n), qy=np.zeros(n), qz=np.zeros(n),
                kind=np.zeros(n, np.uint8))
    full.update(cols)
    if frame_start is None:
        frame_start = [0, n]
    B = len(frame_start) - 1
    lam = np.broadcast_to(np.asarray(lam, dtype=np.float64), (B,)).copy()
    NA = np.broadcast_to(np.asarray(NA, dtype=np.float64), (B,)).copy()
    return _pack(name, seed, H, W, B, lam, NA, full, frame_start, **kw)


def subset(scene: Scene, idx) -> Scene:
    """Single-frame scene holding particles ``idx`` (in that order) of a single-frame scene."""
    assert scene.B == 1
    idx = np.asarray(idx, dtype=np.int64)
    cols = {k: np.ascontiguousarray(v[idx]) for k, v in scene.cols.items()}
    return replace(scene, cols=cols, frame_start=np.asarray([0, idx.size], dtype=np.int32))
