"""OSOG forward-render ORACLE, Python side (test infrastructure, NOT the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It shares nothing with paper_2606_21381_b200/ (no kernels, headers, helpers, tables).

Pieces, each following the passage it cites (line numbers are /root/reference/PAPER.md):
  render_opd      float64 loop over pixels x particles in C (oracle/osog_oracle.c)   Eq. 1, 2, 7
  field           U = exp(i 2 pi (OPD/lambda + fx0 x + fy0 y))                        Eq. 2 (A == 1), :113-115
  pupil_mask      circ(|k| / k_NA) on the FFT grid, integer comparison                Eq. 3 (delta z = 0)
  intensity       I = | IFFT2( FFT2(U) * P ) |^2                                      :90, :99
  defocus_factor  exp(i dz sqrt(k0^2 - kx^2 - ky^2)) on the FFT grid                  Eq. 3 (delta z != 0), A20
  pupil_function  P = circ(.) * defocus factor                                        Eq. 3
  dic_image       | U(r+ds) e^{i theta} - U(r-ds) e^{-i theta} |^2 * |h_obj|^2         Eq. 5 (:101-104), A21, A22
  philox4x32_10   counter-based RNG, written from its published description
  read_noise      z ~ N(0,1) per (seed, frame, pixel) by Box-Muller                   :126 (Gaussian term)
  binning         bounding boxes -> tiles -> counts / offsets / ascending lists       DESIGN.md section 3 (B1-B4)
  particle_obbs   oriented bounding box of each silhouette (detector labels)          :76, :138-146, A23
  render_gbuffer  depth map and instance-id map (top-most particle per pixel), in C   :76, A24
  backward_np     dL/dn_p = sum_px G t_n: adjoint of the OPD sum in the indices, in C   :124 (NEXT-3, first step)
  backward_intensity   dL/dOPD from dL/dI: adjoint of field + pupil + |.|^2                :124 (NEXT-3)
  thickness_grad / backward_centre   grad t per pixel; dL/d(cx, cy) = -dn sum_px G grad t  :124 (NEXT-3, second step)
  thickness_param_grad / backward_params   dt/d(dims, quaternion); dL/d(dims, q) = dn sum_px G dt/dtheta   :124 (NEXT-3, third step)
  spectral_loss / spectral_loss_grad   Eq. 8 and its gradient in the image                   :168, A28
  render_height / height_gradient / height_laplacian   h, grad h, lap h of the G-buffer :76, :92, :96-99, A25
  fresnel_transmittance / brightfield_amplitude / render_brightfield   Eq. 4       :94-99, A27
  shot_uniforms / poisson_counts / shot_noise          Poisson shot noise          :126, A26
  topography_factor                                    micro-topography of the height map :74, A29

Every reading of the paper taken here (units, pixel centres, quaternion convention, pupil edge,
FFT normalisation, noise model ...) is listed in DESIGN.md section 3.  Pins: tests/test_oracle_*.py.
"""
from __future__ import annotations

import ctypes
import math
import os

import numpy as np

from . import build as _build

_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        path = _build.build()
        lib = ctypes.CDLL(path)
        fp = ctypes.POINTER(ctypes.c_float)
        u8p = ctypes.POINTER(ctypes.c_uint8)
        dp = ctypes.POINTER(ctypes.c_double)
        lib.osog_oracle_render_opd.argtypes = [ctypes.c_int64] + [fp] * 10 + [u8p] + [
            ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, dp]
        lib.osog_oracle_render_opd.restype = None
        lib.osog_oracle_count_covered.argtypes = [ctypes.c_int64] + [fp] * 10 + [u8p] + [
            ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.POINTER(ctypes.c_int64)]
        lib.osog_oracle_count_covered.restype = None
        lib.osog_oracle_render_gbuffer.argtypes = [ctypes.c_int64] + [fp] * 11 + [u8p] + [
            ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.POINTER(ctypes.c_int32), dp, dp]
        lib.osog_oracle_render_gbuffer.restype = None
        lib.osog_oracle_top_slope.argtypes = [ctypes.c_uint8, dp, dp, ctypes.c_double, ctypes.c_double, dp]
        lib.osog_oracle_top_slope.restype = ctypes.c_int
        lib.osog_oracle_chord.argtypes = [ctypes.c_uint8, dp, dp, ctypes.c_double, ctypes.c_double, dp, dp]
        lib.osog_oracle_chord.restype = ctypes.c_int
        lib.osog_oracle_backward_np.argtypes = [ctypes.c_int64] + [fp] * 10 + [u8p] + [
            ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int, fp, dp]
        lib.osog_oracle_backward_np.restype = None
        lib.osog_oracle_backward_centre.argtypes = [ctypes.c_int64] + [fp] * 10 + [u8p] + [
            ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, fp, dp]
        lib.osog_oracle_backward_centre.restype = None
        lib.osog_oracle_thickness_grad.argtypes = [ctypes.c_uint8, dp, dp, ctypes.c_double, ctypes.c_double, dp]
        lib.osog_oracle_thickness_grad.restype = None
        lib.osog_oracle_thickness_param_grad.argtypes = [ctypes.c_uint8, dp, dp, ctypes.c_double, ctypes.c_double, dp]
        lib.osog_oracle_thickness_param_grad.restype = None
        lib.osog_oracle_backward_params.argtypes = [ctypes.c_int64] + [fp] * 10 + [u8p] + [
            ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, fp, dp]
        lib.osog_oracle_backward_params.restype = None
        lib.osog_oracle_thickness.argtypes = [ctypes.c_uint8, dp, dp, ctypes.c_double, ctypes.c_double]
        lib.osog_oracle_thickness.restype = ctypes.c_double
        lib.osog_oracle_circumradius.argtypes = [ctypes.c_uint8] + [ctypes.c_float] * 3
        lib.osog_oracle_circumradius.restype = ctypes.c_double
        lib.osog_oracle_rot_from_quat.argtypes = [dp, dp]
        lib.osog_oracle_rot_from_quat.restype = None
        lib.osog_oracle_prism_planes.argtypes = [ctypes.c_double] * 3 + [dp, dp]
        lib.osog_oracle_prism_planes.restype = ctypes.c_int
        _LIB = lib
    return _LIB


_COLS = ("cx", "cy", "qw", "qx", "qy", "qz", "d0", "d1", "d2", "n_p")


def _ptr(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


# --------------------------------------------------------------------------------------------
# geometry (C)
# --------------------------------------------------------------------------------------------
def rot_from_quat(q) -> np.ndarray:
    """R(q), q = (w, x, y, z) Hamilton, active body->world; no renormalisation (reading A4)."""
    q = np.ascontiguousarray(q, dtype=np.float64)
    R = np.empty(9, dtype=np.float64)
    _lib().osog_oracle_rot_from_quat(_ptr(q, ctypes.c_double), _ptr(R, ctypes.c_double))
    return R.reshape(3, 3)


def prism_planes(s, L, hc):
    """Body-frame (A[12,3], b[12]) of the capped tetragonal prism, Eq. 1 form A x <= b."""
    A = np.zeros((16, 3), dtype=np.float64)
    b = np.zeros(16, dtype=np.float64)
    m = _lib().osog_oracle_prism_planes(float(s), float(L), float(hc), _ptr(A, ctypes.c_double), _ptr(b, ctypes.c_double))
    return A[:m].copy(), b[:m].copy()


def thickness(kind, q, dims, dx, dy, f32=False) -> float:
    """Chord length along z of one particle at offset (dx, dy) from its centre.  With f32=True q and dims
    are first rounded to float32, as the renderer sees them (the scene is float32)."""
    q = np.asarray(q, dtype=np.float64)
    d = np.asarray(dims, dtype=np.float64)
    if f32:
        q = q.astype(np.float32).astype(np.float64)
        d = d.astype(np.float32).astype(np.float64)
    q = np.ascontiguousarray(q)
    d = np.ascontiguousarray(d)
    return _lib().osog_oracle_thickness(int(kind), _ptr(q, ctypes.c_double), _ptr(d, ctypes.c_double),
                                        float(dx), float(dy))


def circumradius(kind, dims) -> float:
    d = np.asarray(dims, dtype=np.float32)
    return _lib().osog_oracle_circumradius(int(kind), float(d[0]), float(d[1]), float(d[2]))


def render_opd_frame(cols, lo, hi, H, W, pitch, n_medium, mode="bcircle") -> np.ndarray:
    """OPD [H, W] float64 of particles lo..hi-1 of the SoA `cols` (dict of float32 arrays + kind)."""
    out = np.empty((H, W), dtype=np.float64)
    arrs = [np.ascontiguousarray(cols[k][lo:hi], dtype=np.float32) for k in _COLS]
    kind = np.ascontiguousarray(cols["kind"][lo:hi], dtype=np.uint8)
    a = {k: v for k, v in zip(_COLS, arrs)}
    f = ctypes.c_float
    _lib().osog_oracle_render_opd(
        hi - lo, _ptr(a["cx"], f), _ptr(a["cy"], f), _ptr(a["qw"], f), _ptr(a["qx"], f), _ptr(a["qy"], f),
        _ptr(a["qz"], f), _ptr(a["d0"], f), _ptr(a["d1"], f), _ptr(a["d2"], f), _ptr(a["n_p"], f),
        _ptr(kind, ctypes.c_uint8), H, W, float(pitch), float(n_medium),
        {"full": 0, "bcircle": 1}[mode], _ptr(out, ctypes.c_double))
    return out


def chord(kind, q, dims, dx, dy):
    """(z_enter, z_exit) of the vertical line through the body relative to its centre, or None (no positive chord)."""
    R = np.ascontiguousarray(rot_from_quat(q), dtype=np.float64).reshape(9)
    d = np.ascontiguousarray(dims, dtype=np.float64)
    ze, zx = ctypes.c_double(0.0), ctypes.c_double(0.0)
    ok = _lib().osog_oracle_chord(int(kind), _ptr(R, ctypes.c_double), _ptr(d, ctypes.c_double), float(dx), float(dy),
                                  ctypes.byref(ze), ctypes.byref(zx))
    return (ze.value, zx.value) if ok else None


def top_slope(kind, q, dims, dx, dy):
    """(dz/dx, dz/dy) of the body's top surface at the offset (dx, dy) from its centre, or None (no positive chord)."""
    R = np.ascontiguousarray(rot_from_quat(q), dtype=np.float64).reshape(9)
    d = np.ascontiguousarray(dims, dtype=np.float64)
    g = np.zeros(2, dtype=np.float64)
    ok = _lib().osog_oracle_top_slope(int(kind), _ptr(R, ctypes.c_double), _ptr(d, ctypes.c_double), float(dx), float(dy),
                                      _ptr(g, ctypes.c_double))
    return (float(g[0]), float(g[1])) if ok else None


def render_gbuffer(scene, mode="bcircle", normals=False):
    """(top_id int32 [B, H, W], depth float64 [B, H, W]) of a workloads.Scene: index (within the frame's particles,
    i.e. relative to frame_start[b]) and top-surface height of the top-most particle above every pixel (reading A24).
    normals=True adds the slope map float64 [B, H, W, 2] = (dz/dx, dz/dy) of the owner's top surface (0 where none): the
    analytic height gradient of the visible surface, whose normal is <-dz/dx, -dz/dy, 1>."""
    fs = scene.frame_start
    f = ctypes.c_float
    ids, deps, nrm = [], [], []
    for b in range(scene.B):
        lo, hi = int(fs[b]), int(fs[b + 1])
        a = {k: np.ascontiguousarray(scene.cols[k][lo:hi], dtype=np.float32) for k in _COLS + ("cz",)}
        kind = np.ascontiguousarray(scene.cols["kind"][lo:hi], dtype=np.uint8)
        tid = np.empty((scene.H, scene.W), dtype=np.int32)
        dep = np.empty((scene.H, scene.W), dtype=np.float64)
        nm = np.zeros((scene.H, scene.W, 2), dtype=np.float64) if normals else None
        _lib().osog_oracle_render_gbuffer(
            hi - lo, _ptr(a["cx"], f), _ptr(a["cy"], f), _ptr(a["cz"], f), _ptr(a["qw"], f), _ptr(a["qx"], f),
            _ptr(a["qy"], f), _ptr(a["qz"], f), _ptr(a["d0"], f), _ptr(a["d1"], f), _ptr(a["d2"], f), _ptr(a["n_p"], f),
            _ptr(kind, ctypes.c_uint8), scene.H, scene.W, float(scene.pitch_um),
            {"full": 0, "bcircle": 1}[mode], _ptr(tid, ctypes.c_int32), _ptr(dep, ctypes.c_double),
            _ptr(nm, ctypes.c_double) if normals else None)
        ids.append(tid)
        deps.append(dep)
        nrm.append(nm)
    if normals:
        return np.stack(ids), np.stack(deps), np.stack(nrm)
    return np.stack(ids), np.stack(deps)


def backward_np(scene, G, mode="bcircle") -> np.ndarray:
    """dL/dn_p [N] float64 for an upstream gradient G = dL/dOPD (float32 [B, H, W]): sum over the particle's frame of
    G * thickness (the OPD sum is linear in n_p)."""
    fs = scene.frame_start
    f = ctypes.c_float
    out = np.zeros(scene.N, dtype=np.float64)
    G = np.ascontiguousarray(G, dtype=np.float32)
    for b in range(scene.B):
        lo, hi = int(fs[b]), int(fs[b + 1])
        if hi == lo:
            continue
        a = {k: np.ascontiguousarray(scene.cols[k][lo:hi], dtype=np.float32) for k in _COLS}
        kind = np.ascontiguousarray(scene.cols["kind"][lo:hi], dtype=np.uint8)
        g = np.zeros(hi - lo, dtype=np.float64)
        Gb = np.ascontiguousarray(G[b])
        _lib().osog_oracle_backward_np(
            hi - lo, _ptr(a["cx"], f), _ptr(a["cy"], f), _ptr(a["qw"], f), _ptr(a["qx"], f), _ptr(a["qy"], f),
            _ptr(a["qz"], f), _ptr(a["d0"], f), _ptr(a["d1"], f), _ptr(a["d2"], f), _ptr(a["n_p"], f),
            _ptr(kind, ctypes.c_uint8), scene.H, scene.W, float(scene.pitch_um),
            {"full": 0, "bcircle": 1}[mode], _ptr(Gb, f), _ptr(g, ctypes.c_double))
        out[lo:hi] = g
    return out


def backward_intensity(scene, G_I, U=None, pupil_enabled=True, mode="bcircle") -> np.ndarray:
    """Adjoint of the optics stage: for an upstream gradient G_I = dL/dI (real,
    [B, H, W]) of the coherent intensity I = |V|^2, V = U * h_obj = ifft2(fft2(U) P), U = exp(i 2 pi OPD / lambda) ramp,
    returns dL/dOPD [B, H, W] float64:
        g_V = G_I V                      (dL = 2 Re sum conj(g_V) dV)
        g_U = ifft2(conj(P) fft2(g_V))   (adjoint of the linear map U -> V)
        dL/dOPD = (4 pi / lambda) Im(g_U conj(U))      (dU = i (2 pi / lambda) U dOPD)
    The additive read noise has no gradient."""
    if U is None:
        U = render_field(scene, mode=mode)
    dz = float(getattr(scene, "defocus_um", 0.0))
    out = []
    for b in range(scene.B):
        lam = float(scene.lambda_um[b])
        P = pupil_function(scene.H, scene.W, float(scene.NA[b]), scene.pitch_um, lam, scene.n_medium, dz, pupil_enabled)
        V = np.fft.ifft2(np.fft.fft2(U[b]) * P)
        gV = np.asarray(G_I[b], dtype=np.float64) * V
        gU = np.fft.ifft2(np.conj(P) * np.fft.fft2(gV))
        out.append((4.0 * np.pi / lam) * np.imag(gU * np.conj(U[b])))
    return np.stack(out)


def thickness_grad(kind, q, dims, dx, dy):
    """(dt/dx, dt/dy) of one particle's thickness at the offset (dx, dy) from its centre (0 where the chord is empty)."""
    R = np.ascontiguousarray(rot_from_quat(q), dtype=np.float64).reshape(9)
    d = np.ascontiguousarray(dims, dtype=np.float64)
    g = np.zeros(2, dtype=np.float64)
    _lib().osog_oracle_thickness_grad(int(kind), _ptr(R, ctypes.c_double), _ptr(d, ctypes.c_double), float(dx), float(dy),
                                      _ptr(g, ctypes.c_double))
    return float(g[0]), float(g[1])


def backward_centre(scene, G, mode="bcircle") -> np.ndarray:
    """dL/d(cx, cy) [N, 2] float64 for an upstream gradient G = dL/dOPD (float32 [B, H, W]):
    -(n_p - n_medium) * sum over the particle's frame of G * grad t."""
    fs = scene.frame_start
    f = ctypes.c_float
    out = np.zeros((scene.N, 2), dtype=np.float64)
    G = np.ascontiguousarray(G, dtype=np.float32)
    for b in range(scene.B):
        lo, hi = int(fs[b]), int(fs[b + 1])
        if hi == lo:
            continue
        a = {k: np.ascontiguousarray(scene.cols[k][lo:hi], dtype=np.float32) for k in _COLS}
        kind = np.ascontiguousarray(scene.cols["kind"][lo:hi], dtype=np.uint8)
        g = np.zeros((hi - lo, 2), dtype=np.float64)
        Gb = np.ascontiguousarray(G[b])
        _lib().osog_oracle_backward_centre(
            hi - lo, _ptr(a["cx"], f), _ptr(a["cy"], f), _ptr(a["qw"], f), _ptr(a["qx"], f), _ptr(a["qy"], f),
            _ptr(a["qz"], f), _ptr(a["d0"], f), _ptr(a["d1"], f), _ptr(a["d2"], f), _ptr(a["n_p"], f),
            _ptr(kind, ctypes.c_uint8), scene.H, scene.W, float(scene.pitch_um), float(scene.n_medium),
            {"full": 0, "bcircle": 1}[mode], _ptr(Gb, f), _ptr(g, ctypes.c_double))
        out[lo:hi] = g
    return out


def thickness_param_grad(kind, q, dims, dx, dy) -> np.ndarray:
    """float64 [7]: dt/d(d0, d1, d2, qw, qx, qy, qz) of one particle's thickness at the offset (dx, dy) from its centre
    (0 where the chord is empty); the quaternion components are independent variables of the un-normalised rotation formula."""
    qq = np.ascontiguousarray(q, dtype=np.float64)
    d = np.ascontiguousarray(dims, dtype=np.float64)
    g = np.zeros(7, dtype=np.float64)
    _lib().osog_oracle_thickness_param_grad(int(kind), _ptr(qq, ctypes.c_double), _ptr(d, ctypes.c_double), float(dx), float(dy),
                                            _ptr(g, ctypes.c_double))
    return g


def backward_params(scene, G, mode="bcircle") -> np.ndarray:
    """dL/d(d0, d1, d2, qw, qx, qy, qz) [N, 7] float64 for an upstream gradient G = dL/dOPD (float32 [B, H, W]):
    (n_p - n_medium) * sum over the particle's frame of G * dt/dtheta."""
    fs = scene.frame_start
    f = ctypes.c_float
    out = np.zeros((scene.N, 7), dtype=np.float64)
    G = np.ascontiguousarray(G, dtype=np.float32)
    for b in range(scene.B):
        lo, hi = int(fs[b]), int(fs[b + 1])
        if hi == lo:
            continue
        a = {k: np.ascontiguousarray(scene.cols[k][lo:hi], dtype=np.float32) for k in _COLS}
        kind = np.ascontiguousarray(scene.cols["kind"][lo:hi], dtype=np.uint8)
        g = np.zeros((hi - lo, 7), dtype=np.float64)
        Gb = np.ascontiguousarray(G[b])
        _lib().osog_oracle_backward_params(
            hi - lo, _ptr(a["cx"], f), _ptr(a["cy"], f), _ptr(a["qw"], f), _ptr(a["qx"], f), _ptr(a["qy"], f),
            _ptr(a["qz"], f), _ptr(a["d0"], f), _ptr(a["d1"], f), _ptr(a["d2"], f), _ptr(a["n_p"], f),
            _ptr(kind, ctypes.c_uint8), scene.H, scene.W, float(scene.pitch_um), float(scene.n_medium),
            {"full": 0, "bcircle": 1}[mode], _ptr(Gb, f), _ptr(g, ctypes.c_double))
        out[lo:hi] = g
    return out


def spectral_loss(I, I_target, eps) -> float:
    """Eq. 8 for one frame: || log(|F(I)| + eps) - log(|F(I_target)| + eps) ||^2 summed over all FFT bins,
    F = the unnormalised 2-D DFT (reading A28: eps > 0 keeps the logarithm finite at empty bins; natural logarithm)."""
    a = np.log(np.abs(np.fft.fft2(np.asarray(I, dtype=np.float64))) + eps)
    b = np.log(np.abs(np.fft.fft2(np.asarray(I_target, dtype=np.float64))) + eps)
    return float(((a - b) ** 2).sum())


def spectral_loss_grad(I, I_target, eps) -> np.ndarray:
    """dL_spectral / dI [H, W] float64.  With F_k = sum_x I_x e^{-i theta_kx}: d|F_k|/dI_x = Re(conj(F_k) e^{-i theta_kx}) / |F_k|,
    so dL/dI_x = Re sum_k W_k e^{-i theta_kx} = Re(DFT2(W))_x with W_k = 2 (a_k - b_k) / (|F_k| + eps) * conj(F_k) / |F_k|
    (W_k = 0 where F_k = 0)."""
    F = np.fft.fft2(np.asarray(I, dtype=np.float64))
    absF = np.abs(F)
    a = np.log(absF + eps)
    b = np.log(np.abs(np.fft.fft2(np.asarray(I_target, dtype=np.float64))) + eps)
    with np.errstate(divide="ignore", invalid="ignore"):
        Wk = np.where(absF > 0.0, 2.0 * (a - b) / (absF + eps) * np.conj(F) / absF, 0.0)
    return np.real(np.fft.fft2(Wk))


def count_covered(scene, mode="bcircle"):
    """Workload statistic: (ellipsoid pairs, prism pairs) = number of (particle, pixel) pairs with positive
    thickness, summed over the frames of a workloads.Scene (the "true covered pairs" of SURVEY.md 8(d))."""
    fs = scene.frame_start
    f = ctypes.c_float
    tot = np.zeros(2, dtype=np.int64)
    for b in range(scene.B):
        lo, hi = int(fs[b]), int(fs[b + 1])
        a = {k: np.ascontiguousarray(scene.cols[k][lo:hi], dtype=np.float32) for k in _COLS}
        kind = np.ascontiguousarray(scene.cols["kind"][lo:hi], dtype=np.uint8)
        out = np.zeros(2, dtype=np.int64)
        _lib().osog_oracle_count_covered(
            hi - lo, _ptr(a["cx"], f), _ptr(a["cy"], f), _ptr(a["qw"], f), _ptr(a["qx"], f), _ptr(a["qy"], f),
            _ptr(a["qz"], f), _ptr(a["d0"], f), _ptr(a["d1"], f), _ptr(a["d2"], f), _ptr(a["n_p"], f),
            _ptr(kind, ctypes.c_uint8), scene.H, scene.W, float(scene.pitch_um),
            {"full": 0, "bcircle": 1}[mode], _ptr(out, ctypes.c_int64))
        tot += out
    return int(tot[0]), int(tot[1])


def topography_factor(scene, b) -> np.ndarray:
    """Micro-topography of PAPER.md:74 (reading A29): the factor 1 + a eta[i, j] that multiplies every particle's thickness at
    pixel (i, j) of frame b; eta ~ N(0, 1) white per pixel, Box-Muller on the Philox stream with counter (pixel, frame, 2, 0)
    (the read noise uses word 2 = 0, the shot noise 1); a = scene.topography_amplitude (0: smooth bodies, factor 1)."""
    a = float(getattr(scene, "topography_amplitude", 0.0))
    if a == 0.0:
        return np.ones((scene.H, scene.W), dtype=np.float64)
    return 1.0 + a * _stream_normal(scene.seed, b, scene.H, scene.W, 2)


def render_opd(scene, mode="bcircle") -> np.ndarray:
    """OPD [B, H, W] float64 for a workloads.Scene (with the micro-topography factor of the scene, if any)."""
    fs = scene.frame_start
    return np.stack([render_opd_frame(scene.cols, int(fs[b]), int(fs[b + 1]), scene.H, scene.W,
                                      scene.pitch_um, scene.n_medium, mode) * topography_factor(scene, b) for b in range(scene.B)])


# --------------------------------------------------------------------------------------------
# optics (numpy, float64 / complex128)
# --------------------------------------------------------------------------------------------
def field(opd, lam, pitch, tilt_x=0.0, tilt_y=0.0) -> np.ndarray:
    """Exit wave of Eq. 2 with A == 1 and phase sign +i, times the oblique-illumination ramp
    exp(i 2 pi (fx0 x + fy0 y)), fx0 = sin(tilt_x)/lambda (reading A11), at pixel centres."""
    H, W = opd.shape
    x = (np.arange(W, dtype=np.float64) + 0.5) * pitch
    y = (np.arange(H, dtype=np.float64) + 0.5) * pitch
    fx0 = math.sin(tilt_x) / lam
    fy0 = math.sin(tilt_y) / lam
    turns = opd / lam + fx0 * x[None, :] + fy0 * y[:, None]
    return np.exp(2j * np.pi * turns)


def pupil_threshold(H, W, NA, pitch, lam) -> int:
    """floor((NA p / lambda)^2 H^2 W^2): bin (my, mx) passes iff mx^2 H^2 + my^2 W^2 <= this (A10)."""
    r = NA * pitch / lam
    return int(math.floor(r * r * (float(H) * H) * (float(W) * W)))


def pupil_mask(H, W, NA, pitch, lam) -> np.ndarray:
    """circ(|k|/k_NA) of Eq. 3 on the FFT grid: spatial frequency of bin m is m/(W p) with m the signed
    FFT index; inclusive edge; cutoff NA/lambda; compared in 64-bit integers."""
    mx = np.fft.fftfreq(W, d=1.0 / W).round().astype(np.int64)
    my = np.fft.fftfreq(H, d=1.0 / H).round().astype(np.int64)
    lhs = (mx * mx)[None, :] * (H * H) + (my * my)[:, None] * (W * W)
    return lhs <= pupil_threshold(H, W, NA, pitch, lam)


def propagating_threshold(H, W, n_medium, pitch, lam) -> int:
    """floor((n_medium p / lambda)^2 H^2 W^2): bin (my, mx) is a propagating wave (real k_z) iff
    mx^2 H^2 + my^2 W^2 <= this - the same integer form as the pupil edge (A10), with NA replaced by n_medium."""
    r = n_medium * pitch / lam
    return int(math.floor(r * r * (float(H) * H) * (float(W) * W)))


def defocus_factor(H, W, pitch, lam, n_medium, dz) -> np.ndarray:
    """exp(i dz sqrt(k0^2 - kx^2 - ky^2)) of Eq. 3 on the FFT grid (reading A20): angular spatial
    frequency k = 2 pi f with f = m / (W p) (m the signed FFT index, as for the pupil, A10) and k0 = 2 pi n_medium /
    lambda, the wavenumber in the medium the particles sit in; so the phase in turns is dz sqrt((n_m/lambda)^2 - fx^2 -
    fy^2).  Evanescent bins (negative radicand; always outside a physical pupil, NA <= n_m) carry no propagating
    wave: they are set to 0 whenever dz != 0.  dz == 0 gives exactly 1 on every bin (Eq. 3 reduces to circ)."""
    if dz == 0.0:
        return np.ones((H, W), dtype=np.complex128)
    mx = np.fft.fftfreq(W, d=1.0 / W).round().astype(np.int64)
    my = np.fft.fftfreq(H, d=1.0 / H).round().astype(np.int64)
    lhs = (mx * mx)[None, :] * (H * H) + (my * my)[:, None] * (W * W)
    prop = lhs <= propagating_threshold(H, W, n_medium, pitch, lam)
    fx = mx.astype(np.float64) / (W * pitch)
    fy = my.astype(np.float64) / (H * pitch)
    rad = (n_medium / lam) ** 2 - (fx * fx)[None, :] - (fy * fy)[:, None]
    turns = dz * np.sqrt(np.maximum(rad, 0.0))
    return np.where(prop, np.exp(2j * np.pi * turns), 0.0)


def pupil_function(H, W, NA, pitch, lam, n_medium, dz=0.0, pupil_enabled=True) -> np.ndarray:
    """P(kx, ky) of Eq. 3: circ(|k| / k_NA) times the defocus factor; complex128 [H, W]."""
    P = defocus_factor(H, W, pitch, lam, n_medium, dz)
    if pupil_enabled:
        P = P * pupil_mask(H, W, NA, pitch, lam)
    return P


def dic_image(U, P, shear_px, theta) -> np.ndarray:
    """Eq. 5:  I_DIC(r) = | U(r + ds) e^{i theta} - U(r - ds) e^{-i theta} |^2  *  |h_obj(r)|^2.
    U: exit wave [H, W]; P: pupil function on the FFT grid (None = all-pass), h_obj = F^-1{P} (the same
    normalised inverse FFT as coherent_image, so that U * h_obj = ifft2(fft2(U) P)); shear_px = (sx, sy): the half
    shear ds in whole pixels along x (columns) and y (rows), the two copies are 2 ds apart (A21); theta: bias phase.
    Both the shear and the convolution are circular, like the FFT stage of the coherent path (A11, A22).
    |h_obj|^2 is used as Eq. 5 writes it, without renormalising it to unit sum (A22)."""
    sx, sy = int(shear_px[0]), int(shear_px[1])
    Up = np.roll(U, shift=(-sy, -sx), axis=(0, 1))          # Up[i, j] = U[i + sy, j + sx] = U(r + ds)
    Um = np.roll(U, shift=(sy, sx), axis=(0, 1))            # U(r - ds)
    d = Up * np.exp(1j * theta) - Um * np.exp(-1j * theta)
    D = d.real * d.real + d.imag * d.imag
    H, W = U.shape
    h = np.fft.ifft2(np.ones((H, W), dtype=np.complex128) if P is None else P)
    psf = h.real * h.real + h.imag * h.imag
    return np.fft.ifft2(np.fft.fft2(D) * np.fft.fft2(psf)).real


def coherent_image(U, mask=None) -> np.ndarray:
    """U * h_obj, h_obj = F^-1{P}: forward FFT, multiply by the pupil, inverse FFT
    (normalised so that an all-pass pupil returns U)."""
    F = np.fft.fft2(U)
    if mask is not None:
        F = F * mask
    return np.fft.ifft2(F)


def intensity(U, mask=None) -> np.ndarray:
    """I_BF = |U * h_obj|^2."""
    V = coherent_image(U, mask)
    return V.real * V.real + V.imag * V.imag


# --------------------------------------------------------------------------------------------
# Philox4x32-10 and Gaussian read noise
# --------------------------------------------------------------------------------------------
_PHILOX_M0 = np.uint64(0xD2511F53)
_PHILOX_M1 = np.uint64(0xCD9E8D57)
_PHILOX_W0 = 0x9E3779B9
_PHILOX_W1 = 0xBB67AE85
_MASK32 = np.uint64(0xFFFFFFFF)


def philox4x32_10(counter, key) -> np.ndarray:
    """Philox-4x32 with 10 rounds (Salmon, Moraes, Dror, Shaw, SC'11).  counter: uint32 [..., 4],
    key: (k0, k1).  One round maps (c0, c1, c2, c3) to (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2),
    hi(M0 c0) ^ c3 ^ k1, lo(M0 c0)); the key is bumped by the Weyl constants between rounds."""
    c = np.asarray(counter, dtype=np.uint64) & _MASK32
    c0, c1, c2, c3 = (c[..., k].copy() for k in range(4))
    k0 = int(key[0]) & 0xFFFFFFFF
    k1 = int(key[1]) & 0xFFFFFFFF
    for _ in range(10):
        p0 = _PHILOX_M0 * c0
        p1 = _PHILOX_M1 * c2
        n0 = (p1 >> np.uint64(32)) ^ c1 ^ np.uint64(k0)
        n1 = p1 & _MASK32
        n2 = (p0 >> np.uint64(32)) ^ c3 ^ np.uint64(k1)
        n3 = p0 & _MASK32
        c0, c1, c2, c3 = n0, n1, n2, n3
        k0 = (k0 + _PHILOX_W0) & 0xFFFFFFFF
        k1 = (k1 + _PHILOX_W1) & 0xFFFFFFFF
    return np.stack([c0, c1, c2, c3], axis=-1).astype(np.uint32)


def read_noise(seed, frame, H, W) -> np.ndarray:
    """Standard normal z[i, j] for one frame (reading A13): Philox key = (seed low 32, seed high 32),
    counter = (pixel = i W + j, frame, 0, 0); u1 = (r0 + 1) 2^-32 in (0, 1], u2 = r1 2^-32 in [0, 1);
    z = sqrt(-2 ln u1) cos(2 pi u2) (Box-Muller)."""
    return _stream_normal(seed, frame, H, W, 0)


def _stream_normal(seed, frame, H, W, stream) -> np.ndarray:
    """Box-Muller normals of the Philox stream with counter (pixel, frame, stream, 0)."""
    pix = np.arange(H * W, dtype=np.uint64)
    ctr = np.zeros((H * W, 4), dtype=np.uint64)
    ctr[:, 0] = pix
    ctr[:, 1] = np.uint64(frame)
    ctr[:, 2] = np.uint64(stream)
    r = philox4x32_10(ctr, (seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF))
    u1 = (r[:, 0].astype(np.float64) + 1.0) * 2.0 ** -32
    u2 = r[:, 1].astype(np.float64) * 2.0 ** -32
    z = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    return z.reshape(H, W)


# --------------------------------------------------------------------------------------------
# Poisson shot noise ("P(lambda) + G(0, sigma^2)"; reading A26)
# --------------------------------------------------------------------------------------------
POISSON_SMALL = 10.0       # below: inversion by sequential search; from here on: transformed rejection (PTRS)


def shot_uniforms(seed, frame, pixels, block) -> np.ndarray:
    """Two uniforms in [0, 1) with 53 random bits each for every pixel, from Philox block `block` of the shot-noise
    stream: key = (seed low 32, seed high 32), counter = (pixel, frame, 1, block) (the read noise uses (pixel, frame, 0, 0));
    u_a = ((r0 >> 5) 2^26 + (r1 >> 6)) 2^-53, u_b likewise from (r2, r3).  Returns float64 [n, 2]."""
    pixels = np.asarray(pixels, dtype=np.uint64)
    ctr = np.zeros((pixels.size, 4), dtype=np.uint64)
    ctr[:, 0] = pixels
    ctr[:, 1] = np.uint64(frame)
    ctr[:, 2] = np.uint64(1)
    ctr[:, 3] = np.uint64(block)
    r = philox4x32_10(ctr, (seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)).astype(np.uint64)
    ua = ((r[:, 0] >> np.uint64(5)) * np.uint64(1 << 26) + (r[:, 1] >> np.uint64(6))).astype(np.float64) * 2.0 ** -53
    ub = ((r[:, 2] >> np.uint64(5)) * np.uint64(1 << 26) + (r[:, 3] >> np.uint64(6))).astype(np.float64) * 2.0 ** -53
    return np.stack([ua, ub], axis=1)


def poisson_counts(lam, seed, frame, pixels=None) -> np.ndarray:
    """One Poisson(lam[k]) draw per pixel (int64), a pure function of (seed, frame, pixel, lam) (reading A26).
    lam < 10: inversion by sequential search with the first uniform of block 0: the smallest k with
    sum_{j <= k} e^-lam lam^j / j! >= u (terms by the recurrence p_j = p_{j-1} lam / j, float64).
    lam >= 10: Hoermann's transformed rejection with squeeze (PTRS, 1993), round j using the two uniforms of block j:
    U = u_a - 1/2, V = u_b, us = 1/2 - |U|, k = floor((2 a / us + b) U + lam + 0.43); accept if us >= 0.07 and V <= v_r;
    reject if k < 0 or (us < 0.013 and V > us); else accept iff
    ln V + ln(1/alpha) - ln(a / us^2 + b) <= -lam + k ln lam - ln k!,
    with b = 0.931 + 2.53 sqrt(lam), a = -0.059 + 0.02483 b, 1/alpha = 1.1239 + 1.1328 / (b - 3.4),
    v_r = 0.9277 - 3.6224 / (b - 2)."""
    from scipy.special import gammaln
    lam = np.asarray(lam, dtype=np.float64).ravel()
    n = lam.size
    pixels = np.arange(n, dtype=np.uint64) if pixels is None else np.asarray(pixels, dtype=np.uint64).ravel()
    out = np.zeros(n, dtype=np.int64)
    small = (lam > 0.0) & (lam < POISSON_SMALL)
    if small.any():
        idx = np.flatnonzero(small)
        l = lam[idx]
        u = shot_uniforms(seed, frame, pixels[idx], 0)[:, 0]
        p = np.exp(-l)
        F = p.copy()
        k = np.zeros(idx.size, dtype=np.int64)
        for _ in range(200):                       # P(k > 200 | lam < 10) is far below 2^-53
            more = u > F
            if not more.any():
                break
            k = np.where(more, k + 1, k)
            p = np.where(more, p * l / np.maximum(k, 1), p)
            F = np.where(more, F + p, F)
        out[idx] = k
    large = lam >= POISSON_SMALL
    todo = np.flatnonzero(large)
    block = 0
    while todo.size:
        l = lam[todo]
        uv = shot_uniforms(seed, frame, pixels[todo], block)
        slam = np.sqrt(l)
        b = 0.931 + 2.53 * slam
        a = -0.059 + 0.02483 * b
        inv_alpha = 1.1239 + 1.1328 / (b - 3.4)
        vr = 0.9277 - 3.6224 / (b - 2.0)
        U = uv[:, 0] - 0.5
        V = uv[:, 1]
        us = 0.5 - np.abs(U)
        k = np.floor((2.0 * a / us + b) * U + l + 0.43)
        fast = (us >= 0.07) & (V <= vr)
        rej = (k < 0.0) | ((us < 0.013) & (V > us))
        with np.errstate(divide="ignore", invalid="ignore"):
            lhs = np.log(V) + np.log(inv_alpha) - np.log(a / (us * us) + b)
            rhs = -l + k * np.log(l) - gammaln(k + 1.0)
        acc = fast | (~rej & (lhs <= rhs))
        out[todo[acc]] = k[acc].astype(np.int64)
        todo = todo[~acc]
        block += 1
        if block > 1000:
            raise RuntimeError("PTRS did not terminate")
    return out


def shot_noise(I, photons, seed, frame) -> np.ndarray:
    """Photon-counted intensity of one frame: Poisson(photons * max(I, 0)) / photons (same units as I); photons = expected
    photon count at I = 1; photons = 0 leaves I unchanged (reading A26)."""
    if photons == 0.0:
        return np.asarray(I, dtype=np.float64)
    I = np.asarray(I, dtype=np.float64)
    lam = photons * np.maximum(I.ravel(), 0.0)
    return (poisson_counts(lam, seed, frame).astype(np.float64) / photons).reshape(I.shape)


# --------------------------------------------------------------------------------------------
# whole path for a Scene
# --------------------------------------------------------------------------------------------
def render_field(scene, opd=None, mode="bcircle") -> np.ndarray:
    """complex128 [B, H, W]."""
    if opd is None:
        opd = render_opd(scene, mode)
    return np.stack([field(opd[b], float(scene.lambda_um[b]), scene.pitch_um, scene.tilt_x_rad, scene.tilt_y_rad)
                     for b in range(scene.B)])


def render_intensity(scene, U=None, pupil_enabled=True, mode="bcircle") -> np.ndarray:
    """float64 [B, H, W]: |coherent image|^2 + sigma * z."""
    if U is None:
        U = render_field(scene, mode=mode)
    dz = float(getattr(scene, "defocus_um", 0.0))
    out = []
    for b in range(scene.B):
        if dz != 0.0:
            mask = pupil_function(scene.H, scene.W, float(scene.NA[b]), scene.pitch_um, float(scene.lambda_um[b]),
                                  scene.n_medium, dz, pupil_enabled)
        else:
            mask = pupil_mask(scene.H, scene.W, float(scene.NA[b]), scene.pitch_um, float(scene.lambda_um[b])) \
                if pupil_enabled else None
        I = intensity(U[b], mask)
        I = shot_noise(I, float(getattr(scene, "shot_noise_photons", 0.0)), scene.seed, b)
        if scene.read_noise_sigma != 0.0:
            I = I + scene.read_noise_sigma * read_noise(scene.seed, b, scene.H, scene.W)
        out.append(I)
    return np.stack(out)


# --------------------------------------------------------------------------------------------
# brightfield amplitude, Eq. 4 (reading A27)
# --------------------------------------------------------------------------------------------
def fresnel_transmittance(cos_i, n1, n2) -> np.ndarray:
    """Unpolarised Fresnel power transmittance T_F = 1 - (R_s + R_p) / 2 of a plane interface from index n1 into n2 at
    incidence angle theta_i (cos_i = cos theta_i): Snell sin theta_t = (n1 / n2) sin theta_i,
    R_s = ((n1 cos_i - n2 cos_t) / (n1 cos_i + n2 cos_t))^2, R_p = ((n1 cos_t - n2 cos_i) / (n1 cos_t + n2 cos_i))^2;
    total internal reflection (sin theta_t > 1) gives 0."""
    ci = np.clip(np.asarray(cos_i, dtype=np.float64), 0.0, 1.0)
    if n1 == n2:                                   # no interface
        return np.ones_like(ci)
    si2 = 1.0 - ci * ci
    st2 = (n1 / n2) ** 2 * si2
    tir = st2 > 1.0
    ct = np.sqrt(np.where(tir, 0.0, 1.0 - st2))
    with np.errstate(divide="ignore", invalid="ignore"):
        rs = ((n1 * ci - n2 * ct) / (n1 * ci + n2 * ct)) ** 2
        rp = ((n1 * ct - n2 * ci) / (n1 * ct + n2 * ci)) ** 2
    graze = ci == 0.0                              # theta_i = 90 degrees: everything is reflected
    rs = np.where(graze, 1.0, rs)
    rp = np.where(graze, 1.0, rp)
    return np.where(tir, 0.0, 1.0 - 0.5 * (rs + rp))


def brightfield_amplitude(h, pitch, n_medium, n_particle, delta_mu, caustic_gain) -> np.ndarray:
    """A(x, y) of Eq. 4 for one frame: T_F(theta_i) exp(-h (mu_p - mu_s)) + C, with (reading A27) the normal
    N = <-dh/dx, -dh/dy, 1> of PAPER.md:92 from the G-buffer's height gradient (A25), illumination along L = +z so that
    cos theta_i = N.L / |N| = 1 / sqrt(1 + |grad h|^2), T_F the unpolarised Fresnel transmittance from the medium
    (n_medium) into the particle material (n_particle, one value per call), delta_mu = mu_p - mu_s in 1/um, and the caustic
    term C = -caustic_gain * laplacian(h) (gain in um, the paper only gives the proportionality)."""
    h = np.asarray(h, dtype=np.float64)
    gx, gy = height_gradient(h, pitch)
    lap = height_laplacian(h, pitch)
    cos_i = 1.0 / np.sqrt(1.0 + gx ** 2 + gy ** 2)
    return fresnel_transmittance(cos_i, n_medium, n_particle) * np.exp(-h * delta_mu) - caustic_gain * lap


def render_brightfield(scene, n_particle, delta_mu, caustic_gain, pupil_enabled=True, mode="bcircle") -> np.ndarray:
    """float64 [B, H, W]: I_BF = |(A U_exit) * h_obj|^2 with A of Eq. 4 multiplying the exit wave of Eq. 2
    (which the hot path renders with A = 1), then the sensor (shot noise, read noise)."""
    U = render_field(scene, mode=mode)
    h = render_height(scene, mode)
    A = np.stack([brightfield_amplitude(h[b], scene.pitch_um, scene.n_medium, n_particle, delta_mu, caustic_gain)
                  for b in range(scene.B)])
    return render_intensity(scene, U=A * U, pupil_enabled=pupil_enabled, mode=mode)


def render_dic(scene, shear_px, theta, U=None, pupil_enabled=True, mode="bcircle") -> np.ndarray:
    """float64 [B, H, W]: Eq. 5 on the scene's exit wave, through the scene's pupil (with its defocus), + sigma * z."""
    if U is None:
        U = render_field(scene, mode=mode)
    dz = float(getattr(scene, "defocus_um", 0.0))
    out = []
    for b in range(scene.B):
        P = pupil_function(scene.H, scene.W, float(scene.NA[b]), scene.pitch_um, float(scene.lambda_um[b]),
                           scene.n_medium, dz, pupil_enabled)
        I = dic_image(U[b], P, shear_px, theta)
        I = shot_noise(I, float(getattr(scene, "shot_noise_photons", 0.0)), scene.seed, b)
        if scene.read_noise_sigma != 0.0:
            I = I + scene.read_noise_sigma * read_noise(scene.seed, b, scene.H, scene.W)
        out.append(I)
    return np.stack(out)


# --------------------------------------------------------------------------------------------
# binning (float64 -> integers), B1-B4
# --------------------------------------------------------------------------------------------
BBOX_PAD_PX = 2.0 ** -10


def _rot_all(cols):
    w, x, y, z = (cols[k].astype(np.float64) for k in ("qw", "qx", "qy", "qz"))
    R = np.empty((w.size, 3, 3), dtype=np.float64)
    R[:, 0, 0] = 1.0 - 2.0 * (y * y + z * z); R[:, 0, 1] = 2.0 * (x * y - w * z); R[:, 0, 2] = 2.0 * (x * z + w * y)
    R[:, 1, 0] = 2.0 * (x * y + w * z); R[:, 1, 1] = 1.0 - 2.0 * (x * x + z * z); R[:, 1, 2] = 2.0 * (y * z - w * x)
    R[:, 2, 0] = 2.0 * (x * z - w * y); R[:, 2, 1] = 2.0 * (y * z + w * x); R[:, 2, 2] = 1.0 - 2.0 * (x * x + y * y)
    return R


def particle_valid(cols) -> np.ndarray:
    ok = np.ones(cols["cx"].shape[0], dtype=bool)
    for k in _COLS:
        ok &= np.isfinite(cols[k])
    for k in ("d0", "d1", "d2"):
        ok &= cols[k] > 0
    ok &= cols["kind"] <= 1
    return ok


def half_extents(cols):
    """B1: half-extent of the body's projection along world x and y.
    Ellipsoid: hx = sqrt(R_x0^2 a^2 + R_x1^2 b^2 + R_x2^2 c^2); prism: max over the 10 vertices
    (+-s/2, +-s/2, +-L/2), (0, 0, +-(L/2 + hc)) of |(R v)_x|; same with row y."""
    R = _rot_all(cols)
    d0, d1, d2 = (cols[k].astype(np.float64) for k in ("d0", "d1", "d2"))
    dims = np.stack([d0, d1, d2], axis=1)
    he = np.sqrt(((R[:, 0:2, :] * dims[:, None, :]) ** 2).sum(axis=2))          # [N, 2]
    s, L, hc = d0, d1, d2
    verts = []
    for sx in (1.0, -1.0):
        for sy in (1.0, -1.0):
            for sz in (1.0, -1.0):
                verts.append(np.stack([sx * 0.5 * s, sy * 0.5 * s, sz * 0.5 * L], axis=1))
    for sz in (1.0, -1.0):
        verts.append(np.stack([0.0 * s, 0.0 * s, sz * (0.5 * L + hc)], axis=1))
    V = np.stack(verts, axis=1)                                                   # [N, 10, 3]
    RV = np.einsum("nrc,nvc->nvr", R, V)                                          # [N, 10, 3]
    hp = np.abs(RV[:, :, 0:2]).max(axis=1)                                        # [N, 2]
    isp = (cols["kind"] == 1)[:, None]
    h = np.where(isp, hp, he)
    return h[:, 0], h[:, 1]


def render_height(scene, mode="bcircle") -> np.ndarray:
    """Height (total thickness) map h [B, H, W] float64 of the G-buffer ("spatially varying thickness
    h(x, y)"): the sum over the frame's particles of their thickness along z, i.e. the OPD loop with n_p - n_medium = 1
    exactly (n_p = 1, n_medium = 0 are passed to the same C loop)."""
    fs = scene.frame_start
    ones = dict(scene.cols)
    ones["n_p"] = np.ones_like(scene.cols["n_p"])
    return np.stack([render_opd_frame(ones, int(fs[b]), int(fs[b + 1]), scene.H, scene.W, scene.pitch_um, 0.0, mode)
                     * topography_factor(scene, b) for b in range(scene.B)])


def height_gradient(h, pitch):
    """Finite-difference gradient of a height map on the pixel grid (reading A25; the paper takes the normals
    N = <-grad_x h, -grad_y h, 1> "from the G-buffer"): central differences (h[j+1] - h[j-1]) / (2 p) inside,
    one-sided differences (h[1] - h[0]) / p and (h[W-1] - h[W-2]) / p on the frame border.  Returns (gx, gy), x = columns."""
    H, W = h.shape
    gx = np.empty_like(h)
    gy = np.empty_like(h)
    for j in range(W):
        jm, jp = max(j - 1, 0), min(j + 1, W - 1)
        gx[:, j] = (h[:, jp] - h[:, jm]) / ((jp - jm) * pitch) if jp > jm else 0.0
    for i in range(H):
        im, ip = max(i - 1, 0), min(i + 1, H - 1)
        gy[i, :] = (h[ip, :] - h[im, :]) / ((ip - im) * pitch) if ip > im else 0.0
    return gx, gy


def height_laplacian(h, pitch):
    """Five-point Laplacian of a height map (the curvature term of Eq. 4, "C(x, y) ~ -lap h"; reading A25):
    (h[i, j+1] + h[i, j-1] + h[i+1, j] + h[i-1, j] - 4 h[i, j]) / p^2 with the border pixels replicated outwards."""
    H, W = h.shape
    out = np.empty_like(h)
    for i in range(H):
        im, ip = max(i - 1, 0), min(i + 1, H - 1)
        for j in range(W):
            jm, jp = max(j - 1, 0), min(j + 1, W - 1)
            out[i, j] = (h[i, jp] + h[i, jm] + h[ip, j] + h[im, j] - 4.0 * h[i, j]) / (pitch * pitch)
    return out


def particle_obbs(scene) -> np.ndarray:
    """Oriented bounding box of every particle's silhouette, the geometric label the paper's detector is trained on
    ("YOLOv11 ... OBB"; instance geometry of the G-buffer): float64 [N, 6] =
    (centre x, centre y, axis u_x, axis u_y, half length along u, half length across u), lengths and centre in pixel
    units (pixel-index coordinates c / p - 1/2), u a unit vector with u_x >= 0.  Reading A23:
      ellipsoid  the body is {q : q^T M q <= 1}, M = R diag(1/a^2, 1/b^2, 1/c^2) R^T exactly as in the thickness function
                 (R is not renormalised, A4, so M^-1 is not quite R diag(a^2, b^2, c^2) R^T); its shadow is the ellipse
                 {d : d^T Q^-1 d <= 1} with Q = (M^-1) restricted to x, y; the box is the principal-axis box of that
                 ellipse: u = eigenvector of the larger eigenvalue of Q, half lengths sqrt(eigenvalues)
      prism      u = normalised projection of the body's long axis (R e_z)_{xy} ((1, 0) if that projection vanishes);
                 half lengths = largest |(R v)_{xy} . u| and |(R v)_{xy} . u_perp| over the 10 vertices (vertices R v
                 as in the binning spec B1)
    Invalid particles give NaN."""
    cols = scene.cols
    R = _rot_all(cols)
    n = R.shape[0]
    p = scene.pitch_um
    out = np.full((n, 6), np.nan)
    ok = particle_valid(cols)
    d = np.stack([cols[k].astype(np.float64) for k in ("d0", "d1", "d2")], axis=1)
    for k in range(n):
        if not ok[k]:
            continue
        if cols["kind"][k] == 0:
            Q = np.linalg.inv(R[k] @ np.diag(1.0 / d[k] ** 2) @ R[k].T)[:2, :2]
            lam, V = np.linalg.eigh(Q)                       # ascending eigenvalues
            u = V[:, 1]
            ha, hb = math.sqrt(lam[1]), math.sqrt(max(lam[0], 0.0))
        else:
            s_, L, hc = d[k]
            u = R[k][:2, 2].copy()
            nu = math.hypot(u[0], u[1])
            u = u / nu if nu > 1e-12 else np.array([1.0, 0.0])
            verts = [(sx * s_ / 2, sy * s_ / 2, sz * L / 2) for sx in (1, -1) for sy in (1, -1) for sz in (1, -1)]
            verts += [(0.0, 0.0, L / 2 + hc), (0.0, 0.0, -(L / 2 + hc))]
            P2 = (R[k] @ np.asarray(verts).T)[:2].T          # projected vertices [10, 2]
            ha = float(np.abs(P2 @ u).max())
            hb = float(np.abs(P2 @ np.array([-u[1], u[0]])).max())
        if u[0] < 0.0:
            u = -u
        out[k] = (float(cols["cx"][k]) / p - 0.5, float(cols["cy"][k]) / p - 0.5, u[0], u[1], ha / p, hb / p)
    return out


def bboxes(cols, H, W, pitch):
    """B2: inclusive pixel range whose centres can lie inside the projection, padded by 2^-10 px,
    clamped to the frame.  Returns int64 arrays j0, j1, i0, i1 and a bool `listed` (valid and not empty)."""
    with np.errstate(invalid="ignore", over="ignore"):
        hx, hy = half_extents(cols)
        cx = cols["cx"].astype(np.float64)
        cy = cols["cy"].astype(np.float64)
        ok = particle_valid(cols)
        fj0 = np.ceil((cx - hx) / pitch - 0.5 - BBOX_PAD_PX)
        fj1 = np.floor((cx + hx) / pitch - 0.5 + BBOX_PAD_PX)
        fi0 = np.ceil((cy - hy) / pitch - 0.5 - BBOX_PAD_PX)
        fi1 = np.floor((cy + hy) / pitch - 0.5 + BBOX_PAD_PX)
        ok &= np.isfinite(fj0) & np.isfinite(fj1) & np.isfinite(fi0) & np.isfinite(fi1)
    big = 2.0 ** 30
    def clampi(f, lo, hi):
        f = np.where(ok, np.clip(f, -big, big), 0.0)
        return np.clip(f.astype(np.int64), lo, hi)
    j0 = clampi(fj0, 0, W); j1 = clampi(fj1, -1, W - 1)
    i0 = clampi(fi0, 0, H); i1 = clampi(fi1, -1, H - 1)
    listed = ok & (j0 <= j1) & (i0 <= i1)
    return j0, j1, i0, i1, listed


def binning(scene, T):
    """B3-B4 for a Scene: tiles of T x T pixels, row-major per frame, frames concatenated
    (global tile id = frame * tiles_per_frame + ty * ceil(W/T) + tx).  A particle is listed in every
    tile its bounding box touches.  Returns (count uint32 [n_tiles], offset uint32 [n_tiles + 1],
    list uint32 [pairs]) with each tile's segment in ascending GLOBAL particle index."""
    H, W, B = scene.H, scene.W, scene.B
    ntx = -(-W // T)
    nty = -(-H // T)
    tpf = ntx * nty
    j0, j1, i0, i1, listed = bboxes(scene.cols, H, W, scene.pitch_um)
    fs = scene.frame_start
    frame_of = np.repeat(np.arange(B), np.diff(fs))
    count = np.zeros(B * tpf, dtype=np.int64)
    pairs_t = []
    pairs_n = []
    for n in np.nonzero(listed)[0]:
        tx = np.arange(j0[n] // T, j1[n] // T + 1)
        ty = np.arange(i0[n] // T, i1[n] // T + 1)
        t = (frame_of[n] * tpf + ty[:, None] * ntx + tx[None, :]).ravel()
        count[t] += 1
        pairs_t.append(t)
        pairs_n.append(np.full(t.size, n, dtype=np.int64))
    offset = np.zeros(B * tpf + 1, dtype=np.int64)
    np.cumsum(count, out=offset[1:])
    if pairs_t:
        pt = np.concatenate(pairs_t)
        pn = np.concatenate(pairs_n)
        order = np.lexsort((pn, pt))          # by tile, then ascending particle index
        lst = pn[order]
    else:
        lst = np.zeros(0, dtype=np.int64)
    return count.astype(np.uint32), offset.astype(np.uint32), lst.astype(np.uint32)
