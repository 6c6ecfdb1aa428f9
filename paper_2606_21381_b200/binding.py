"""Thin ctypes binding of libosog.so (include/osog.h).  Argument marshalling only: every step of the
render path runs in the CUDA kernels of the library.  PyTorch supplies device memory and the stream.

There is no CPU fallback: if libosog.so is missing and cannot be built, or no CUDA device is present,
the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

OSOG_OK, OSOG_EINVAL, OSOG_ECUDA, OSOG_ECAPACITY, OSOG_ENOMEM, OSOG_ELIMIT = 0, -1, -2, -3, -4, -5
OSOG_WBADPARTICLE, OSOG_WOVERFLOW = 1, 2

_F32_COLS = ("cx", "cy", "cz", "qw", "qx", "qy", "qz", "d0", "d1", "d2", "n_p")


class osog_config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("device", C.c_int32), ("stream", C.c_void_p),
                ("H", C.c_int32), ("W", C.c_int32), ("max_frames", C.c_int32),
                ("max_particles", C.c_int64), ("max_pairs", C.c_int64)]


class osog_particles(C.Structure):
    _fields_ = [("struct_size", C.c_uint32)] + [(k, C.c_void_p) for k in _F32_COLS] + \
               [("kind", C.c_void_p), ("frame_start", C.c_void_p)]


class osog_optics(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("B", C.c_int32), ("pitch_um", C.c_double), ("n_medium", C.c_double),
                ("lambda_um", C.POINTER(C.c_double)), ("NA", C.POINTER(C.c_double)),
                ("tilt_x_rad", C.c_double), ("tilt_y_rad", C.c_double), ("read_noise_sigma", C.c_double),
                ("seed", C.c_uint64), ("pupil_enabled", C.c_int32), ("defocus_um", C.c_double),
                ("shot_noise_photons", C.c_double), ("topography_amplitude", C.c_double)]


class osog_dic(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("shear_x_px", C.c_int32), ("shear_y_px", C.c_int32),
                ("bias_rad", C.c_double)]


class osog_brightfield(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_particle", C.c_double), ("delta_mu_per_um", C.c_double),
                ("caustic_gain_um", C.c_double)]


class OsogError(RuntimeError):
    def __init__(self, code, what, pairs_needed=None):
        self.code = code
        self.pairs_needed = pairs_needed      # OSOG_ECAPACITY: the max_pairs that would have sufficed
        extra = f"; max_pairs >= {pairs_needed} needed" if pairs_needed is not None else ""
        super().__init__(f"{what}: {lib().osog_strerror(code).decode()} ({code}){extra}")


_LIB = None


def lib_path() -> str:
    return _build.LIB


def lib():
    """Load (building first if the sources are newer) libosog.so and declare every exported symbol."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = _build.LIB
    if _build.needs_build():
        path = _build.build()
    L = C.CDLL(path)
    ctx = C.c_void_p
    L.osog_create.argtypes = [C.POINTER(ctx), C.POINTER(osog_config)]
    for name in ("osog_render_opd", "osog_render_field", "osog_render_intensity", "osog_render_opd_atomic",
                 "osog_render_opd_smem_atomic", "osog_particle_obbs"):
        getattr(L, name).argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics), C.c_void_p]
    L.osog_field_to_intensity.argtypes = [ctx, C.POINTER(osog_optics), C.c_void_p, C.c_void_p]
    L.osog_render_dic.argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics),
                                  C.POINTER(osog_dic), C.c_void_p]
    L.osog_render_brightfield.argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics),
                                          C.POINTER(osog_brightfield), C.c_void_p]
    L.osog_field_to_dic.argtypes = [ctx, C.POINTER(osog_optics), C.POINTER(osog_dic), C.c_void_p, C.c_void_p]
    L.osog_backward_np.argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics), C.c_void_p, C.c_void_p]
    L.osog_backward_intensity.argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics), C.c_void_p, C.c_void_p]
    L.osog_spectral_loss.argtypes = [ctx, C.c_int32, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
    L.osog_backward_params.argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics), C.c_void_p, C.c_void_p]
    L.osog_backward_particles.argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.osog_backward_centre.argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics), C.c_void_p, C.c_void_p]
    L.osog_render_gbuffer.argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics), C.c_void_p, C.c_void_p]
    L.osog_render_gbuffer_normals.argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics), C.c_void_p, C.c_void_p,
                                              C.c_void_p]
    L.osog_render_height.argtypes = [ctx, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics), C.c_void_p, C.c_void_p,
                                     C.c_void_p]
    L.osog_render_opd_static.argtypes = [C.c_int, C.c_void_p, C.c_int, C.c_int, C.POINTER(osog_particles), C.c_int64, C.POINTER(osog_optics),
                                         C.c_void_p, C.c_void_p]
    L.osog_debug_recompose_field.argtypes = [ctx, C.c_void_p]
    L.osog_debug_check_guards.argtypes = [ctx]
    L.osog_debug_poisson.argtypes = [ctx, C.c_void_p, C.c_int64, C.c_uint64, C.c_uint32, C.c_void_p]
    L.osog_destroy.argtypes = [ctx]
    L.osog_status.argtypes = [ctx, C.POINTER(C.c_uint32), C.POINTER(C.c_int64)]
    L.osog_debug_bins.argtypes = [ctx, C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.osog_tile_size.argtypes = []
    L.osog_last_cuda_error.argtypes = [ctx]
    L.osog_strerror.argtypes = [C.c_int]
    L.osog_strerror.restype = C.c_char_p
    for name in EXPORTS:
        if name != "osog_strerror":
            getattr(L, name).restype = C.c_int
    _LIB = L
    return L


EXPORTS = ("osog_create", "osog_render_opd", "osog_render_field", "osog_render_intensity",
           "osog_field_to_intensity", "osog_render_dic", "osog_field_to_dic", "osog_render_brightfield", "osog_render_opd_atomic", "osog_render_opd_smem_atomic", "osog_particle_obbs", "osog_render_gbuffer", "osog_render_gbuffer_normals", "osog_render_height", "osog_backward_np", "osog_backward_centre", "osog_backward_params", "osog_backward_particles", "osog_spectral_loss", "osog_backward_intensity", "osog_render_opd_static", "osog_debug_recompose_field", "osog_debug_check_guards", "osog_debug_poisson", "osog_destroy", "osog_status",
           "osog_debug_bins", "osog_tile_size", "osog_last_cuda_error", "osog_strerror")


def osog_tile_size() -> int:
    return lib().osog_tile_size()


def lib_limits() -> dict:
    """The fixed limits of osog_render_opd_static (OSOG_STATIC_MAX_* of include/osog.h)."""
    return {"particles": 4096, "frames": 4, "tiles": 256, "pairs": 65536}


def render_opd_static(p, o, H, W, out=None, status=None, stream=None):
    """float32 [B, H, W] OPD through osog_render_opd_static: no context, no allocation inside the call (its scratch is a fixed
    device array of the library; limits in osog.h, OSOG_ELIMIT beyond them).  `out` (float32 [B, H, W]) and `status` (a
    1-element device tensor of 4-byte integers receiving the OSOG_W* bits) are the caller's; `out` is made here only when not
    passed.  Enqueue-only on `stream` (default: torch's current stream); calls that overlap on the GPU race on the scratch."""
    import torch
    dev = p.device if p.device.index is not None else torch.device("cuda", torch.cuda.current_device())
    if out is None:
        out = torch.empty((o.B, int(H), int(W)), dtype=torch.float32, device=dev)
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    r = lib().osog_render_opd_static(dev.index if dev.index is not None else torch.cuda.current_device(), C.c_void_p(st.cuda_stream),
                                     int(H), int(W), C.byref(p.c), p.N, C.byref(o), out.data_ptr(),
                                     status.data_ptr() if status is not None else None)
    if r != OSOG_OK:
        raise OsogError(r, "osog_render_opd_static")
    return out


class Particles:
    """SoA particle state resident on the device (torch tensors), plus the osog_particles view of it."""

    def __init__(self, cols: dict, frame_start=None, device="cuda:0"):
        import torch
        self.device = torch.device(device)
        self.t = {}
        for k in _F32_COLS:
            if k in cols and cols[k] is not None:
                self.t[k] = self._dev(cols[k], torch.float32)
        self.t["kind"] = self._dev(cols["kind"], torch.uint8)
        self.N = int(self.t["kind"].numel())
        self.frame_start = None
        if frame_start is not None:
            self.frame_start = self._dev(np.asarray(frame_start, dtype=np.int32), torch.int32)
        self.c = osog_particles()
        self.c.struct_size = C.sizeof(osog_particles)
        for k in _F32_COLS:
            setattr(self.c, k, self.t[k].data_ptr() if k in self.t and self.N > 0 else None)
        self.c.kind = self.t["kind"].data_ptr() if self.N > 0 else None
        self.c.frame_start = self.frame_start.data_ptr() if self.frame_start is not None else None

    def _dev(self, a, dtype):
        import torch
        if isinstance(a, torch.Tensor):
            return a.to(device=self.device, dtype=dtype).contiguous()
        return torch.from_numpy(np.ascontiguousarray(a)).to(dtype).to(self.device)

    @classmethod
    def from_scene(cls, scene, device="cuda:0"):
        return cls(scene.cols, scene.frame_start if scene.B > 1 else None, device)


def make_optics(B, pitch_um, n_medium, lambda_um, NA=None, tilt_x_rad=0.0, tilt_y_rad=0.0,
                read_noise_sigma=0.0, seed=0, pupil_enabled=True, defocus_um=0.0, shot_noise_photons=0.0,
                topography_amplitude=0.0):
    """osog_optics plus the host arrays it points to (kept alive as attributes)."""
    o = osog_optics()
    o.struct_size = C.sizeof(osog_optics)
    o.B = int(B)
    o.pitch_um = float(pitch_um)
    o.n_medium = float(n_medium)
    lam = np.ascontiguousarray(np.broadcast_to(np.asarray(lambda_um, dtype=np.float64), (B,)))
    o._lam = lam
    o.lambda_um = lam.ctypes.data_as(C.POINTER(C.c_double))
    if NA is not None:
        na = np.ascontiguousarray(np.broadcast_to(np.asarray(NA, dtype=np.float64), (B,)))
        o._na = na
        o.NA = na.ctypes.data_as(C.POINTER(C.c_double))
    o.tilt_x_rad = float(tilt_x_rad)
    o.tilt_y_rad = float(tilt_y_rad)
    o.read_noise_sigma = float(read_noise_sigma)
    o.seed = int(seed) & 0xFFFFFFFFFFFFFFFF
    o.pupil_enabled = 1 if pupil_enabled else 0
    o.defocus_um = float(defocus_um)
    o.shot_noise_photons = float(shot_noise_photons)
    o.topography_amplitude = float(topography_amplitude)
    return o


def make_dic(shear_x_px, shear_y_px, bias_rad):
    d = osog_dic()
    d.struct_size = C.sizeof(osog_dic)
    d.shear_x_px, d.shear_y_px, d.bias_rad = int(shear_x_px), int(shear_y_px), float(bias_rad)
    return d


def make_brightfield(n_particle, delta_mu_per_um=0.0, caustic_gain_um=0.0):
    b = osog_brightfield()
    b.struct_size = C.sizeof(osog_brightfield)
    b.n_particle, b.delta_mu_per_um, b.caustic_gain_um = float(n_particle), float(delta_mu_per_um), float(caustic_gain_um)
    return b


def optics_from_scene(scene, pupil_enabled=True):
    return make_optics(scene.B, scene.pitch_um, scene.n_medium, scene.lambda_um, scene.NA, scene.tilt_x_rad,
                       scene.tilt_y_rad, scene.read_noise_sigma, scene.seed, pupil_enabled,
                       getattr(scene, "defocus_um", 0.0), getattr(scene, "shot_noise_photons", 0.0),
                       getattr(scene, "topography_amplitude", 0.0))


class Context:
    """osog_ctx owner.  Methods mirror the C entry points and return torch tensors on the device."""

    def __init__(self, H, W, max_particles, max_frames=1, max_pairs=0, device="cuda:0", stream=None, check=True):
        """check=True: every render / backward call is followed by osog_status (which synchronises the stream) and raises
        OsogError(OSOG_ECAPACITY) when the call needed more (particle, tile) pairs than max_pairs - its outputs are then
        zero-filled.  check=False leaves the calls enqueue-only (timed loops); call status() yourself."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("osog: no CUDA device; this library has no CPU fallback")
        self.torch = torch
        self.check = bool(check)
        self.device = torch.device(device)
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.H, self.W, self.max_frames = int(H), int(W), int(max_frames)
        cfg = osog_config()
        cfg.struct_size = C.sizeof(osog_config)
        cfg.device = self.device.index
        cfg.stream = self.stream.cuda_stream
        cfg.H, cfg.W, cfg.max_frames = self.H, self.W, self.max_frames
        cfg.max_particles = int(max_particles)
        cfg.max_pairs = int(max_pairs)
        self._ctx = C.c_void_p()
        r = lib().osog_create(C.byref(self._ctx), C.byref(cfg))
        if r != OSOG_OK:
            self._ctx = None
            raise OsogError(r, "osog_create")

    def close(self):
        if getattr(self, "_ctx", None):
            lib().osog_destroy(self._ctx)
            self._ctx = None

    __del__ = close

    def _out(self, B, *tail, out=None):
        if out is not None:
            return out
        return self.torch.empty((B, self.H, self.W) + tail, dtype=self.torch.float32, device=self.device)

    def _done(self, r, name):
        """Return-code check of an entry point, then (check=True) the device status of the call it enqueued."""
        if r != OSOG_OK:
            raise OsogError(r, name)
        if self.check:
            bits, pairs = C.c_uint32(0), C.c_int64(0)
            r = lib().osog_status(self._ctx, C.byref(bits), C.byref(pairs))
            if r != OSOG_OK:
                raise OsogError(r, name, pairs.value if r == OSOG_ECAPACITY else None)

    def _in(self, t, shape, name):
        """A caller-supplied device tensor the library reads: float32, contiguous, on this device, of the stated shape."""
        torch = self.torch
        if t.is_complex():
            t = torch.view_as_real(t)
        if tuple(t.shape) != tuple(shape):
            raise ValueError(f"{name}: shape {tuple(t.shape)}, expected {tuple(shape)}")
        if t.device != self.device:
            raise ValueError(f"{name}: on {t.device}, the context is on {self.device}")
        if t.dtype != torch.float32 or not t.is_contiguous():
            t = t.to(torch.float32).contiguous()
        return t

    def _call(self, name, p, o, out):
        self._done(getattr(lib(), name)(self._ctx, C.byref(p.c), p.N, C.byref(o), out.data_ptr()), name)
        return out

    def render_opd(self, p: Particles, o, out=None):
        """float32 [B, H, W] OPD in micrometres (osog_render_opd)."""
        return self._call("osog_render_opd", p, o, self._out(o.B, out=out))

    def render_opd_atomic(self, p: Particles, o, out=None):
        return self._call("osog_render_opd_atomic", p, o, self._out(o.B, out=out))

    def render_height(self, p: Particles, o, grad=True, lap=True):
        """(h float32 [B, H, W], grad float32 [B, H, W, 2] or None, lap float32 [B, H, W] or None) (osog_render_height)."""
        h = self._out(o.B)
        g = self._out(o.B, 2) if grad else None
        l = self._out(o.B) if lap else None
        self._done(lib().osog_render_height(self._ctx, C.byref(p.c), p.N, C.byref(o), h.data_ptr(),
                                            g.data_ptr() if grad else None, l.data_ptr() if lap else None), "osog_render_height")
        return h, g, l

    def backward_np(self, p: Particles, o, gopd):
        """float32 [N] dL/dn_p for an upstream gradient gopd = dL/dOPD (float32 [B, H, W]) (osog_backward_np)."""
        out = self.torch.empty((p.N,), dtype=self.torch.float32, device=self.device)
        gopd = self._in(gopd, (o.B, self.H, self.W), "gopd")
        self._done(lib().osog_backward_np(self._ctx, C.byref(p.c), p.N, C.byref(o), gopd.data_ptr(), out.data_ptr()), "osog_backward_np")
        return out

    def backward_intensity(self, p: Particles, o, gI):
        """float32 [B, H, W] dL/dOPD for an upstream gradient gI = dL/dI of the coherent intensity (osog_backward_intensity)."""
        out = self._out(o.B)
        gI = self._in(gI, (o.B, self.H, self.W), "gI")
        self._done(lib().osog_backward_intensity(self._ctx, C.byref(p.c), p.N, C.byref(o), gI.data_ptr(), out.data_ptr()),
                   "osog_backward_intensity")
        return out

    def backward_centre(self, p: Particles, o, gopd):
        """float32 [N, 2] (dL/dcx, dL/dcy) for an upstream gradient gopd = dL/dOPD (osog_backward_centre)."""
        out = self.torch.empty((p.N, 2), dtype=self.torch.float32, device=self.device)
        gopd = self._in(gopd, (o.B, self.H, self.W), "gopd")
        self._done(lib().osog_backward_centre(self._ctx, C.byref(p.c), p.N, C.byref(o), gopd.data_ptr(), out.data_ptr()),
                   "osog_backward_centre")
        return out

    def backward_params(self, p: Particles, o, gopd):
        """float32 [N, 7] dL/d(d0, d1, d2, qw, qx, qy, qz) for an upstream gradient gopd = dL/dOPD (osog_backward_params)."""
        out = self.torch.empty((p.N, 7), dtype=self.torch.float32, device=self.device)
        gopd = self._in(gopd, (o.B, self.H, self.W), "gopd")
        self._done(lib().osog_backward_params(self._ctx, C.byref(p.c), p.N, C.byref(o), gopd.data_ptr(), out.data_ptr()),
                   "osog_backward_params")
        return out

    def backward_particles(self, p: Particles, o, gopd, np_=True, centre=True, params=True):
        """(float32 [N] dL/dn_p, float32 [N, 2] dL/d(cx, cy), float32 [N, 7] dL/d(d0, d1, d2, qw, qx, qy, qz)) from ONE pass over
        the pixels; an output that is switched off is None (osog_backward_particles)."""
        t = self.torch
        gnp = t.empty((p.N,), dtype=t.float32, device=self.device) if np_ else None
        gc = t.empty((p.N, 2), dtype=t.float32, device=self.device) if centre else None
        gpar = t.empty((p.N, 7), dtype=t.float32, device=self.device) if params else None
        gopd = self._in(gopd, (o.B, self.H, self.W), "gopd")
        ptr = lambda x: x.data_ptr() if x is not None else None
        self._done(lib().osog_backward_particles(self._ctx, C.byref(p.c), p.N, C.byref(o), gopd.data_ptr(), ptr(gnp), ptr(gc), ptr(gpar)),
                   "osog_backward_particles")
        return gnp, gc, gpar

    def spectral_loss(self, I, I_target, eps, grad=True):
        """(float64 [B] loss of Eq. 8, float32 [B, H, W] dL/dI or None) for images I, I_target (float32 [B, H, W]) (osog_spectral_loss)."""
        B = int(I.shape[0])
        I = self._in(I, (B, self.H, self.W), "I")
        T = self._in(I_target, (B, self.H, self.W), "I_target")
        loss = self.torch.empty((B,), dtype=self.torch.float64, device=self.device)
        g = self._out(B) if grad else None
        r = lib().osog_spectral_loss(self._ctx, B, I.data_ptr(), T.data_ptr(), float(eps), loss.data_ptr(), g.data_ptr() if grad else None)
        if r != OSOG_OK:
            raise OsogError(r, "osog_spectral_loss")
        return loss, g

    def render_gbuffer(self, p: Particles, o, normals=False):
        """(int32 [B, H, W] instance id of the top-most particle, float32 [B, H, W] height of its top surface); with
        normals=True also float32 [B, H, W, 2], the analytic slope (dz/dx, dz/dy) of that surface (osog_render_gbuffer_normals)."""
        tid = self.torch.empty((o.B, self.H, self.W), dtype=self.torch.int32, device=self.device)
        dep = self.torch.empty((o.B, self.H, self.W), dtype=self.torch.float32, device=self.device)
        if normals:
            nrm = self._out(o.B, 2)
            self._done(lib().osog_render_gbuffer_normals(self._ctx, C.byref(p.c), p.N, C.byref(o), tid.data_ptr(), dep.data_ptr(),
                                                         nrm.data_ptr()), "osog_render_gbuffer_normals")
            return tid, dep, nrm
        self._done(lib().osog_render_gbuffer(self._ctx, C.byref(p.c), p.N, C.byref(o), tid.data_ptr(), dep.data_ptr()),
                   "osog_render_gbuffer")
        return tid, dep

    def particle_obbs(self, p: Particles, o, out=None):
        """float32 [N, 6] oriented-bounding-box labels (osog_particle_obbs)."""
        if out is None:
            out = self.torch.empty((p.N, 6), dtype=self.torch.float32, device=self.device)
        r = lib().osog_particle_obbs(self._ctx, C.byref(p.c), p.N, C.byref(o), out.data_ptr())
        if r != OSOG_OK:
            raise OsogError(r, "osog_particle_obbs")      # (runs the preparation kernel only: no list capacity involved)
        return out

    def render_opd_smem_atomic(self, p: Particles, o, out=None):
        return self._call("osog_render_opd_smem_atomic", p, o, self._out(o.B, out=out))

    def render_field(self, p: Particles, o, out=None):
        """complex64 [B, H, W] exit wave (osog_render_field); `out` is a float32 [B, H, W, 2] buffer."""
        buf = self._call("osog_render_field", p, o, self._out(o.B, 2, out=out))
        return self.torch.view_as_complex(buf)

    def render_intensity(self, p: Particles, o, out=None):
        """float32 [B, H, W] coherent intensity (osog_render_intensity)."""
        return self._call("osog_render_intensity", p, o, self._out(o.B, out=out))

    def field_to_intensity(self, o, field, out=None):
        out = self._out(o.B, out=out)
        f = self._in(field, (o.B, self.H, self.W, 2), "field")
        r = lib().osog_field_to_intensity(self._ctx, C.byref(o), f.data_ptr(), out.data_ptr())
        if r != OSOG_OK:
            raise OsogError(r, "osog_field_to_intensity")
        return out

    def render_dic(self, p: Particles, o, dic, out=None):
        """float32 [B, H, W] DIC image of Eq. 5 (osog_render_dic); `dic` from make_dic."""
        out = self._out(o.B, out=out)
        self._done(lib().osog_render_dic(self._ctx, C.byref(p.c), p.N, C.byref(o), C.byref(dic), out.data_ptr()), "osog_render_dic")
        return out

    def render_brightfield(self, p: Particles, o, bf, out=None):
        """float32 [B, H, W] brightfield image with the amplitude of Eq. 4 (osog_render_brightfield); `bf` from make_brightfield."""
        out = self._out(o.B, out=out)
        self._done(lib().osog_render_brightfield(self._ctx, C.byref(p.c), p.N, C.byref(o), C.byref(bf), out.data_ptr()),
                   "osog_render_brightfield")
        return out

    def field_to_dic(self, o, dic, field, out=None):
        out = self._out(o.B, out=out)
        f = self._in(field, (o.B, self.H, self.W, 2), "field")
        r = lib().osog_field_to_dic(self._ctx, C.byref(o), C.byref(dic), f.data_ptr(), out.data_ptr())
        if r != OSOG_OK:
            raise OsogError(r, "osog_field_to_dic")
        return out

    def recompose_field(self, out):
        """Re-run only the composition kernel of the last render call into `out` (float32 [B, H, W, 2])."""
        r = lib().osog_debug_recompose_field(self._ctx, out.data_ptr())
        if r != OSOG_OK:
            raise OsogError(r, "osog_debug_recompose_field")
        return out

    def poisson(self, lam, seed, frame):
        """int32 [n] Poisson draws of the sensor's shot-noise stream for the rates `lam` (float32 [n]) (osog_debug_poisson)."""
        lam = lam.to(device=self.device, dtype=self.torch.float32).contiguous().view(-1)
        out = self.torch.empty(lam.numel(), dtype=self.torch.int32, device=self.device)
        r = lib().osog_debug_poisson(self._ctx, lam.data_ptr(), lam.numel(), int(seed) & 0xFFFFFFFFFFFFFFFF, int(frame), out.data_ptr())
        if r != OSOG_OK:
            raise OsogError(r, "osog_debug_poisson")
        return out

    def check_guards(self):
        """Number of scratch guard bands a kernel has written into (0 = none); synchronises (osog_debug_check_guards)."""
        r = lib().osog_debug_check_guards(self._ctx)
        if r < 0:
            raise OsogError(r, "osog_debug_check_guards")
        return r

    def status(self):
        """(status bits, pairs needed) of the last render call; synchronises the stream."""
        bits, pairs = C.c_uint32(0), C.c_int64(0)
        r = lib().osog_status(self._ctx, C.byref(bits), C.byref(pairs))
        return r, bits.value, pairs.value

    def debug_bins(self):
        """(count, offset, list) of the last render call as numpy uint32 arrays."""
        nt, npairs = C.c_int64(0), C.c_int64(0)
        r = lib().osog_debug_bins(self._ctx, None, None, 0, C.byref(nt), C.byref(npairs))
        if r not in (OSOG_OK, OSOG_ECAPACITY):
            raise OsogError(r, "osog_debug_bins")
        offset = np.zeros(nt.value + 1, dtype=np.uint32)
        lst = np.zeros(npairs.value, dtype=np.uint32)
        r = lib().osog_debug_bins(self._ctx, offset.ctypes.data, lst.ctypes.data, lst.size, C.byref(nt), C.byref(npairs))
        if r != OSOG_OK:
            raise OsogError(r, "osog_debug_bins")
        return np.diff(offset).astype(np.uint32), offset, lst
