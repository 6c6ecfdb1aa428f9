/*
 * osog.h - C ABI of the B200-native OSOG forward-render hot path.
 *
 * What the library computes (citations: /root/reference/PAPER.md line numbers; readings A1-A19 and the
 * binning spec B1-B4 are listed in DESIGN.md section 3):
 *
 *   For every frame b and pixel (i, j) (row i, column j, centre x = (j + 1/2) p, y = (i + 1/2) p):
 *     OPD[b,i,j] = sum over the frame's particles n of (n_p[n] - n_medium) * thickness_n(x - cx, y - cy)
 *                  - the integrand of Eq. 2 accumulated as Eq. 7 does;
 *                  thickness = chord of the vertical line through the convex body: ellipsoid quadric, or the
 *                  half-space intersection {x | A x <= b} of Eq. 1 for the capped tetragonal prism.
 *     U[b,i,j]   = exp(i 2 pi (OPD / lambda_b + fx0 x + fy0 y)),  fx0 = sin(tilt_x) / lambda_b   (Eq. 2 with A == 1,
 *                  oblique illumination as a phase ramp)
 *     I[b]       = | IFFT2( FFT2(U[b]) * P_b ) |^2  (-> Poisson(S I) / S)  (+ sigma * z[b,i,j]),
 *                  P_b = circ(|k| / (NA_b / lambda_b)) * exp(i dz sqrt(k0^2 - kx^2 - ky^2)),  k0 = 2 pi n_medium / lambda_b
 *                  (Eq. 3, readings A9, A10, A20; I_BF; Gaussian read noise)
 *     I_DIC[b]   = | U(r + ds) e^{i theta} - U(r - ds) e^{-i theta} |^2  (*)  | IFFT2(P_b) |^2   (+ sigma * z)
 *                  (Eq. 5; ds in whole pixels, shear and convolution circular, readings A21, A22)
 *
 * Conventions
 *   - One context per (device, stream).  Every render call ENQUEUES work on the context's stream and returns
 *     without synchronising; outputs are valid once the caller has synchronised that stream.
 *   - All particle arrays and all output buffers are DEVICE pointers, caller-owned, 16-byte aligned.  The
 *     library reads the inputs, OVERWRITES the whole output (never accumulates into it) and owns only its own
 *     scratch, allocated in osog_create and freed in osog_destroy.  The hot-path calls (osog_render_opd / _field and the
 *     binning they share) never allocate.  A context's FIRST call of each of these kinds adds scratch of its own and keeps it:
 *     intensity on a power-of-two frame (kept-column buffer, twiddle tables), DIC (two complex frame batches), brightfield
 *     (one real batch), osog_backward_intensity / osog_spectral_loss (one complex batch, block sums).  Callers that must not
 *     allocate at all: osog_render_opd_static.
 *   - Results are bitwise reproducible from run to run: every pixel sums its particles in an order fixed by the
 *     data alone, never by thread scheduling (the two *_atomic alternatives are the stated exceptions).  The order is
 *     NOT plain ascending n: the tile's list is sorted ascending; a warp queues the entries that touch its 16 x 8 pixels
 *     (prisms and ellipsoids apart) and sums them in groups of 32, class by class (prisms by evaluation class, then
 *     ellipsoids), ascending n inside a class; thicknesses are fp32 values (error about 1e-7 um each)
 *     added into fp32 partial sums of at most 8 particles, which are added into the pixel's double-precision sum
 *     (DESIGN.md section 2).  Measured against the ascending double-precision sum of the oracle: <= 1.5e-6 um at OPDs of
 *     10-14 um on the five workloads.
 *   - There is no CPU fallback and no backend dispatch: without a CUDA device osog_create fails.
 *   - Return value: 0 = OK, negative = error (see the enum).  Nothing is printed, nothing throws or aborts.
 *   - Particles with a non-finite parameter, a non-positive dimension or kind > 1 are skipped (they join no
 *     tile) and set the OSOG_WBADPARTICLE bit reported by osog_status.
 */
#ifndef OSOG_H_
#define OSOG_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OSOG_API_VERSION 7   /* 2: osog_optics.defocus_um, osog_dic, osog_render_dic, osog_field_to_dic
                                3: max_pairs is a TOTAL capacity (device scan + CSR lists), osog_status reports the exact need
                                4: osog_optics.shot_noise_photons (Poisson shot noise), osog_debug_poisson, osog_debug_check_guards
                                5: osog_optics.topography_amplitude (micro-topography), brightfield, backward_params, spectral loss
                                6: osog_backward_particles
                                7: osog_render_opd_static, OSOG_ELIMIT */

enum {
    OSOG_OK = 0,
    OSOG_EINVAL = -1,     /* null / misaligned pointer, bad size, N > max_particles, B > max_frames, bad optics */
    OSOG_ECUDA = -2,      /* CUDA runtime, launch or cuFFT failure (osog_last_cuda_error gives the code)       */
    OSOG_ECAPACITY = -3,  /* the call produced more (particle, tile) pairs in total than max_pairs: its frames are zero-filled */
    OSOG_ENOMEM = -4,     /* allocation failure in osog_create                                                 */
    OSOG_ELIMIT = -5      /* osog_render_opd_static: more particles, frames or tiles than its fixed scratch holds */
};
/* status bits returned by osog_status (sticky until the next render call) */
#define OSOG_WBADPARTICLE 1u   /* at least one particle was skipped as invalid                    */
#define OSOG_WOVERFLOW    2u   /* pair list overflow happened on the device (see OSOG_ECAPACITY) */

typedef struct osog_ctx osog_ctx;   /* opaque: scratch buffers, tables, cuFFT plans */

/* Sizes fixed at creation.  struct_size = sizeof(osog_config) (ABI check). */
typedef struct {
    uint32_t struct_size;
    int32_t  device;         /* CUDA device ordinal                                                        */
    void*    stream;         /* cudaStream_t the context enqueues on (0 = legacy default stream)           */
    int32_t  H, W;           /* frame height / width in pixels, 1 .. 32768; need not be tile multiples     */
    int32_t  max_frames;     /* largest batch B of one call, >= 1                                          */
    int64_t  max_particles;  /* largest N (total over the batch) of one call, 0 .. 2^29 - 1                */
    int64_t  max_pairs;      /* capacity of the tile lists = largest TOTAL number of (particle, tile) pairs of one call
                                (the compact CSR list that the device scan addresses); 0 = 64 * max_particles + 1024.
                                How the pairs are spread over the tiles does not matter: one crowded tile may hold them all */
} osog_config;

/* Particle state, Structure of Arrays ("S in R^{N x D}"): one DEVICE array of length N per
 * column, const, caller-owned.  Frame b owns particles frame_start[b] .. frame_start[b+1]-1. */
typedef struct {
    uint32_t struct_size;
    const float *cx, *cy, *cz;        /* centre, um; cz is used by osog_render_gbuffer only (projection along z); may be NULL */
    const float *qw, *qx, *qy, *qz;   /* unit quaternion (w, x, y, z), Hamilton, active body -> world, not renormalised */
    const float *d0, *d1, *d2;        /* kind 0: semi-axes a, b, c;  kind 1: side s, length L, cap height hc (um) */
    const float *n_p;                 /* refractive index of the particle                                    */
    const uint8_t *kind;              /* 0 = ellipsoid (sphere = equal axes), 1 = capped tetragonal prism    */
    const int32_t *frame_start;       /* DEVICE int32 [B + 1], ascending, [0] = 0, [B] = N; NULL iff B == 1 */
} osog_particles;

/* Optics of one call.  lambda_um and NA are HOST arrays of length B (read before the call returns). */
typedef struct {
    uint32_t struct_size;
    int32_t  B;                       /* frames in this call, 1 .. max_frames                                */
    double   pitch_um;                /* pixel pitch p > 0                                                    */
    double   n_medium;                /* refractive index of the medium                                       */
    const double *lambda_um;          /* [B] vacuum wavelength > 0                                            */
    const double *NA;                 /* [B] numerical aperture > 0 (used by osog_render_intensity only)      */
    double   tilt_x_rad, tilt_y_rad;  /* oblique illumination: phase ramp exp(i 2 pi sin(tilt)/lambda * x); 0 = none */
    double   read_noise_sigma;        /* intensity only: I += sigma * z, z ~ N(0,1) Philox4x32-10 keyed (seed, frame, pixel); 0 = none */
    uint64_t seed;
    int32_t  pupil_enabled;           /* 0 = all-pass pupil (Parseval check), else circ(NA / lambda)          */
    double   defocus_um;              /* delta z of Eq. 3 (intensity / DIC only): the pupil is multiplied by
                                         exp(i 2 pi dz sqrt((n_medium/lambda)^2 - fx^2 - fy^2)); evanescent bins are
                                         zeroed when dz != 0; 0 = in focus (exactly the circ-only pupil)            */
    double   shot_noise_photons;      /* intensity / DIC only: expected photon count S at unit intensity; the image becomes
                                         Poisson(S max(I, 0)) / S (before the read noise), one draw per (seed, frame, pixel)
                                         from the Philox stream with counter (pixel, frame, 1, block): inversion below
                                         lambda = 10, transformed rejection (PTRS) above (reading A26); 0 = no shot noise  */
    double   topography_amplitude;    /* procedural micro-topography (reading A29), every render call: each
                                         particle's thickness at pixel (i, j) is multiplied by 1 + a * eta[b, i, j], eta ~ N(0, 1)
                                         white per pixel from the Philox stream with counter (pixel, frame, 2, 0) of `seed`, so
                                         OPD -> OPD (1 + a eta) before the phase is formed; 0 = smooth bodies                 */
} osog_optics;

/* Differential interference contrast, Eq. 5.  struct_size = sizeof(osog_dic). */
typedef struct {
    uint32_t struct_size;
    int32_t  shear_x_px, shear_y_px;  /* half shear ds in whole pixels along x (columns) / y (rows); the two copies
                                         of the field are 2 ds apart; |shear| < W resp. H; wraps around the frame   */
    double   bias_rad;                /* bias phase theta                                                         */
} osog_dic;

/* Brightfield amplitude, Eq. 4 (reading A27).  struct_size = sizeof(osog_brightfield). */
typedef struct {
    uint32_t struct_size;
    double   n_particle;              /* refractive index of the particle material for the Fresnel term (one value per call;
                                         the medium side is osog_optics.n_medium)                                          */
    double   delta_mu_per_um;         /* mu_p - mu_s of the Beer-Lambert term, 1/um                                         */
    double   caustic_gain_um;         /* C = -caustic_gain * laplacian(h); the paper gives only the proportionality         */
} osog_brightfield;

/* Create a context: allocates all scratch (records, tile ranges, per-tile counters, scan offsets, staging slices and the
 * CSR pair list, one complex frame batch and the cuFFT plans).  *out is set to NULL on failure. */
int osog_create(osog_ctx** out, const osog_config* cfg);

/* OPD frame(s): d_opd is DEVICE float [B, H, W], row-major, micrometres.  Steps H1-H6 of DESIGN.md: prepare + bounding box
 * + per-tile count (the same atomic stages the entry in the tile's slice), exclusive scan of the counts (warp shuffles, one
 * block), fill of the CSR list in ascending particle index + per-tile cull, per-tile ordered composition. */
int osog_render_opd(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, float* d_opd);

/* Complex exit wave: d_field is DEVICE float [B, H, W, 2] (interleaved re, im = complex64).  Same steps as
 * osog_render_opd with the phase-to-complex conversion and the ramp fused into the tile write-out (H7). */
int osog_render_field(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, float* d_field);

/* Coherent intensity through the circular pupil: d_intensity is DEVICE float [B, H, W].  Runs the hot path
 * into the context's own complex frame, then the library stage: cuFFT forward, pupil mask (integer
 * comparison m_x^2 H^2 + m_y^2 W^2 <= floor((NA p / lambda)^2 H^2 W^2)) and 1/(HW), cuFFT inverse, |.|^2,
 * optional read noise.  With o->defocus_um != 0 the pupil also carries the defocus phase of Eq. 3. */
int osog_render_intensity(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, float* d_intensity);

/* Library stage alone on a caller-supplied field (DEVICE complex64 [B, H, W], left untouched): used to time
 * the cuFFT stage separately from the hot path. */
int osog_field_to_intensity(osog_ctx* ctx, const osog_optics* o, const float* d_field, float* d_intensity);

/* DIC image (Eq. 5): d_dic is DEVICE float [B, H, W].  Runs the hot path into the context's own complex frame, then
 * the library stage: D = |U(r+ds) e^{i theta} - U(r-ds) e^{-i theta}|^2, cuFFT forward of D; the pupil function P
 * (circ and defocus of `o`) -> cuFFT inverse -> |h_obj|^2 -> cuFFT forward (the optical transfer function); product,
 * cuFFT inverse, real part, optional read noise (same generator as the intensity).  The transfer function depends on
 * the optics alone: it is kept in the context and rebuilt only when B, pitch, n_medium, defocus, pupil_enabled, a
 * wavelength or an NA differ from the previous DIC call.  The first DIC call of a context allocates two more complex
 * frame batches (cudaMalloc, synchronous); later calls allocate nothing. */
int osog_render_dic(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, const osog_dic* dic,
                    float* d_dic);

/* Brightfield image with the amplitude of Eq. 4: d_intensity is DEVICE float [B, H, W],
 * I_BF = |(A U_exit) * h_obj|^2 (+ shot / read noise), A = T_F(theta_i) exp(-h (mu_p - mu_s)) - gain * laplacian(h),
 * T_F = unpolarised Fresnel transmittance from n_medium into n_particle at cos theta_i = 1 / sqrt(1 + |grad h|^2)
 * (normal <-h_x, -h_y, 1> of PAPER.md:92, light along +z), h / grad h / laplacian h as osog_render_height gives them.
 * Runs the hot path twice (height map with unit index contrast, then the exit wave), one element-wise pass that multiplies
 * A into the wave, and the library stage of osog_render_intensity.  The first call allocates one real frame batch. */
int osog_render_brightfield(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, const osog_brightfield* bf,
                            float* d_intensity);

/* Library stage of osog_render_dic alone on a caller-supplied field (DEVICE complex64 [B, H, W], left untouched). */
int osog_field_to_dic(osog_ctx* ctx, const osog_optics* o, const osog_dic* dic, const float* d_field, float* d_dic);

/* Measured alternative to the ordered tile composition (paper-style scatter-add): one warp
 * per particle, global atomicAdd into d_opd.  NOT deterministic in the last bits; kept for comparison only. */
int osog_render_opd_atomic(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, float* d_opd);

/* Instance labels (reading A23; the paper's detector is trained on oriented bounding boxes,
 * PAPER.md:76, 138-146): d_obb is DEVICE float [N, 6] = (centre x, centre y, u_x, u_y, half length along u, half length
 * across u) of every particle's silhouette, centre and lengths in pixels (pixel-index coordinates c / p - 1/2), u a unit
 * vector with u_x >= 0.  Ellipsoid: principal-axis box of the silhouette ellipse; prism: box along the projected long
 * axis over the 10 projected vertices.  From the geometry alone: no clipping to the frame, no visibility test.  Invalid
 * particles give NaN.  Runs the per-particle preparation kernel only (fp64 arithmetic, results rounded to float). */
int osog_particle_obbs(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, float* d_obb);

/* Height map of the G-buffer and its derivatives (reading A25): d_h is DEVICE
 * float [B, H, W], the sum of the particles' thicknesses in um (the hot path of osog_render_opd with the index contrast
 * n_p - n_medium replaced by 1); d_grad (DEVICE float [B, H, W, 2], may be NULL) = (dh/dx, dh/dy) by central differences
 * on the pixel grid, one-sided on the frame border (the normal of PAPER.md:92 is (-g_x, -g_y, 1)); d_lap (DEVICE float
 * [B, H, W], may be NULL) = 5-point Laplacian of h in 1/um with the border pixels replicated (curvature term of Eq. 4). */
int osog_render_height(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, float* d_h, float* d_grad,
                       float* d_lap);

/* G-buffer extras (reading A24; "depth maps ... strict instance masks"): for every pixel,
 * among the frame's particles whose chord there has positive length, the one whose top surface cz + z_exit is highest
 * (+z points at the objective; this is the one call that uses cz; a NULL cz means 0, a non-finite cz removes the particle
 * from these maps).  d_top_id is DEVICE int32 [B, H, W]: that particle's index within its frame (relative to
 * frame_start[b]; ties go to the smallest index; -1 = no particle); d_depth is DEVICE float [B, H, W]: the height of that
 * top surface in um (0 where d_top_id is -1).  Runs the binning, then one fp64 evaluation per listed (particle, pixel). */
int osog_render_gbuffer(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, int32_t* d_top_id, float* d_depth);

/* osog_render_gbuffer plus the ANALYTIC normal of the visible surface: d_normal is DEVICE
 * float [B, H, W, 2] = (dz/dx, dz/dy) of the owner's top surface at the pixel centre (0, 0 where d_top_id is -1), straight from
 * the ray test: -n_x / n_z, -n_y / n_z of the active exit plane of a prism, the derivative of the quadric's upper root for an
 * ellipsoid (it grows like 1 / sqrt(w) towards the outline).  The surface normal is <-dz/dx, -dz/dy, 1> (unnormalised).
 * Unlike the finite differences of osog_render_height (reading A25) this is the slope of ONE body, the visible one. */
int osog_render_gbuffer_normals(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, int32_t* d_top_id,
                                float* d_depth, float* d_normal);

/* Adjoint of the optics stage: d_gI = dL/dI (DEVICE float [B, H, W], read only) is an upstream
 * gradient of the coherent intensity of osog_render_intensity (noise-free part); d_gopd (DEVICE float [B, H, W], overwritten)
 * receives dL/dOPD = (4 pi / lambda) Im(g_U conj(U)), g_U = F^-1{conj(P) F{d_gI V}}, V = U * h_obj.  Runs the hot path for U,
 * then 4 cuFFTs and 4 element-wise passes; the result feeds osog_backward_np / osog_backward_centre.  The first call
 * allocates one more complex frame batch (shared with the DIC path). */
int osog_backward_intensity(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, const float* d_gI, float* d_gopd);

/* The three gathers below (osog_backward_np / _centre / _params) differentiate the SMOOTH bodies: they return OSOG_EINVAL when
 * o->topography_amplitude != 0 (with micro-topography the OPD is OPD (1 + a eta), so the caller would have to multiply the
 * upstream gradient by the same per-pixel factor, which only the library can draw).
 *
 * First step of the backward pass ("the gradient of the final image with respect to the initial state
 * tensor"): the OPD frame is linear in the refractive indices, OPD = sum_n (n_p[n] - n_medium) t_n, so for an
 * upstream gradient d_gopd = dL/dOPD (DEVICE float [B, H, W], read only) the gradient is
 * d_gnp[n] = dL/dn_p[n] = sum over the pixels of the particle's frame of d_gopd * t_n  (DEVICE float [N], overwritten;
 * 0 for invalid or off-canvas particles).  One warp per particle gathers over the particle's pixel bounding box in a fixed
 * order (fp64 thickness and sum): reproducible bit for bit. */
int osog_backward_np(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, const float* d_gopd, float* d_gnp);

/* Second step of the backward pass: gradient in the particle centres.  The thickness depends on (pixel position - centre),
 * so d_gc[n] = (dL/dcx[n], dL/dcy[n]) = -(n_p[n] - n_medium) * sum over the pixels of d_gopd * grad t_n, DEVICE float [N, 2]
 * in 1/um, overwritten (0 for invalid or off-canvas particles).  grad t is analytic: the slopes of the active exit and
 * entry faces of a prism, T0 grad w / (2 sqrt w) for an ellipsoid (it grows like 1 / sqrt(w) towards the ellipsoid's
 * outline: the sum over pixel centres is finite but dominated by the outline pixels; it is the almost-everywhere derivative
 * of the pixel-sampled loss, which for ellipsoids also jumps whenever the outline crosses a pixel centre).  Same fixed-order fp64 gather as
 * osog_backward_np.  (Rotation and dimensions: osog_backward_params.) */
int osog_backward_centre(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, const float* d_gopd, float* d_gc);

/* Third step of the backward pass: gradient in the shape parameters.  d_gpar[n] = (dL/dd0, dL/dd1, dL/dd2, dL/dqw, dL/dqx,
 * dL/dqy, dL/dqz)[n] = (n_p[n] - n_medium) * sum over the pixels of d_gopd * dt_n/dtheta, DEVICE float [N, 7], overwritten
 * (0 for invalid or off-canvas particles).  d0..d2 are the semi-axes (ellipsoid) or side, length, cap height (prism), in
 * 1/um; the four quaternion components are independent variables of the rotation formula (the library never renormalises the
 * quaternion, reading A4: project the gradient onto the tangent space of the unit sphere if the caller keeps |q| = 1).
 * dt/dtheta is analytic (chain rule through R(q), the quadric M = R D R^T or the 12 planes; the active exit and entry planes
 * of a prism) and shares the caveat of osog_backward_centre for ellipsoids (it grows like 1 / sqrt(w) at the outline).
 * Works from the particle columns in fp64, same fixed-order gather as osog_backward_np. */
int osog_backward_params(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, const float* d_gopd, float* d_gpar);

/* The three gathers above in ONE pass over the pixels (the gradient "with respect to the initial state tensor"):
 * d_gnp [N], d_gc [N, 2], d_gpar [N, 7] as defined for osog_backward_np / _centre / _params; any of them may be NULL, not all.
 * dt/dtheta, grad t and t itself are linear in a few per-pixel quantities, so the pixel walk only accumulates moments (per active
 * exit / entry plane of a prism: sum of G (1, dx, dy); for an ellipsoid: sum of G / sqrt(disc) times (1, dx, dy, dx^2, dx dy,
 * dy^2) and sum of G sqrt(disc)) and all ten gradients are formed once per particle.  fp64, fixed order (reproducible bits); the
 * values agree with the separate calls up to the rounding of a different fp64 summation order.  Same argument checks. */
int osog_backward_particles(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, const float* d_gopd,
                            float* d_gnp, float* d_gc, float* d_gpar);

/* Spectral loss of Eq. 8 (reading A28) and its gradient in the image: for every frame b,
 * d_loss[b] = sum over all FFT bins of (log(|F(I_b)| + eps) - log(|F(T_b)| + eps))^2 (DEVICE double [B]), F the unnormalised
 * 2-D DFT, natural logarithm, eps > 0; d_gI (DEVICE float [B, H, W], may be NULL) receives dL/dI = Re DFT2(W),
 * W = 2 (a - b) / (|F| + eps) * conj(F) / |F|.  d_I, d_I_target: DEVICE float [B, H, W], read only.  3 cuFFTs (2 without the
 * gradient) + 3 element-wise passes; the block sums of the loss are added in a fixed order (reproducible bits).  The result
 * feeds osog_backward_intensity -> osog_backward_np / _centre / _params.  Overwrites the context's complex frames; the first
 * call allocates one more complex frame batch (shared with the DIC path) and the block-sum scratch. */
int osog_spectral_loss(osog_ctx* ctx, int32_t B, const float* d_I, const float* d_I_target, double eps, double* d_loss, float* d_gI);

/* Second measured alternative: the same tile lists, but one CTA per tile accumulates the tile in SHARED memory with fp32
 * atomics (one warp per listed particle) and writes it out once.  NOT deterministic in the last bits, fp32 sum; kept for
 * comparison with the ordered register accumulation only. */
int osog_render_opd_smem_atomic(osog_ctx* ctx, const osog_particles* p, int64_t N, const osog_optics* o, float* d_opd);

int osog_destroy(osog_ctx* ctx);

/* Synchronises the stream.  *status_bits = OSOG_W* bits of the last render call, *pairs = total number of
 * (particle, tile) pairs of that call (the device scan's total); if the call overflowed, this is exactly the max_pairs
 * that would have sufficed.  Either pointer may be NULL.
 * Returns OSOG_ECAPACITY if the last call overflowed, OSOG_ECUDA on a sticky CUDA error, else OSOG_OK. */
int osog_status(osog_ctx* ctx, uint32_t* status_bits, int64_t* pairs);

/* Test / diagnostics: synchronises, then copies the binning of the last render call to HOST arrays, as the device holds
 * it: h_offset [n_tiles + 1] = the exclusive scan of the per-tile counts (H3), h_list [min(pairs, cap)] = the CSR list,
 * each tile's segment in ascending particle index (H4; filled by calls that run the sort: every osog_render_* except
 * osog_render_opd_atomic).  Tile id = frame * tiles_per_frame + (i / T) * ceil(W / T) + (j / T).
 * Any pointer may be NULL.  *n_tiles and *n_pairs are always written. */
int osog_debug_bins(osog_ctx* ctx, uint32_t* h_offset, uint32_t* h_list, int64_t cap,
                    int64_t* n_tiles, int64_t* n_pairs);

/* Test / measurement: re-runs ONLY the composition kernel (H5-H7) of the last call on its binning (tile lists, records,
 * optics are still in the context) and writes the complex field again.  Lets bench.py time the dominant
 * kernel alone with CUDA events.  OSOG_EINVAL unless the last call on this context was one of osog_render_opd / _field /
 * _intensity / _dic / _height or osog_backward_intensity (the calls that leave sorted lists and a composition behind). */
int osog_debug_recompose_field(osog_ctx* ctx, float* d_field);

/* Test hook of the shot noise (reading A26): d_counts[k] = the Poisson((double)d_lambda[k]) draw of
 * pixel k of frame `frame` under `seed` (DEVICE float [n] in, DEVICE int32 [n] out), exactly the draw the sensor stage
 * takes; lets the tests compare the integer draw with the oracle's bit for bit on given rates. */
int osog_debug_poisson(osog_ctx* ctx, const float* d_lambda, int64_t n, uint64_t seed, uint32_t frame, int32_t* d_counts);

/* Test / diagnostics: every scratch array of the context (records, tile ranges, counters, offsets, staging slices, CSR
 * list, meta words, optics, status, complex frames) is followed by a 256-byte guard band written once in
 * osog_create.  Synchronises and returns the number of guard bands that no longer hold their pattern (0 = no kernel wrote
 * past the end of its scratch), or a negative error code.  (compute-sanitizer is not available on every pool.) */
int osog_debug_check_guards(osog_ctx* ctx);

/* The hot path for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): osog_render_opd (H1-H6, the same three kernels, the same bits) without a context.  All scratch of the call lives in
 * ONE file-scope device array of OSOG_STATIC_SCRATCH_BYTES (about 2.5 MB) that every GPU loading the library holds until exit; the
 * call itself calls no cudaMalloc / cudaFree / cudaMallocHost and no allocating library routine (no cuFFT).  Fixed limits, beyond
 * which the call returns OSOG_ELIMIT and enqueues nothing:
 *   N <= OSOG_STATIC_MAX_PARTICLES, o->B <= OSOG_STATIC_MAX_FRAMES, o->B * ceil(H / 32) * ceil(W / 32) <= OSOG_STATIC_MAX_TILES
 *   (one 512 x 512 frame, four 256 x 256 frames, ...).
 * A call that produces more than OSOG_STATIC_MAX_PAIRS (particle, tile) pairs zero-fills d_opd and sets OSOG_WOVERFLOW, as
 * osog_render_opd does beyond max_pairs.
 * device: CUDA device ordinal (the pointers below live there); stream: cudaStream_t the work is enqueued on (NULL = default).
 * p, N, o: as for osog_render_opd (DEVICE columns, host structs; read only).  d_opd: DEVICE float [B, H, W], 16-byte aligned,
 * overwritten.  d_status_bits: DEVICE uint32 [1] or NULL; receives the call's warning bits (OSOG_W*) by a 4-byte
 * device-to-device copy enqueued behind the kernels (there is no osog_status for this call: read the word after the stream has
 * finished).  Enqueue-only, never synchronises.
 * EVERY call on a GPU shares the one array, which keeps the last call's contents: the call first clears what must start at zero
 * (tile counters, scan ticket, status words; three small memsets on `stream`).  Two calls that OVERLAP on the GPU (different
 * streams without an ordering between them, or a captured graph replayed concurrently with itself) RACE on the scratch and
 * produce garbage: order them.  Host threads are serialised by a mutex for the duration of the enqueue only. */
#define OSOG_STATIC_MAX_PARTICLES 4096
#define OSOG_STATIC_MAX_FRAMES 4
#define OSOG_STATIC_MAX_TILES 256
#define OSOG_STATIC_MAX_PAIRS 65536
#define OSOG_STATIC_SCRATCH_BYTES (2560 * 1024)
int osog_render_opd_static(int device, void* stream, int H, int W, const osog_particles* p, int64_t N, const osog_optics* o,
                           float* d_opd, uint32_t* d_status_bits);

/* Tile edge T in pixels (build-time constant of the binning, B3). */
int osog_tile_size(void);

/* Last CUDA / cuFFT error code seen by this context (0 = none). */
int osog_last_cuda_error(const osog_ctx* ctx);

const char* osog_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* OSOG_H_ */
