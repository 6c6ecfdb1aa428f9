// Library stage (timed separately from the hot path, L1-L3):
// pupil function circ(|k| / (NA / lambda)) exp(i dz k_z) with the 1/(HW) normalisation (Eq. 3),
// the DIC shear-and-interfere step and the element-wise helpers of its incoherent convolution (Eq. 5),
// and the sensor: I = |.|^2 plus optional Poisson shot noise and Gaussian read noise from
// Philox4x32-10.  First half of the file: the element-wise kernels that go around cuFFT (any frame size).  Second half
// ("L1-L3 fused and pruned"): the whole stage as three FFT kernels of this library for power-of-two frames.
#include "osog_internal.cuh"

namespace osog {

// Bin (ky, kx) of the unshifted FFT grid has signed index m = k for k <= (n-1)/2, else k - n.
// It passes iff m_x^2 H^2 + m_y^2 W^2 <= floor((NA p / lambda)^2 H^2 W^2)  (64-bit integers, reading A10).
// DEFOCUS: the passing bin is also multiplied by exp(i 2 pi dz sqrt((n_m / lambda)^2 - fx^2 - fy^2)), f = m / (W p)
// (Eq. 3, reading A20): turns in fp64, reduced to [-1/2, 1/2], sincospi in fp32; evanescent bins
// (m_x^2 H^2 + m_y^2 W^2 > floor((n_m p / lambda)^2 H^2 W^2)) are zeroed.
// Returns the pupil value of the bin times `scale` (0 = blocked).
template <bool DEFOCUS>
__device__ __forceinline__ float2 pupil_value(const FrameOptics& fo, int kx, int ky, int H, int W, double inv_wp,
                                              double inv_hp, float scale)
{
    const long long mx = kx <= (W - 1) / 2 ? kx : kx - W;
    const long long my = ky <= (H - 1) / 2 ? ky : ky - H;
    const long long lhs = mx * mx * ((long long)H * H) + my * my * ((long long)W * W);
    bool pass = fo.pupil_thresh < 0 || lhs <= fo.pupil_thresh;
    if (!DEFOCUS) return make_float2(pass ? scale : 0.0f, 0.0f);
    pass = pass && (fo.prop_thresh < 0 || lhs <= fo.prop_thresh);
    if (!pass) return make_float2(0.0f, 0.0f);
    const double fx = (double)mx * inv_wp, fy = (double)my * inv_hp;
    const double rad = fo.nm_over_lambda_sq - fx * fx - fy * fy;
    double turns = fo.defocus_um * sqrt(fmax(rad, 0.0));
    turns -= rint(turns);
    float sn, cs;
    sincospif(2.0f * (float)turns, &sn, &cs);
    return make_float2(cs * scale, sn * scale);
}

// spec *= P * scale (in place), or with FILL: spec = P * scale
// imag_sign = -1: multiply by conj(P) (adjoint of the optics stage); only the defocus phase has an imaginary part
template <bool DEFOCUS, bool FILL>
__global__ void __launch_bounds__(256) k_pupil(float2* __restrict__ spec, const FrameOptics* __restrict__ optics,
                                               int H, int W, double inv_wp, double inv_hp, float scale, float imag_sign)
{
    const int kx = blockIdx.x * blockDim.x + threadIdx.x;
    const int ky = blockIdx.y, b = blockIdx.z;
    if (kx >= W) return;
    float2 pv = pupil_value<DEFOCUS>(optics[b], kx, ky, H, W, inv_wp, inv_hp, scale);
    if (DEFOCUS) pv.y *= imag_sign;
    const size_t idx = ((size_t)b * H + ky) * W + kx;
    if (FILL) {
        spec[idx] = pv;
    } else {
        const float2 v = spec[idx];
        spec[idx] = DEFOCUS ? make_float2(v.x * pv.x - v.y * pv.y, v.x * pv.y + v.y * pv.x)
                            : make_float2(v.x * pv.x, v.y * pv.x);
    }
}

// DIC, Eq. 5: out = (|U(r + ds) e^{i theta} - U(r - ds) e^{-i theta}|^2, 0); ds = (sx, sy) whole
// pixels, indices wrap around the frame (readings A21, A22).  e = (cos theta, sin theta).
__global__ void __launch_bounds__(256) k_dic_shear(const float2* __restrict__ field, float2* __restrict__ out, int H,
                                                   int W, int sx, int sy, float2 e)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = blockIdx.y, b = blockIdx.z;
    if (j >= W) return;
    int jp = j + sx, jm = j - sx, ip = i + sy, im = i - sy;         // |sx| < W, |sy| < H
    jp += jp < 0 ? W : (jp >= W ? -W : 0);
    jm += jm < 0 ? W : (jm >= W ? -W : 0);
    ip += ip < 0 ? H : (ip >= H ? -H : 0);
    im += im < 0 ? H : (im >= H ? -H : 0);
    const float2* f = field + (size_t)b * H * W;
    const float2 up = f[(size_t)ip * W + jp], um = f[(size_t)im * W + jm];
    const float dr = (up.x * e.x - up.y * e.y) - (um.x * e.x + um.y * e.y);
    const float di = (up.x * e.y + up.y * e.x) - (um.y * e.x - um.x * e.y);
    out[((size_t)b * H + i) * W + j] = make_float2(dr * dr + di * di, 0.0f);
}

// G-buffer (reading A25): finite differences of the height map h on the pixel grid.  grad = (g_x, g_y) interleaved:
// central differences inside, one-sided on the frame border; lap = 5-point Laplacian with the border pixels replicated.
__global__ void __launch_bounds__(256) k_height_stencil(const float* __restrict__ h, int H, int W, float inv_p,
                                                        float2* __restrict__ grad, float* __restrict__ lap)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = blockIdx.y, b = blockIdx.z;
    if (j >= W) return;
    const float* f = h + (size_t)b * H * W;
    const int jm = max(j - 1, 0), jp = min(j + 1, W - 1), im = max(i - 1, 0), ip = min(i + 1, H - 1);
    const float c = f[(size_t)i * W + j];
    const float xl = f[(size_t)i * W + jm], xr = f[(size_t)i * W + jp];
    const float yu = f[(size_t)im * W + j], yd = f[(size_t)ip * W + j];
    const size_t idx = ((size_t)b * H + i) * W + j;
    if (grad != nullptr) {
        const float gx = jp > jm ? (xr - xl) * (inv_p / (float)(jp - jm)) : 0.0f;
        const float gy = ip > im ? (yd - yu) * (inv_p / (float)(ip - im)) : 0.0f;
        grad[idx] = make_float2(gx, gy);
    }
    if (lap != nullptr) lap[idx] = ((xl + xr) + (yu + yd) - 4.0f * c) * (inv_p * inv_p);
}

cudaError_t launch_brightfield(osog_ctx* c, int B, float2* field, const float* d_h, double pitch, double n1, double n2,
                               double dmu, double gain);
// Brightfield amplitude, Eq. 4 (reading A27), multiplied into the exit wave in place:
// A = T_F(theta_i) exp(-h dmu) + C, cos theta_i = 1 / sqrt(1 + |grad h|^2) (normal <-h_x, -h_y, 1>, light along +z), T_F the
// unpolarised Fresnel transmittance from index n1 into n2, C = -gain lap h; grad h and lap h are the finite differences of
// reading A25 (k_height_stencil's formulas), taken here straight from the height map.
__global__ void __launch_bounds__(256) k_brightfield(float2* __restrict__ field, const float* __restrict__ h, int H, int W,
                                                     float inv_p, float n1, float n2, float dmu, float gain)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = blockIdx.y, b = blockIdx.z;
    if (j >= W) return;
    const float* f = h + (size_t)b * H * W;
    const int jm = max(j - 1, 0), jp = min(j + 1, W - 1), im = max(i - 1, 0), ip = min(i + 1, H - 1);
    const float c = f[(size_t)i * W + j];
    const float xl = f[(size_t)i * W + jm], xr = f[(size_t)i * W + jp];
    const float yu = f[(size_t)im * W + j], yd = f[(size_t)ip * W + j];
    const float gx = jp > jm ? (xr - xl) * (inv_p / (float)(jp - jm)) : 0.0f;
    const float gy = ip > im ? (yd - yu) * (inv_p / (float)(ip - im)) : 0.0f;
    const float lap = ((xl + xr) + (yu + yd) - 4.0f * c) * (inv_p * inv_p);
    const float g2 = gx * gx + gy * gy;
    float T = 1.0f;
    if (n1 != n2) {
        const float ci = rsqrtf(1.0f + g2);                      // cos theta_i
        const float si2 = g2 / (1.0f + g2);                      // sin^2 theta_i (no cancellation near normal incidence)
        const float r = n1 / n2, st2 = r * r * si2;
        if (st2 > 1.0f) {
            T = 0.0f;                                            // total internal reflection
        } else {
            const float ct = sqrtf(1.0f - st2);
            const float as = n1 * ci, bs = n2 * ct, ap = n1 * ct, bp = n2 * ci;
            const float rs = (as - bs) / (as + bs), rp = (ap - bp) / (ap + bp);
            T = 1.0f - 0.5f * (rs * rs + rp * rp);
        }
    }
    const float A = T * expf(-c * dmu) - gain * lap;
    const size_t idx = ((size_t)b * H + i) * W + j;
    const float2 u = field[idx];
    field[idx] = make_float2(u.x * A, u.y * A);
}

cudaError_t launch_brightfield(osog_ctx* c, int B, float2* field, const float* d_h, double pitch, double n1, double n2,
                               double dmu, double gain)
{
    const dim3 grid((c->W + 255) / 256, c->H, B);
    k_brightfield<<<grid, 256, 0, c->stream>>>(field, d_h, c->H, c->W, (float)(1.0 / pitch), (float)n1, (float)n2, (float)dmu,
                                              (float)gain);
    return cudaGetLastError();
}

// ---- spectral loss of Eq. 8 (reading A28) and its gradient in the image -----------------
__global__ void __launch_bounds__(256) k_real_to_complex(const float* __restrict__ a, const float* __restrict__ b,
                                                         float2* __restrict__ ca, float2* __restrict__ cb, size_t n)
{
    const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    ca[k] = make_float2(a[k], 0.0f);
    cb[k] = make_float2(b[k], 0.0f);
}

// per bin: d = log(|F| + eps) - log(|T| + eps); partial[b][block] = sum of d^2 over the block's bins (fixed order);
// F <- W = 2 d / (|F| + eps) * conj(F) / |F|  (0 where F = 0): the forward DFT of W has dL/dI as its real part
__global__ void __launch_bounds__(256) k_spectral_terms(float2* __restrict__ F, const float2* __restrict__ T, size_t npx, double eps,
                                                        double* __restrict__ partial, int want_grad)
{
    __shared__ double s_sum[8];
    const size_t pix = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int b = blockIdx.y;
    double d2 = 0.0;
    if (pix < npx) {
        const float2 f = F[(size_t)b * npx + pix], t = T[(size_t)b * npx + pix];
        const double af = sqrt((double)f.x * f.x + (double)f.y * f.y), at = sqrt((double)t.x * t.x + (double)t.y * t.y);
        const double d = log(af + eps) - log(at + eps);
        d2 = d * d;
        if (want_grad) {
            const double w = af > 0.0 ? 2.0 * d / ((af + eps) * af) : 0.0;
            F[(size_t)b * npx + pix] = make_float2((float)(w * f.x), (float)(-w * f.y));
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) d2 += __shfl_xor_sync(0xffffffffu, d2, o);
    if ((threadIdx.x & 31) == 0) s_sum[threadIdx.x >> 5] = d2;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) v += s_sum[w];
        partial[(size_t)b * gridDim.x + blockIdx.x] = v;
    }
}

// loss[b] = sum of the frame's block partials, in a fixed order (one block per frame)
__global__ void __launch_bounds__(256) k_sum_partials(const double* __restrict__ partial, int nblk, double* __restrict__ loss)
{
    __shared__ double s_sum[8];
    const int b = blockIdx.x;
    double v = 0.0;
    for (int k = threadIdx.x; k < nblk; k += 256) v += partial[(size_t)b * nblk + k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) s_sum[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) t += s_sum[w];
        loss[b] = t;
    }
}

__global__ void __launch_bounds__(256) k_real_part(const float2* __restrict__ c, float* __restrict__ out, size_t n)
{
    const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) out[k] = c[k].x;
}

cudaError_t launch_real_to_complex(osog_ctx* c, int B, const float* a, const float* b, float2* ca, float2* cb)
{
    const size_t n = (size_t)B * c->H * c->W;
    k_real_to_complex<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(a, b, ca, cb, n);
    return cudaGetLastError();
}

cudaError_t launch_spectral_terms(osog_ctx* c, int B, float2* F, const float2* T, double eps, double* partial, double* d_loss, bool want_grad)
{
    const size_t npx = (size_t)c->H * c->W;
    const unsigned nblk = (unsigned)((npx + 255) / 256);
    k_spectral_terms<<<dim3(nblk, B), 256, 0, c->stream>>>(F, T, npx, eps, partial, want_grad ? 1 : 0);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    k_sum_partials<<<B, 256, 0, c->stream>>>(partial, (int)nblk, d_loss);
    return cudaGetLastError();
}

cudaError_t launch_real_part(osog_ctx* c, int B, const float2* in, float* out)
{
    const size_t n = (size_t)B * c->H * c->W;
    k_real_part<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(in, out, n);
    return cudaGetLastError();
}

// buf = (|buf|^2 * scale, 0)
__global__ void __launch_bounds__(256) k_abs2(float2* __restrict__ buf, size_t n, float scale)
{
    const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const float2 v = buf[k];
    buf[k] = make_float2((v.x * v.x + v.y * v.y) * scale, 0.0f);
}

// a = a * b * scale (complex)
__global__ void __launch_bounds__(256) k_cmul(float2* __restrict__ a, const float2* __restrict__ b, size_t n, float scale)
{
    const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const float2 x = a[k], y = b[k];
    a[k] = make_float2((x.x * y.x - x.y * y.y) * scale, (x.x * y.y + x.y * y.x) * scale);
}

// Standard normal of the read noise (reading A13): stream 0 of the shared Philox generator (osog_internal.cuh)
__device__ __forceinline__ float read_noise_z(uint64_t seed, uint32_t frame, uint32_t pixel)
{
    return philox_normal(seed, frame, pixel, 0u);
}

// ---- Poisson shot noise ("P(lambda) + G(0, sigma^2)"; reading A26) ---------------------
// Two uniforms in [0, 1) with 53 random bits each from block `block` of the shot-noise stream of (seed, frame, pixel):
// Philox4x32-10, key = (seed low, seed high), counter = (pixel, frame, 1, block); u_a = ((r0 >> 5) 2^26 + (r1 >> 6)) 2^-53.
__device__ __forceinline__ void shot_uniforms(uint64_t seed, uint32_t frame, uint32_t pixel, uint32_t block, double* ua, double* ub)
{
    uint32_t c[4] = {pixel, frame, 1u, block};
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        philox_round(c, k0, k1);
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    *ua = ((double)(c[0] >> 5) * 67108864.0 + (double)(c[1] >> 6)) * 1.1102230246251565e-16;
    *ub = ((double)(c[2] >> 5) * 67108864.0 + (double)(c[3] >> 6)) * 1.1102230246251565e-16;
}

// One Poisson(lam) draw, a pure function of (seed, frame, pixel, lam), all decisions in fp64.  lam < 10: inversion by
// sequential search with the first uniform of block 0 (smallest k with CDF(k) >= u, terms by p_j = p_{j-1} lam / j).
// lam >= 10: Hoermann's transformed rejection with squeeze (PTRS, 1993), round j using the two uniforms of block j.
__device__ double poisson_draw(double lam, uint64_t seed, uint32_t frame, uint32_t pixel)
{
    if (!(lam > 0.0)) return 0.0;
    double ua, ub;
    if (lam < 10.0) {
        shot_uniforms(seed, frame, pixel, 0u, &ua, &ub);
        double p = exp(-lam), F = p;
        int k = 0;
        while (ua > F && k < 200) {
            ++k;
            p = p * lam / (double)k;
            F += p;
        }
        return (double)k;
    }
    const double slam = sqrt(lam), b = 0.931 + 2.53 * slam, a = -0.059 + 0.02483 * b;
    const double inv_alpha = 1.1239 + 1.1328 / (b - 3.4), vr = 0.9277 - 3.6224 / (b - 2.0);
    const double llam = log(lam);
    for (uint32_t block = 0; block <= 1000u; ++block) {
        shot_uniforms(seed, frame, pixel, block, &ua, &ub);
        const double U = ua - 0.5, V = ub, us = 0.5 - fabs(U);
        const double k = floor((2.0 * a / us + b) * U + lam + 0.43);
        if (us >= 0.07 && V <= vr) return k;
        if (k < 0.0 || (us < 0.013 && V > us)) continue;
        if (log(V) + log(inv_alpha) - log(a / (us * us) + b) <= -lam + k * llam - lgamma(k + 1.0)) return k;
    }
    return floor(lam);                                           // (never reached: the acceptance rate is > 0.85)
}

// REAL = false: I = |img|^2; REAL = true: I = Re img (the DIC image is a real convolution).  Then the
// sensor: photon counting I <- Poisson(photons max(I, 0)) / photons (photons = 0: off), read noise + sigma z.
template <bool REAL, bool SHOT>
__global__ void __launch_bounds__(256) k_sensor(const float2* __restrict__ img, float* __restrict__ out, int H, int W,
                                                float sigma, double photons, uint64_t seed)
{
    const size_t npx = (size_t)H * W;
    const size_t pix = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int b = blockIdx.y;
    if (pix >= npx) return;
    const float2 v = img[(size_t)b * npx + pix];
    float I = REAL ? v.x : v.x * v.x + v.y * v.y;
    if (SHOT) I = (float)(poisson_draw(photons * fmax((double)I, 0.0), seed, (uint32_t)b, (uint32_t)pix) / photons);
    if (sigma != 0.0f) I = fmaf(sigma, read_noise_z(seed, (uint32_t)b, (uint32_t)pix), I);
    out[(size_t)b * npx + pix] = I;
}

// test hook: counts[k] = Poisson((double)lam[k]) for pixel k of `frame`
__global__ void __launch_bounds__(256) k_poisson(const float* __restrict__ lam, size_t n, uint64_t seed, uint32_t frame,
                                                 int32_t* __restrict__ counts)
{
    const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) counts[k] = (int32_t)poisson_draw((double)lam[k], seed, frame, (uint32_t)k);
}

cudaError_t launch_poisson(osog_ctx* c, const float* d_lam, size_t n, uint64_t seed, uint32_t frame, int32_t* d_counts)
{
    if (n == 0) return cudaSuccess;
    k_poisson<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(d_lam, n, seed, frame, d_counts);
    return cudaGetLastError();
}

static cudaError_t pupil_launch(osog_ctx* c, int B, float2* spec, double pitch, bool defocus, bool fill, float scale,
                                float imag_sign = 1.0f)
{
    const dim3 grid((c->W + 255) / 256, c->H, B);
    const double inv_wp = 1.0 / ((double)c->W * pitch), inv_hp = 1.0 / ((double)c->H * pitch);
    if (fill) {
        if (defocus) k_pupil<true, true><<<grid, 256, 0, c->stream>>>(spec, c->optics, c->H, c->W, inv_wp, inv_hp, scale, imag_sign);
        else k_pupil<false, true><<<grid, 256, 0, c->stream>>>(spec, c->optics, c->H, c->W, inv_wp, inv_hp, scale, imag_sign);
    } else {
        if (defocus) k_pupil<true, false><<<grid, 256, 0, c->stream>>>(spec, c->optics, c->H, c->W, inv_wp, inv_hp, scale, imag_sign);
        else k_pupil<false, false><<<grid, 256, 0, c->stream>>>(spec, c->optics, c->H, c->W, inv_wp, inv_hp, scale, imag_sign);
    }
    return cudaGetLastError();
}

cudaError_t launch_pupil(osog_ctx* c, int B, float2* spec, double pitch, bool defocus)
{
    return pupil_launch(c, B, spec, pitch, defocus, false, (float)(1.0 / ((double)c->H * c->W)));
}

cudaError_t launch_pupil_conj(osog_ctx* c, int B, float2* spec, double pitch, bool defocus)
{
    return pupil_launch(c, B, spec, pitch, defocus, false, (float)(1.0 / ((double)c->H * c->W)), -1.0f);
}

// Adjoint of the optics stage: v *= g (g real, per pixel): g_V = G_I V
__global__ void __launch_bounds__(256) k_mul_real(float2* __restrict__ v, const float* __restrict__ g, size_t n)
{
    const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const float2 x = v[k];
    const float s = g[k];
    v[k] = make_float2(x.x * s, x.y * s);
}

// dL/dOPD = (4 pi / lambda) Im(g_U conj(U))
__global__ void __launch_bounds__(256) k_gopd(const float2* __restrict__ gu, const float2* __restrict__ u,
                                              const FrameOptics* __restrict__ optics, size_t npx, float* __restrict__ gopd)
{
    const size_t pix = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int b = blockIdx.y;
    if (pix >= npx) return;
    const float2 a = gu[(size_t)b * npx + pix], w = u[(size_t)b * npx + pix];
    const float k = (float)(12.566370614359172 * optics[b].inv_lambda);
    gopd[(size_t)b * npx + pix] = k * (a.y * w.x - a.x * w.y);
}

cudaError_t launch_mul_real(osog_ctx* c, int B, float2* v, const float* g)
{
    const size_t n = (size_t)B * c->H * c->W;
    k_mul_real<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(v, g, n);
    return cudaGetLastError();
}

cudaError_t launch_gopd(osog_ctx* c, int B, const float2* gu, const float2* u, float* d_gopd)
{
    const size_t npx = (size_t)c->H * c->W;
    const dim3 grid((unsigned)((npx + 255) / 256), B);
    k_gopd<<<grid, 256, 0, c->stream>>>(gu, u, c->optics, npx, d_gopd);
    return cudaGetLastError();
}

cudaError_t launch_pupil_fill(osog_ctx* c, int B, float2* spec, double pitch, bool defocus)
{
    return pupil_launch(c, B, spec, pitch, defocus, true, 1.0f);
}

cudaError_t launch_dic_shear(osog_ctx* c, int B, const float2* field, float2* out, int sx, int sy, double theta)
{
    const dim3 grid((c->W + 255) / 256, c->H, B);
    k_dic_shear<<<grid, 256, 0, c->stream>>>(field, out, c->H, c->W, sx, sy, make_float2((float)cos(theta), (float)sin(theta)));
    return cudaGetLastError();
}

cudaError_t launch_height_stencil(osog_ctx* c, int B, const float* d_h, double pitch, float* d_grad, float* d_lap)
{
    const dim3 grid((c->W + 255) / 256, c->H, B);
    k_height_stencil<<<grid, 256, 0, c->stream>>>(d_h, c->H, c->W, (float)(1.0 / pitch), reinterpret_cast<float2*>(d_grad), d_lap);
    return cudaGetLastError();
}

cudaError_t launch_abs2(osog_ctx* c, int B, float2* buf, double scale)
{
    const size_t n = (size_t)B * c->H * c->W;
    k_abs2<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(buf, n, (float)scale);
    return cudaGetLastError();
}

cudaError_t launch_cmul(osog_ctx* c, int B, float2* a, const float2* b, double scale)
{
    const size_t n = (size_t)B * c->H * c->W;
    k_cmul<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(a, b, n, (float)scale);
    return cudaGetLastError();
}

cudaError_t launch_sensor(osog_ctx* c, int B, const float2* img, float* d_intensity, double sigma, double photons, uint64_t seed)
{
    const size_t npx = (size_t)c->H * c->W;
    const dim3 grid((unsigned)((npx + 255) / 256), B);
    if (photons != 0.0) k_sensor<false, true><<<grid, 256, 0, c->stream>>>(img, d_intensity, c->H, c->W, (float)sigma, photons, seed);
    else k_sensor<false, false><<<grid, 256, 0, c->stream>>>(img, d_intensity, c->H, c->W, (float)sigma, photons, seed);
    return cudaGetLastError();
}

cudaError_t launch_sensor_real(osog_ctx* c, int B, const float2* img, float* d_out, double sigma, double photons, uint64_t seed)
{
    const size_t npx = (size_t)c->H * c->W;
    const dim3 grid((unsigned)((npx + 255) / 256), B);
    if (photons != 0.0) k_sensor<true, true><<<grid, 256, 0, c->stream>>>(img, d_out, c->H, c->W, (float)sigma, photons, seed);
    else k_sensor<true, false><<<grid, 256, 0, c->stream>>>(img, d_out, c->H, c->W, (float)sigma, photons, seed);
    return cudaGetLastError();
}


// ---- L1-L3 fused and pruned (power-of-two frames): row FFT -> [column FFT, pupil, inverse column FFT] -> inverse row FFT + sensor ----
// The pupil passes |m_x| <= r_x only (NA 0.65 on config 4: 487 of 2048 columns), so after the forward row transforms only
// those columns are kept (written transposed, one contiguous column each), one kernel does the forward column transform,
// the pupil and the inverse column transform of the kept columns, and the inverse row transforms read the kept columns back
// into zero-filled rows and end in the sensor.  Three kernels and ~85 MB of traffic per 2048^2 frame instead of six (two
// cuFFT launches of two kernels each, pupil, sensor) and 385 MB.
// The transforms: n / 8 threads per row, 8 complex values per thread in registers, decimation in frequency with the radix
// sequence r1, 8, 8, ... (r1 = 2, 4 or 8 takes what the power of two leaves), one shared-memory exchange between two stages.
// The spectrum stays in digit-reversed order (the pupil only needs to know which frequency sits where) and the inverse runs
// the conjugate-transposed stages in reverse order: no reordering pass, and the stage next to the pupil needs no exchange.
constexpr int kFoThreads = 512;                     // threads per CTA (one row of 4096, two of 2048, ...)

// compile-time plan of a transform of length n = 2^LG = 2^lg_r1 * 8^(nstage - 1): every shift below is a constant and every
// stage loop unrolls (the run-time version of this code spent two thirds of its instructions on index arithmetic)
template <int LG>
struct FoPlan {
    static constexpr int lg_n = LG, n = 1 << LG;
    static constexpr int lg_r1 = LG % 3 == 0 ? 3 : LG % 3;
    static constexpr int nstage = 1 + (LG - lg_r1) / 3;
};

// position p of the digit-reversed spectrum holds frequency k:  p = m1 n/r1 + m2 n/(r1 r2) + ...,  k = m1 + r1 (m2 + r2 (...))
template <class PL>
__device__ __forceinline__ int fo_freq_of_pos(int p)
{
    int lg_L = PL::lg_n - PL::lg_r1;
    int k = p >> lg_L, sh = PL::lg_r1;
    p &= (1 << lg_L) - 1;
#pragma unroll
    for (int s = 1; s < PL::nstage; ++s) {
        lg_L -= 3;
        k += (p >> lg_L) << sh;
        p &= (1 << lg_L) - 1;
        sh += 3;
    }
    return k;
}
template <class PL>
__device__ __forceinline__ int fo_pos_of_freq(int k)
{
    int lg_L = PL::lg_n - PL::lg_r1;
    int p = (k & ((1 << PL::lg_r1) - 1)) << lg_L;
    k >>= PL::lg_r1;
#pragma unroll
    for (int s = 1; s < PL::nstage; ++s) {
        lg_L -= 3;
        p += (k & 7) << lg_L;
        k >>= 3;
    }
    return p;
}

__device__ __forceinline__ float2 fo_cmul(float2 a, float2 w) { return make_float2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x); }
__device__ __forceinline__ float2 fo_cmulc(float2 a, float2 w) { return make_float2(a.x * w.x + a.y * w.y, a.y * w.x - a.x * w.y); }   // a conj(w)
__device__ __forceinline__ float2 fo_conj(float2 a) { return make_float2(a.x, -a.y); }
// complex add / subtract as ONE packed instruction (Blackwell add.f32x2): the butterflies are issue bound
__device__ __forceinline__ float2 fo_add(float2 a, float2 b)
{
    unsigned long long ra, rb, rd;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(b.x), "f"(b.y));
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(rd));
    return d;
}
__device__ __forceinline__ float2 fo_sub(float2 a, float2 b)
{
    unsigned long long ra, rb, rd;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(b.x), "f"(b.y));
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(rd));
    return d;
}

// y_m = sum_j a_j w4^{j m}, w4 = exp(-2 pi i / 4) = -i (forward), in place
__device__ __forceinline__ void fo_r4(float2& a0, float2& a1, float2& a2, float2& a3)
{
    const float2 s02 = fo_add(a0, a2), d02 = fo_sub(a0, a2), s13 = fo_add(a1, a3), d13 = fo_sub(a1, a3);
    a0 = fo_add(s02, s13);
    a2 = fo_sub(s02, s13);
    a1 = make_float2(d02.x + d13.y, d02.y - d13.x);               // d02 - i d13
    a3 = make_float2(d02.x - d13.y, d02.y + d13.x);               // d02 + i d13
}
// y_m = sum_j a_j w8^{j m}, w8 = exp(-2 pi i / 8) (forward), in place: a[m] <- y_m
__device__ __forceinline__ void fo_r8(float2 (&a)[8])
{
    const float h = 0.70710678118654752f;
    float2 s0 = fo_add(a[0], a[4]), s1 = fo_add(a[1], a[5]), s2 = fo_add(a[2], a[6]), s3 = fo_add(a[3], a[7]);
    float2 d0 = fo_sub(a[0], a[4]), d1 = fo_sub(a[1], a[5]), d2 = fo_sub(a[2], a[6]), d3 = fo_sub(a[3], a[7]);
    d1 = make_float2((d1.x + d1.y) * h, (d1.y - d1.x) * h);       // d1 (1 - i) / sqrt 2
    d2 = make_float2(d2.y, -d2.x);                                // -i d2
    d3 = make_float2((d3.y - d3.x) * h, -(d3.x + d3.y) * h);      // d3 (-1 - i) / sqrt 2
    fo_r4(s0, s1, s2, s3);                                        // even outputs y0 y2 y4 y6
    fo_r4(d0, d1, d2, d3);                                        // odd outputs  y1 y3 y5 y7
    a[0] = s0; a[2] = s1; a[4] = s2; a[6] = s3;
    a[1] = d0; a[3] = d1; a[5] = d2; a[7] = d3;
}

// shared-memory index of row position p: one pad element per 8 keeps the strided exchanges (sub = 1, 8, 64 ...) off the same banks
__device__ __forceinline__ int fo_phys(int p) { return p + (p >> 3); }
// element stride of positions p0 + k sub (sub = 1 or a multiple of 8, p0 + 7 sub inside one block) in the padded layout
__device__ __forceinline__ int fo_stride(int lg_sub) { return lg_sub >= 3 ? 9 << (lg_sub - 3) : 1; }

// twiddles of one butterfly: a[m] *= w^m (forward) or its conjugate (inverse), w = tw[q << lg_step], tw[k] = exp(-2 pi i k / n);
// w, w^2, w^4 come from the table, the other four powers by one multiplication each (error ~ 1e-7; three loads instead of seven)
template <bool INV>
__device__ __forceinline__ void fo_twiddle8(float2 (&a)[8], int q, int lg_step, const float2* __restrict__ tw)
{
    const int i1 = q << lg_step;
    const float2 w1 = __ldg(tw + i1), w2 = __ldg(tw + 2 * i1), w4 = __ldg(tw + 4 * i1);
    const float2 w3 = fo_cmul(w1, w2), w5 = fo_cmul(w4, w1), w6 = fo_cmul(w4, w2), w7 = fo_cmul(w4, w3);
    const float2 w[8] = {make_float2(1.f, 0.f), w1, w2, w3, w4, w5, w6, w7};
#pragma unroll
    for (int m = 1; m < 8; ++m) a[m] = INV ? fo_cmulc(a[m], w[m]) : fo_cmul(a[m], w[m]);
}

// first forward stage (block length n, radix r1) on a[k] = x[t + k T], T = n / 8, in place (positions unchanged)
template <class PL>
__device__ __forceinline__ void fo_first_fwd(float2 (&a)[8], int t, const float2* __restrict__ tw)
{
    const int T = PL::n >> 3;
    if (PL::lg_r1 == 3) {
        fo_r8(a);
        fo_twiddle8<false>(a, t, 0, tw);
    } else if (PL::lg_r1 == 2) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int q = t + i * T;
            fo_r4(a[i], a[i + 2], a[i + 4], a[i + 6]);
            a[i + 2] = fo_cmul(a[i + 2], __ldg(tw + q));
            a[i + 4] = fo_cmul(a[i + 4], __ldg(tw + 2 * q));
            a[i + 6] = fo_cmul(a[i + 6], __ldg(tw + 3 * q));
        }
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 d = fo_sub(a[i], a[i + 4]);
            a[i] = fo_add(a[i], a[i + 4]);
            a[i + 4] = fo_cmul(d, __ldg(tw + t + i * T));
        }
    }
}
// its conjugate transpose (last inverse stage)
template <class PL>
__device__ __forceinline__ void fo_first_inv(float2 (&a)[8], int t, const float2* __restrict__ tw)
{
    const int T = PL::n >> 3;
    if (PL::lg_r1 == 3) {
        fo_twiddle8<true>(a, t, 0, tw);
#pragma unroll
        for (int m = 0; m < 8; ++m) a[m] = fo_conj(a[m]);
        fo_r8(a);
#pragma unroll
        for (int m = 0; m < 8; ++m) a[m] = fo_conj(a[m]);
    } else if (PL::lg_r1 == 2) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int q = t + i * T;
            float2 y0 = fo_conj(a[i]), y1 = fo_conj(fo_cmulc(a[i + 2], __ldg(tw + q)));
            float2 y2 = fo_conj(fo_cmulc(a[i + 4], __ldg(tw + 2 * q))), y3 = fo_conj(fo_cmulc(a[i + 6], __ldg(tw + 3 * q)));
            fo_r4(y0, y1, y2, y3);
            a[i] = fo_conj(y0); a[i + 2] = fo_conj(y1); a[i + 4] = fo_conj(y2); a[i + 6] = fo_conj(y3);
        }
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 y1 = fo_cmulc(a[i + 4], __ldg(tw + t + i * T));
            const float2 y0 = a[i];
            a[i] = fo_add(y0, y1);
            a[i + 4] = fo_sub(y0, y1);
        }
    }
}

// Forward transform of one row held as a[k] = x[t + k T]; on return a[m] is the value at digit-reversed position 8 t + m.
// xr: this row's exchange buffer in shared memory (9 n / 8 elements); every thread of the CTA must call (barriers inside).
template <class PL>
__device__ __forceinline__ void fo_forward(float2 (&a)[8], int t, const float2* __restrict__ tw, float2* xr)
{
    fo_first_fwd<PL>(a, t, tw);
    int lg_L = PL::lg_n, lg_sub = PL::lg_n - 3, blk = 0, q = t;    // positions of a[k]: (blk << lg_L) + q + (k << lg_sub)
    int lg_Ln = PL::lg_n - PL::lg_r1;                               // block length of the next stage
#pragma unroll
    for (int s = 1; s < PL::nstage; ++s) {
        {
            float2* w = xr + fo_phys((blk << lg_L) + q);
            const int st = fo_stride(lg_sub);
#pragma unroll
            for (int k = 0; k < 8; ++k) w[k * st] = a[k];
        }
        __syncthreads();
        lg_L = lg_Ln; lg_sub = lg_L - 3;
        blk = t >> lg_sub; q = t & ((1 << lg_sub) - 1);
        {
            const float2* rd = xr + fo_phys((blk << lg_L) + q);
            const int st = fo_stride(lg_sub);
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = rd[k * st];
        }
        __syncthreads();
        fo_r8(a);
        if (lg_sub > 0) fo_twiddle8<false>(a, q, PL::lg_n - lg_L, tw);
        lg_Ln = lg_sub;
    }
}
// Inverse (unnormalised): a[m] at digit-reversed position 8 t + m on entry, a[k] = x[t + k T] on return.
template <class PL>
__device__ __forceinline__ void fo_inverse(float2 (&a)[8], int t, const float2* __restrict__ tw, float2* xr)
{
    int lg_L = 3, lg_sub = 0;
#pragma unroll
    for (int s = PL::nstage - 1; s >= 1; --s) {
        const int blk = t >> lg_sub, q = t & ((1 << lg_sub) - 1);
        if (lg_sub > 0) fo_twiddle8<true>(a, q, PL::lg_n - lg_L, tw);
#pragma unroll
        for (int m = 0; m < 8; ++m) a[m] = fo_conj(a[m]);
        fo_r8(a);
#pragma unroll
        for (int m = 0; m < 8; ++m) a[m] = fo_conj(a[m]);
        {
            float2* w = xr + fo_phys((blk << lg_L) + q);
            const int st = fo_stride(lg_sub);
#pragma unroll
            for (int k = 0; k < 8; ++k) w[k * st] = a[k];
        }
        __syncthreads();
        // the stage before: block length 8 L (the first stage: n, whatever its radix; its threads hold x[t + k n / 8])
        int lg_Lp, lg_subp;
        if (s == 1) { lg_Lp = PL::lg_n; lg_subp = PL::lg_n - 3; }
        else { lg_Lp = lg_L + 3; lg_subp = lg_L; }
        const int blkp = t >> lg_subp, qp = t & ((1 << lg_subp) - 1);
        {
            const float2* rd = xr + fo_phys((blkp << lg_Lp) + qp);
            const int st = fo_stride(lg_subp);
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = rd[k * st];
        }
        __syncthreads();
        lg_L = lg_Lp; lg_sub = lg_subp;
    }
    fo_first_inv<PL>(a, t, tw);
}

struct FoArgs {
    const float2* tw_w;            // exp(-2 pi i k / W)
    const float2* tw_h;            // exp(-2 pi i k / H)
    int H, W;
    int nc, m_lo;                  // kept columns: signed frequency m_x = m_lo + c, c = 0 .. nc-1
    float2* spec_t;                // [B][nc][H] kept columns, transposed
};

__device__ __forceinline__ int fo_kx(const FoArgs& a, int c)
{
    const int m = a.m_lo + c;
    return m < 0 ? m + a.W : m;
}

struct FoShear {                   // DIC prologue of K1 (Eq. 5): D = |U(r + ds) e^{i theta} - U(r - ds) e^{-i theta}|^2
    int sx, sy;
    float2 e;                      // (cos theta, sin theta)
};

// K1: forward row transforms, kFoThreads / (W / 8) rows per CTA; the kept columns are written transposed.
// SHEAR: the row that is transformed is the DIC interference image D of the field (real), formed on the fly.
template <class PL, bool SHEAR>
__global__ void __launch_bounds__(kFoThreads) k_fo_rows_fwd(const FoArgs a, const float2* __restrict__ field, const FoShear sh)
{
    extern __shared__ __align__(16) float2 fo_x[];
    constexpr int lgT = PL::lg_n - 3, T = 1 << lgT, lgR = 9 - lgT, R = 1 << lgR, stride = PL::n + (PL::n >> 3);
    const int r = threadIdx.x >> lgT, t = threadIdx.x & (T - 1), b = blockIdx.y, row0 = blockIdx.x << lgR;
    float2* xr = fo_x + r * stride;
    float2 v[8];
    if (!SHEAR) {
        const float2* src = field + ((size_t)b * a.H + row0 + r) * a.W + t;
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = src[k << lgT];
    } else {
        const int i = row0 + r;
        int ip = i + sh.sy, im = i - sh.sy;                          // |sy| < H, |sx| < W: one wrap each (readings A21, A22)
        ip += ip < 0 ? a.H : (ip >= a.H ? -a.H : 0);
        im += im < 0 ? a.H : (im >= a.H ? -a.H : 0);
        const float2* fp = field + ((size_t)b * a.H + ip) * a.W;
        const float2* fm = field + ((size_t)b * a.H + im) * a.W;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int j = t + (k << lgT);
            int jp = j + sh.sx, jm = j - sh.sx;
            jp += jp < 0 ? a.W : (jp >= a.W ? -a.W : 0);
            jm += jm < 0 ? a.W : (jm >= a.W ? -a.W : 0);
            const float2 up = fp[jp], um = fm[jm];
            const float dr = (up.x * sh.e.x - up.y * sh.e.y) - (um.x * sh.e.x + um.y * sh.e.y);
            const float di = (up.x * sh.e.y + up.y * sh.e.x) - (um.y * sh.e.x - um.x * sh.e.y);
            v[k] = make_float2(dr * dr + di * di, 0.0f);
        }
    }
    fo_forward<PL>(v, t, a.tw_w, xr);
#pragma unroll
    for (int m = 0; m < 8; ++m) xr[(m << lgT) + t] = v[m];          // position 8 t + m, stored transposed (conflict free)
    __syncthreads();
    for (int idx = threadIdx.x; idx < (a.nc << lgR); idx += kFoThreads) {
        const int rr = idx & (R - 1), c = idx >> lgR;
        const int p = fo_pos_of_freq<PL>(fo_kx(a, c));
        a.spec_t[((size_t)b * a.nc + c) * a.H + row0 + rr] = fo_x[rr * stride + ((p & 7) << lgT) + (p >> 3)];
    }
}

// K2: kept columns: forward transform along y, multiplication, inverse transform along y, in place.
// MUL = 0 / 1: the pupil function (without / with the defocus phase) times scale = 1 / (H W); MUL = 2: scale times the
// transfer-function array tf[B][H][W] (natural FFT order; the DIC stage's OTF)
template <class PL, int MUL>
__global__ void __launch_bounds__(kFoThreads) k_fo_cols(const FoArgs a, const FrameOptics* __restrict__ optics, double inv_wp,
                                                        double inv_hp, float scale, float imag_sign, const float2* __restrict__ tf)
{
    extern __shared__ __align__(16) float2 fo_x[];
    constexpr int lgT = PL::lg_n - 3, T = 1 << lgT, lgR = 9 - lgT, stride = PL::n + (PL::n >> 3);
    const int r = threadIdx.x >> lgT, t = threadIdx.x & (T - 1), b = blockIdx.y, c = (blockIdx.x << lgR) + r;
    const bool valid = c < a.nc;
    float2* xr = fo_x + r * stride;
    float2* col = a.spec_t + ((size_t)b * a.nc + (valid ? c : 0)) * a.H + t;
    float2 v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = valid ? col[k << lgT] : make_float2(0.f, 0.f);
    fo_forward<PL>(v, t, a.tw_h, xr);
    const int kx = fo_kx(a, valid ? c : 0);
    const FrameOptics fo = optics[b];
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        const int ky = fo_freq_of_pos<PL>(8 * t + m);
        if (MUL == 2) {
            const float2 w = __ldg(tf + ((size_t)b * a.H + ky) * a.W + kx);
            v[m] = fo_cmul(v[m], make_float2(w.x * scale, w.y * scale));
        } else {
            float2 pv = pupil_value<MUL == 1>(fo, kx, ky, a.H, a.W, inv_wp, inv_hp, scale);
            if (MUL == 1) pv.y *= imag_sign;                         // -1: conj(P), the adjoint of the stage
            v[m] = MUL == 1 ? fo_cmul(v[m], pv) : make_float2(v[m].x * pv.x, v[m].y * pv.x);
        }
    }
    fo_inverse<PL>(v, t, a.tw_h, xr);
    if (valid) {
#pragma unroll
        for (int k = 0; k < 8; ++k) col[k << lgT] = v[k];
    }
}

// what K3 does with the image V it has transformed back
enum { kFoSensor = 0, kFoSensorShot = 1, kFoTimesReal = 2, kFoGopd = 3, kFoRealSensor = 4, kFoRealSensorShot = 5 };
struct FoEpi {
    float* out;                    // sensor: intensity [B, H, W]; kFoGopd: dL/dOPD [B, H, W]
    float2* cout;                  // kFoTimesReal: g_V = g V [B, H, W] complex
    const float* g;                // kFoTimesReal: the real factor (dL/dI)
    const float2* u;               // kFoGopd: the exit wave U
    const FrameOptics* optics;     // kFoGopd: 1 / lambda per frame
    float sigma;
    double photons;
    uint64_t seed;
};

// K3: inverse row transforms from the kept columns (all other bins are zero), then the sensor (I = |V|^2, shot and read noise),
// or, for the adjoint of the stage (osog_backward_intensity), g_V = (dL/dI) V  resp.  dL/dOPD = (4 pi / lambda) Im(g_U conj U)
template <class PL, int MODE>
__global__ void __launch_bounds__(kFoThreads) k_fo_rows_inv(const FoArgs a, const FoEpi ep)
{
    extern __shared__ __align__(16) float2 fo_x[];
    constexpr int lgT = PL::lg_n - 3, T = 1 << lgT, lgR = 9 - lgT, R = 1 << lgR, stride = PL::n + (PL::n >> 3);
    const int r = threadIdx.x >> lgT, t = threadIdx.x & (T - 1), b = blockIdx.y, row0 = blockIdx.x << lgR;
    float2* xr = fo_x + r * stride;
    for (int k = threadIdx.x; k < R * stride; k += kFoThreads) fo_x[k] = make_float2(0.f, 0.f);
    __syncthreads();
    for (int idx = threadIdx.x; idx < (a.nc << lgR); idx += kFoThreads) {
        const int rr = idx & (R - 1), c = idx >> lgR;
        const int p = fo_pos_of_freq<PL>(fo_kx(a, c));
        fo_x[rr * stride + ((p & 7) << lgT) + (p >> 3)] = a.spec_t[((size_t)b * a.nc + c) * a.H + row0 + rr];
    }
    __syncthreads();
    float2 v[8];
#pragma unroll
    for (int m = 0; m < 8; ++m) v[m] = xr[(m << lgT) + t];
    __syncthreads();
    fo_inverse<PL>(v, t, a.tw_w, xr);
    const size_t pix0 = (size_t)(row0 + r) * a.W + t;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const size_t pix = pix0 + (k << lgT), gpix = (size_t)b * a.H * a.W + pix;
        if (MODE == kFoTimesReal) {
            const float gv = ep.g[gpix];
            ep.cout[gpix] = make_float2(v[k].x * gv, v[k].y * gv);
        } else if (MODE == kFoGopd) {
            const float2 w = ep.u[gpix];
            const float kk = (float)(12.566370614359172 * ep.optics[b].inv_lambda);
            ep.out[gpix] = kk * (v[k].y * w.x - v[k].x * w.y);
        } else {
            float I = (MODE == kFoRealSensor || MODE == kFoRealSensorShot) ? v[k].x : v[k].x * v[k].x + v[k].y * v[k].y;
            if (MODE == kFoSensorShot || MODE == kFoRealSensorShot)
                I = (float)(poisson_draw(ep.photons * fmax((double)I, 0.0), ep.seed, (uint32_t)b, (uint32_t)pix) / ep.photons);
            if (ep.sigma != 0.0f) I = fmaf(ep.sigma, read_noise_z(ep.seed, (uint32_t)b, (uint32_t)pix), I);
            ep.out[gpix] = I;
        }
    }
}

__global__ void k_fo_twiddles(float2* tw, int n)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    double s, c;
    sincospi(-2.0 * (double)k / (double)n, &s, &c);
    tw[k] = make_float2((float)c, (float)s);
}

cudaError_t launch_fo_twiddles(osog_ctx* c, float2* tw, int n)
{
    k_fo_twiddles<<<(n + 255) / 256, 256, 0, c->stream>>>(tw, n);
    return cudaGetLastError();
}

bool fused_optics_applies(const osog_ctx* c)
{
    auto pow2 = [](int v) { return v >= 64 && v <= 4096 && (v & (v - 1)) == 0; };
    return pow2(c->H) && pow2(c->W);
}

// in: [B, H, W] complex frames (read only); spec_t: scratch of B * W * H complex values; tw_w / tw_h: twiddle tables of W / H
// tf == nullptr: multiply by the pupil function; else by the transfer-function array tf (support: twice the pupil's radius);
// sh != nullptr: K1 transforms the DIC interference image of `in`
static cudaError_t fo_run(osog_ctx* c, const osog_optics* o, const float2* in, float2* spec_t, const float2* tw_w, const float2* tw_h,
                          int mode, float imag_sign, const FoEpi& ep, const float2* tf = nullptr, const FoShear* sh = nullptr)
{
    const int B = o->B, H = c->H, W = c->W;
    FoArgs a;
    a.tw_w = tw_w; a.tw_h = tw_h; a.H = H; a.W = W;
    a.spec_t = spec_t;
    // widest pupil of the batch in x: m_x^2 H^2 <= floor((NA p / lambda)^2 H^2 W^2)  =>  |m_x| <= NA p W / lambda
    long long rx = 0;
    for (int b = 0; b < B; ++b) {
        long long rb = W;                                         // all-pass
        if (o->pupil_enabled && o->NA != nullptr) {
            const double r = o->NA[b] * o->pitch_um / o->lambda_um[b] * (double)W;
            if (r < (double)W) rb = (long long)floor(tf ? 2.0 * r : r) + (tf ? 2 : 1);    // (the autocorrelation of the pupil)
        }
        rx = rb > rx ? rb : rx;
    }
    const int m_hi = (int)(rx < W / 2 - 1 ? rx : W / 2 - 1);
    a.m_lo = -(int)(rx < W / 2 ? rx : W / 2);
    a.nc = m_hi - a.m_lo + 1;
    const bool defocus = o->defocus_um != 0.0;
    const double inv_wp = 1.0 / ((double)W * o->pitch_um), inv_hp = 1.0 / ((double)H * o->pitch_um);
    const float scale = (float)(1.0 / ((double)H * W));
    const int Rw = kFoThreads / (W / 8), Rh = kFoThreads / (H / 8);           // rows / columns per CTA
    const size_t smem_rows = (size_t)Rw * (W + W / 8) * sizeof(float2), smem_cols = (size_t)Rh * (H + H / 8) * sizeof(float2);
    const dim3 gcol((a.nc + Rh - 1) / Rh, B), grow(H / Rw, B);
    int lg_w = 0, lg_h = 0;
    while ((1 << lg_w) < W) ++lg_w;
    while ((1 << lg_h) < H) ++lg_h;
    const FoShear shv = sh ? *sh : FoShear{0, 0, make_float2(1.f, 0.f)};
    cudaStream_t st = c->stream;
// one instantiation per transform length 64 .. 4096
#define FO_BY_LENGTH(lg, CALL) \
    switch (lg) { \
        case 6: { using PL = FoPlan<6>; CALL; } break;   case 7: { using PL = FoPlan<7>; CALL; } break; \
        case 8: { using PL = FoPlan<8>; CALL; } break;   case 9: { using PL = FoPlan<9>; CALL; } break; \
        case 10: { using PL = FoPlan<10>; CALL; } break; case 11: { using PL = FoPlan<11>; CALL; } break; \
        case 12: { using PL = FoPlan<12>; CALL; } break; default: return cudaErrorInvalidValue; \
    }
    if (sh) { FO_BY_LENGTH(lg_w, (k_fo_rows_fwd<PL, true><<<grow, kFoThreads, smem_rows, st>>>(a, in, shv))) }
    else { FO_BY_LENGTH(lg_w, (k_fo_rows_fwd<PL, false><<<grow, kFoThreads, smem_rows, st>>>(a, in, shv))) }
    cudaError_t e;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (tf) { FO_BY_LENGTH(lg_h, (k_fo_cols<PL, 2><<<gcol, kFoThreads, smem_cols, st>>>(a, c->optics, inv_wp, inv_hp, scale, imag_sign, tf))) }
    else if (defocus) { FO_BY_LENGTH(lg_h, (k_fo_cols<PL, 1><<<gcol, kFoThreads, smem_cols, st>>>(a, c->optics, inv_wp, inv_hp, scale, imag_sign, tf))) }
    else { FO_BY_LENGTH(lg_h, (k_fo_cols<PL, 0><<<gcol, kFoThreads, smem_cols, st>>>(a, c->optics, inv_wp, inv_hp, scale, imag_sign, tf))) }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    switch (mode) {
        case kFoSensorShot: FO_BY_LENGTH(lg_w, (k_fo_rows_inv<PL, kFoSensorShot><<<grow, kFoThreads, smem_rows, st>>>(a, ep))) break;
        case kFoTimesReal: FO_BY_LENGTH(lg_w, (k_fo_rows_inv<PL, kFoTimesReal><<<grow, kFoThreads, smem_rows, st>>>(a, ep))) break;
        case kFoGopd: FO_BY_LENGTH(lg_w, (k_fo_rows_inv<PL, kFoGopd><<<grow, kFoThreads, smem_rows, st>>>(a, ep))) break;
        case kFoRealSensor: FO_BY_LENGTH(lg_w, (k_fo_rows_inv<PL, kFoRealSensor><<<grow, kFoThreads, smem_rows, st>>>(a, ep))) break;
        case kFoRealSensorShot: FO_BY_LENGTH(lg_w, (k_fo_rows_inv<PL, kFoRealSensorShot><<<grow, kFoThreads, smem_rows, st>>>(a, ep))) break;
        default: FO_BY_LENGTH(lg_w, (k_fo_rows_inv<PL, kFoSensor><<<grow, kFoThreads, smem_rows, st>>>(a, ep))) break;
    }
#undef FO_BY_LENGTH
    return cudaGetLastError();
}

// L1-L3: intensity (with the sensor's noise) of the exit wave `field`
cudaError_t launch_fused_optics(osog_ctx* c, const osog_optics* o, const float2* field, float2* spec_t, const float2* tw_w,
                                const float2* tw_h, float* d_intensity)
{
    FoEpi ep = {};
    ep.out = d_intensity;
    ep.sigma = (float)o->read_noise_sigma; ep.photons = o->shot_noise_photons; ep.seed = o->seed;
    return fo_run(c, o, field, spec_t, tw_w, tw_h, o->shot_noise_photons != 0.0 ? kFoSensorShot : kFoSensor, 1.0f, ep);
}

// DIC stage (Eq. 5) with a ready transfer function: I = Re F^-1{ F{D} OTF / (H W) }, D the interference image of `field`
cudaError_t launch_fused_dic(osog_ctx* c, const osog_optics* o, const float2* field, const float2* otf, float2* spec_t,
                             const float2* tw_w, const float2* tw_h, int sx, int sy, double bias_rad, float* d_dic)
{
    FoEpi ep = {};
    ep.out = d_dic;
    ep.sigma = (float)o->read_noise_sigma; ep.photons = o->shot_noise_photons; ep.seed = o->seed;
    FoShear sh;
    sh.sx = sx; sh.sy = sy;
    sh.e = make_float2((float)cos(bias_rad), (float)sin(bias_rad));
    return fo_run(c, o, field, spec_t, tw_w, tw_h, o->shot_noise_photons != 0.0 ? kFoRealSensorShot : kFoRealSensor, 1.0f, ep, otf, &sh);
}

// Adjoint of L1-L3 (osog_backward_intensity): V = U * h_obj, g_V = (dL/dI) V into `work`; g_U = F^-1{conj(P) F{g_V}},
// dL/dOPD = (4 pi / lambda) Im(g_U conj U) into d_gopd.  Two passes of the same three kernels; `field` (U) is only read.
cudaError_t launch_fused_optics_adjoint(osog_ctx* c, const osog_optics* o, const float2* field, float2* work, float2* spec_t,
                                        const float2* tw_w, const float2* tw_h, const float* d_gI, float* d_gopd)
{
    FoEpi ep = {};
    ep.cout = work; ep.g = d_gI;
    cudaError_t e = fo_run(c, o, field, spec_t, tw_w, tw_h, kFoTimesReal, 1.0f, ep);
    if (e != cudaSuccess) return e;
    FoEpi eq = {};
    eq.out = d_gopd; eq.u = field; eq.optics = c->optics;
    return fo_run(c, o, work, spec_t, tw_w, tw_h, kFoGopd, -1.0f, eq);
}

}  // namespace osog
