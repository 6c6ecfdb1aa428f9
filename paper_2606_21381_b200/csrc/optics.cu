// Library stage around cuFFT (timed separately from the hot path, L1-L3):
// pupil function circ(|k| / (NA / lambda)) exp(i dz k_z) with the 1/(HW) normalisation (Eq. 3),
// the DIC shear-and-interfere step and the element-wise helpers of its incoherent convolution (Eq. 5),
// and the sensor: I = |.|^2 plus optional Gaussian read noise from Philox4x32-10.
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

}  // namespace osog
