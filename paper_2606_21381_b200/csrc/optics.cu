// Library stage around cuFFT (timed separately from the hot path, L1-L3):
// pupil mask circ(|k| / (NA / lambda)) with the 1/(HW) normalisation (Eq. 3 with delta z = 0),
// and the sensor: I = |.|^2 plus optional Gaussian read noise from Philox4x32-10.
#include "osog_internal.cuh"

namespace osog {

// Bin (ky, kx) of the unshifted FFT grid has signed index m = k for k <= (n-1)/2, else k - n.
// It passes iff m_x^2 H^2 + m_y^2 W^2 <= floor((NA p / lambda)^2 H^2 W^2)  (64-bit integers, reading A10).
__global__ void __launch_bounds__(256) k_pupil(float2* __restrict__ spec, const FrameOptics* __restrict__ optics,
                                               int H, int W, float scale)
{
    const int kx = blockIdx.x * blockDim.x + threadIdx.x;
    const int ky = blockIdx.y, b = blockIdx.z;
    if (kx >= W) return;
    const long long thr = optics[b].pupil_thresh;
    const long long mx = kx <= (W - 1) / 2 ? kx : kx - W;
    const long long my = ky <= (H - 1) / 2 ? ky : ky - H;
    const long long lhs = mx * mx * ((long long)H * H) + my * my * ((long long)W * W);
    const size_t idx = ((size_t)b * H + ky) * W + kx;
    float2 v = spec[idx];
    const float s = (thr < 0 || lhs <= thr) ? scale : 0.0f;
    v.x *= s;
    v.y *= s;
    spec[idx] = v;
}

__device__ __forceinline__ void philox_round(uint32_t (&c)[4], uint32_t k0, uint32_t k1)
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t hi0 = __umulhi(M0, c[0]), lo0 = M0 * c[0];
    const uint32_t hi1 = __umulhi(M1, c[2]), lo1 = M1 * c[2];
    const uint32_t n0 = hi1 ^ c[1] ^ k0, n2 = hi0 ^ c[3] ^ k1;
    c[0] = n0; c[1] = lo1; c[2] = n2; c[3] = lo0;
}

// Standard normal for (seed, frame, pixel): Philox4x32-10, key = (seed low, seed high), counter = (pixel, frame, 0, 0);
// u1 = (r0 + 1) 2^-32, u2 = r1 2^-32, z = sqrt(-2 ln u1) cos(2 pi u2)   (reading A13)
__device__ __forceinline__ float read_noise_z(uint64_t seed, uint32_t frame, uint32_t pixel)
{
    uint32_t c[4] = {pixel, frame, 0u, 0u};
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        philox_round(c, k0, k1);
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    const double u1 = ((double)c[0] + 1.0) * 2.3283064365386963e-10;
    const float l = -2.0f * (float)log(u1);
    const float u2 = (float)c[1] * 2.3283064365386963e-10f;
    return sqrtf(l) * cospif(2.0f * u2);
}

__global__ void __launch_bounds__(256) k_sensor(const float2* __restrict__ img, float* __restrict__ out, int H, int W,
                                                float sigma, uint64_t seed)
{
    const size_t npx = (size_t)H * W;
    const size_t pix = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int b = blockIdx.y;
    if (pix >= npx) return;
    const float2 v = img[(size_t)b * npx + pix];
    float I = v.x * v.x + v.y * v.y;
    if (sigma != 0.0f) I = fmaf(sigma, read_noise_z(seed, (uint32_t)b, (uint32_t)pix), I);
    out[(size_t)b * npx + pix] = I;
}

cudaError_t launch_pupil(osog_ctx* c, int B, float2* spec)
{
    const dim3 grid((c->W + 255) / 256, c->H, B);
    k_pupil<<<grid, 256, 0, c->stream>>>(spec, c->optics, c->H, c->W, (float)(1.0 / ((double)c->H * c->W)));
    return cudaGetLastError();
}

cudaError_t launch_sensor(osog_ctx* c, int B, const float2* img, float* d_intensity, double sigma, uint64_t seed)
{
    const size_t npx = (size_t)c->H * c->W;
    const dim3 grid((unsigned)((npx + 255) / 256), B);
    k_sensor<<<grid, 256, 0, c->stream>>>(img, d_intensity, c->H, c->W, (float)sigma, seed);
    return cudaGetLastError();
}

}  // namespace osog
