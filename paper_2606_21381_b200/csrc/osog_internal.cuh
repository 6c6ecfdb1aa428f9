// Internal declarations shared by the CUDA translation units of libosog (NOT part of the C ABI).
// Nothing here is shared with oracle/ ("independence").
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>
#include <utility>
#include <vector>
#include "../../include/osog.h"

namespace osog {

// ---- build-time constants -----------------------------------------------------------------------------------
constexpr int kTile = 32;              // binning tile edge T (pixels); one CTA composes one tile
constexpr int kComposeThreads = 256;   // 8 warps; each warp owns a 16 x 8 pixel sub-tile, each lane 4 x 1 pixels
constexpr int kRecWords = 64;          // 256-byte record per particle: 16 header words + up to 24 doubles
constexpr int kPairWords = 48;         // prisms: 6 slabs x (U, V, Cx, Cn) as (hi, lo) float pairs for the composition kernel
constexpr double kBBoxPadPx = 1.0 / 1024.0;   // delta of DESIGN.md B2
constexpr float kSteepSlope = 16.0f;   // slabs steeper than this (|n_xy| / |n_z|) are refined in fp64 where active
constexpr double kAllF64Slope = 1.0e4; // a slab steeper than this (or vertical) sends the whole particle to fp64

// record header flags (word 8)
constexpr uint32_t kFlagPrism = 1u;
constexpr uint32_t kFlagAllF64 = 16u;
// bits 8..10: number of steep slabs (they come first); bits 16..21: per-slab "vertical" (n_z == 0) mask

// status of one render call (device): status bits, longest tile list, total number of (particle, tile) pairs
struct DeviceStatus {
    uint32_t bits;
    uint32_t max_count;
    unsigned long long pairs;
};

struct FrameOptics {          // per frame, device
    double inv_lambda;        // 1 / lambda  (turns per um of OPD)
    double fx0_pitch;         // sin(tilt_x) / lambda * p : turns per pixel along x
    double fy0_pitch;
    long long pupil_thresh;   // floor((NA p / lambda)^2 H^2 W^2), or -1 = all-pass
    long long prop_thresh;    // floor((n_m p / lambda)^2 H^2 W^2): propagating bins (defocus only), or -1 = all
    double nm_over_lambda_sq; // (n_medium / lambda)^2, cycles^2 / um^2
    double defocus_um;        // delta z of Eq. 3; 0 = none
    double pad_;
};

constexpr int kOpticsChunk = 16;
struct OpticsChunk {          // passed by value to k_set_optics
    int first, count;
    FrameOptics f[kOpticsChunk];
};

}  // namespace osog

struct osog_ctx {
    int device;
    cudaStream_t stream;
    int H, W, max_frames;
    long long max_particles, max_pairs;
    int ntx, nty;                   // tiles per row / column
    long long max_tiles;            // max_frames * ntx * nty
    long long count_stride;         // max_tiles rounded up to a multiple of 4 (128-bit loads of the scan)
    int slice_cap;                  // entries of one tile's staging slice (longer lists take the ordered re-scan of k_sort_cull)
    int last_cuda_error;
    // last call
    int last_B;
    int last_has_ramp;
    long long last_N;
    long long last_tiles;
    double last_topo;               // micro-topography amplitude and seed of the last render call (reading A29)
    unsigned long long last_seed;
    const int32_t* last_frame_start; // device pointer of the last call's frame_start (nullptr: one frame)
    // scratch (device)
    float* rec;                     // [max_particles][kRecWords]
    float* rec2;                    // [max_particles][kPairWords] prism slab coefficients as exact-grid (hi, lo) float pairs
    int4* tbox;                     // [max_particles] tile range tx0, tx1, ty0, ty1 (tx0 > tx1: not listed)
    int* pframe;                    // [max_particles] frame of the particle
    uint32_t* count;                // [2][count_stride] per-tile list length; slot status_idx belongs to the current call, the
                                    // other slot is zeroed by that call's k_sort_cull for the next call
    uint32_t* offset;               // [max_tiles + 1] exclusive scan of the current call's counts (H3, k_prepare's last binning block)
    uint32_t* done;                 // [1] finished binning blocks of the running k_prepare (0 between calls)
    uint32_t* slices;               // [max_tiles][slice_cap] staging: tile t's unsorted entries at slices + t * slice_cap
    uint32_t* list;                 // [max_pairs] CSR list: tile t's particle indices, ascending, at list + offset[t]
    uint16_t* meta;                 // [max_pairs] per list entry: sub-tile mask | evaluation code << 8 (k_sort_cull)
    osog::FrameOptics* optics;      // [max_frames]
    osog::DeviceStatus* status;     // [2]: slot of the current call / slot being reset for the next call
    int status_idx;                 // slot used by the last render call
    long long slot_tiles[2];        // tiles whose counters a slot's last user may have left non-zero
    bool scratch_dirty;             // a call failed midway: count / status must be cleared explicitly
    float2* field;                  // [max_frames][H][W] (intensity path)
    float2* work;                   // [max_frames][H][W] second complex batch (DIC path; allocated by the first DIC call)
    double* spec_partial;           // [max_frames][ceil(H W / 256)] block sums of the spectral loss (allocated by its first call)
    float* bf_h;                    // [max_frames][H][W] height map of the brightfield path (allocated by its first call)
    float2* spec_t;                 // [max_frames][W][H] kept columns of the fused optics stage (allocated by its first call)
    float2* tw_w;                   // [W] exp(-2 pi i k / W), and [H] (the same table if H == W): fused optics stage
    float2* tw_h;
    bool fo_ready;
    float2* otf;                    // [max_frames][H][W] optical transfer function F{|F^-1{P}|^2} of the last DIC call
    std::vector<double>* otf_key;   // optics the cached OTF was built for (B, pitch, n_medium, defocus, pupil, lambda[], NA[])
    osog::DeviceStatus* h_status;   // pinned host mirror
    std::vector<std::pair<unsigned char*, size_t>>* guards;   // (start of the guard band, bytes) behind every scratch array
    cufftHandle plan_one, plan_batch;
    bool has_plan_one, has_plan_batch;
};

namespace osog {

// ---- programmatic dependent launch (sm_90+): a kernel launched with launch_pdl may start while its predecessor in the
// stream is still running; it must call pdl_wait() before it touches anything the predecessor reads or writes.  A kernel
// calls pdl_trigger() once it no longer minds its successor's CTAs becoming resident (they then block in pdl_wait()).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <class... KArgs, class... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ---- counter-based random numbers (Philox4x32-10), shared by the sensor stage and the micro-topography of the write-out ----
__device__ __forceinline__ void philox_round(uint32_t (&c)[4], uint32_t k0, uint32_t k1)
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t hi0 = __umulhi(M0, c[0]), lo0 = M0 * c[0];
    const uint32_t hi1 = __umulhi(M1, c[2]), lo1 = M1 * c[2];
    const uint32_t n0 = hi1 ^ c[1] ^ k0, n2 = hi0 ^ c[3] ^ k1;
    c[0] = n0; c[1] = lo1; c[2] = n2; c[3] = lo0;
}

// Standard normal for (seed, frame, pixel) of stream `stream`: key = (seed low, seed high), counter = (pixel, frame, stream, 0);
// u1 = (r0 + 1) 2^-32, u2 = r1 2^-32, z = sqrt(-2 ln u1) cos(2 pi u2)   (readings A13: stream 0 = read noise; A29: stream 2 =
// micro-topography; stream 1 is the shot noise's)
__device__ __forceinline__ float philox_normal(uint64_t seed, uint32_t frame, uint32_t pixel, uint32_t stream)
{
    uint32_t c[4] = {pixel, frame, stream, 0u};
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

// binning.cu
cudaError_t upload_optics(osog_ctx* c, const osog_optics* o, OpticsChunk* first);
cudaError_t launch_binning(osog_ctx* c, const osog_particles* p, long long N, const osog_optics* o, float* d_obb = nullptr,
                           bool unit_dn = false);
// compose.cu
cudaError_t launch_compose(osog_ctx* c, int B, bool has_ramp, float* d_opd, float2* d_field, bool sort_first = true);   // uses c->last_topo / c->last_seed
cudaError_t launch_compose_atomic(osog_ctx* c, long long N, int B, float* d_opd);
cudaError_t launch_compose_smem_atomic(osog_ctx* c, int B, float* d_opd);
cudaError_t launch_backward_np(osog_ctx* c, long long N, const float* d_gopd, float* d_gnp);
cudaError_t launch_backward_centre(osog_ctx* c, long long N, double pitch, const float* d_gopd, float* d_gc);
cudaError_t launch_backward_params(osog_ctx* c, const osog_particles* p, long long N, double pitch, double n_medium,
                                   const float* d_gopd, float* d_gpar, float* d_gnp = nullptr, float* d_gc = nullptr);
cudaError_t launch_gbuffer(osog_ctx* c, int B, const int32_t* d_frame_start, double pitch, int32_t* d_top_id, float* d_depth,
                           float* d_normal);
// optics.cu
cudaError_t launch_pupil(osog_ctx* c, int B, float2* spec, double pitch, bool defocus);
cudaError_t launch_pupil_fill(osog_ctx* c, int B, float2* spec, double pitch, bool defocus);
cudaError_t launch_pupil_conj(osog_ctx* c, int B, float2* spec, double pitch, bool defocus);
cudaError_t launch_mul_real(osog_ctx* c, int B, float2* v, const float* g);
cudaError_t launch_gopd(osog_ctx* c, int B, const float2* gu, const float2* u, float* d_gopd);
cudaError_t launch_dic_shear(osog_ctx* c, int B, const float2* field, float2* out, int sx, int sy, double theta);
cudaError_t launch_abs2(osog_ctx* c, int B, float2* buf, double scale);
cudaError_t launch_cmul(osog_ctx* c, int B, float2* a, const float2* b, double scale);
cudaError_t launch_brightfield(osog_ctx* c, int B, float2* field, const float* d_h, double pitch, double n1, double n2,
                               double dmu, double gain);
cudaError_t launch_real_to_complex(osog_ctx* c, int B, const float* a, const float* b, float2* ca, float2* cb);
cudaError_t launch_spectral_terms(osog_ctx* c, int B, float2* F, const float2* T, double eps, double* partial, double* d_loss, bool want_grad);
cudaError_t launch_real_part(osog_ctx* c, int B, const float2* in, float* out);
cudaError_t launch_height_stencil(osog_ctx* c, int B, const float* d_h, double pitch, float* d_grad, float* d_lap);
cudaError_t launch_sensor_real(osog_ctx* c, int B, const float2* img, float* d_out, double sigma, double photons, uint64_t seed);
cudaError_t launch_sensor(osog_ctx* c, int B, const float2* img, float* d_intensity, double sigma, double photons, uint64_t seed);
bool fused_optics_applies(const osog_ctx* c);       // power-of-two frames, 64 .. 4096
cudaError_t launch_fo_twiddles(osog_ctx* c, float2* tw, int n);
cudaError_t launch_fused_optics(osog_ctx* c, const osog_optics* o, const float2* field, float2* spec_t, const float2* tw_w,
                                const float2* tw_h, float* d_intensity);
cudaError_t launch_fused_dic(osog_ctx* c, const osog_optics* o, const float2* field, const float2* otf, float2* spec_t,
                             const float2* tw_w, const float2* tw_h, int sx, int sy, double bias_rad, float* d_dic);
cudaError_t launch_fused_optics_adjoint(osog_ctx* c, const osog_optics* o, const float2* field, float2* work, float2* spec_t,
                                        const float2* tw_w, const float2* tw_h, const float* d_gI, float* d_gopd);
cudaError_t launch_poisson(osog_ctx* c, const float* d_lam, size_t n, uint64_t seed, uint32_t frame, int32_t* d_counts);

}  // namespace osog
