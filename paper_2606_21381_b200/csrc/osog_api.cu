// C ABI of libosog (include/osog.h): context management, argument checks, launch sequencing.
#include <mutex>
#include <new>
#include <cstring>
#include <vector>
#include "osog_internal.cuh"

using namespace osog;

namespace {

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int cuda_fail(osog_ctx* c, cudaError_t e)
{
    if (c) c->last_cuda_error = (int)e;
    return OSOG_ECUDA;
}

constexpr size_t kGuardBytes = 256;             // guard band behind every scratch array (osog_debug_check_guards)
constexpr unsigned char kGuardByte = 0xA5;

// scratch array of n elements followed by a guard band that no kernel may touch
template <class T>
cudaError_t dalloc(T** p, size_t n, osog_ctx* c = nullptr)
{
    *p = nullptr;
    const size_t bytes = sizeof(T) * (n ? n : 1);
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(p), bytes + kGuardBytes);
    if (e != cudaSuccess) return e;
    unsigned char* g = reinterpret_cast<unsigned char*>(*p) + bytes;
    if ((e = cudaMemset(g, kGuardByte, kGuardBytes)) != cudaSuccess) return e;
    if (c && c->guards) c->guards->emplace_back(g, kGuardBytes);
    return cudaSuccess;
}

int check_call(const osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, const void* out)
{
    if (!c || !p || !o || !out) return OSOG_EINVAL;
    if (p->struct_size != sizeof(osog_particles) || o->struct_size != sizeof(osog_optics)) return OSOG_EINVAL;
    if (N < 0 || N > c->max_particles) return OSOG_EINVAL;
    if (o->B < 1 || o->B > c->max_frames) return OSOG_EINVAL;
    if (!aligned16(out)) return OSOG_EINVAL;
    if (!(o->pitch_um > 0.0) || !(o->pitch_um < 1.0e300) || !(fabs(o->n_medium) < 1.0e300)) return OSOG_EINVAL;
    if (!o->lambda_um) return OSOG_EINVAL;
    for (int b = 0; b < o->B; ++b)
        if (!(o->lambda_um[b] > 0.0) || !(o->lambda_um[b] < 1.0e300)) return OSOG_EINVAL;
    if (!(fabs(o->tilt_x_rad) < 1.0e300) || !(fabs(o->tilt_y_rad) < 1.0e300)) return OSOG_EINVAL;
    if (!(fabs(o->topography_amplitude) < 1.0e30)) return OSOG_EINVAL;
    if (N > 0) {
        const void* cols[] = {p->cx, p->cy, p->qw, p->qx, p->qy, p->qz, p->d0, p->d1, p->d2, p->n_p, p->kind};
        for (const void* q : cols)
            if (!q) return OSOG_EINVAL;
        const void* fcols[] = {p->cx, p->cy, p->qw, p->qx, p->qy, p->qz, p->d0, p->d1, p->d2, p->n_p};
        for (const void* q : fcols)
            if (reinterpret_cast<uintptr_t>(q) & 3u) return OSOG_EINVAL;
    }
    if (o->B > 1 && !p->frame_start) return OSOG_EINVAL;
    return OSOG_OK;
}

int check_intensity(const osog_optics* o)
{
    if (!(o->read_noise_sigma >= 0.0) || !(o->read_noise_sigma < 1.0e300)) return OSOG_EINVAL;
    if (!(fabs(o->defocus_um) < 1.0e300)) return OSOG_EINVAL;
    if (!(o->shot_noise_photons >= 0.0) || !(o->shot_noise_photons < 1.0e300)) return OSOG_EINVAL;
    if (o->pupil_enabled) {
        if (!o->NA) return OSOG_EINVAL;
        for (int b = 0; b < o->B; ++b)
            if (!(o->NA[b] > 0.0) || !(o->NA[b] < 1.0e300)) return OSOG_EINVAL;
    }
    return OSOG_OK;
}

struct DeviceGuard {
    int prev = -1;
    bool ok = false;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        ok = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

// one 2-D C2C transform of each of the B frames in `src` into `buf` (src == buf: in place; src is never written otherwise)
int fft_frames(osog_ctx* c, float2* buf, int B, int sign, const float2* src = nullptr)
{
    const size_t npx = (size_t)c->H * c->W;
    float2* in = src ? const_cast<float2*>(src) : buf;
    if (B == c->max_frames && c->has_plan_batch) {
        cufftResult r = cufftExecC2C(c->plan_batch, reinterpret_cast<cufftComplex*>(in),
                                     reinterpret_cast<cufftComplex*>(buf), sign);
        if (r != CUFFT_SUCCESS) { c->last_cuda_error = 10000 + (int)r; return OSOG_ECUDA; }
        return OSOG_OK;
    }
    for (int b = 0; b < B; ++b) {
        cufftComplex* f = reinterpret_cast<cufftComplex*>(buf + (size_t)b * npx);
        cufftResult r = cufftExecC2C(c->plan_one, reinterpret_cast<cufftComplex*>(in + (size_t)b * npx), f, sign);
        if (r != CUFFT_SUCCESS) { c->last_cuda_error = 10000 + (int)r; return OSOG_ECUDA; }
    }
    return OSOG_OK;
}

// first use of the fused library stage by this context: the kept-column scratch and the twiddle tables
int ensure_fused_optics(osog_ctx* c)
{
    if (c->fo_ready) return OSOG_OK;
    cudaError_t ea = cudaSuccess;
    if (!c->spec_t) ea = dalloc(&c->spec_t, (size_t)c->max_frames * c->H * c->W, c);
    if (ea == cudaSuccess && !c->tw_w) ea = dalloc(&c->tw_w, (size_t)c->W, c);
    if (ea == cudaSuccess && c->H != c->W && !c->tw_h) ea = dalloc(&c->tw_h, (size_t)c->H, c);
    if (ea == cudaSuccess) ea = launch_fo_twiddles(c, c->tw_w, c->W);
    if (ea == cudaSuccess && c->H != c->W) ea = launch_fo_twiddles(c, c->tw_h, c->H);
    if (ea != cudaSuccess) {                         // (what was allocated stays with the context and is reused by the next call)
        cudaGetLastError();
        return ea == cudaErrorMemoryAllocation ? OSOG_ENOMEM : cuda_fail(c, ea);
    }
    if (c->H == c->W) c->tw_h = c->tw_w;
    c->fo_ready = true;
    return OSOG_OK;
}

// forward FFT of the B frames of `src` into `buf` (src == nullptr: `buf` in place), pupil function, inverse FFT, then the
// sensor into d_intensity
int optics_stage(osog_ctx* c, const osog_optics* o, float2* buf, float* d_intensity, const float2* src = nullptr)
{
    const int B = o->B;
    if (fused_optics_applies(c)) {
        // power-of-two frames: row FFT -> [column FFT, pupil, inverse column FFT] of the columns the pupil keeps -> inverse row
        // FFT + sensor, three kernels of this library (optics.cu); the field is only read
        const int rs = ensure_fused_optics(c);
        if (rs != OSOG_OK) return rs;
        const cudaError_t ef = launch_fused_optics(c, o, src ? src : buf, c->spec_t, c->tw_w, c->tw_h, d_intensity);
        return ef == cudaSuccess ? OSOG_OK : cuda_fail(c, ef);
    }
    int r = fft_frames(c, buf, B, CUFFT_FORWARD, src);
    if (r != OSOG_OK) return r;
    cudaError_t e = launch_pupil(c, B, buf, o->pitch_um, o->defocus_um != 0.0);
    if (e != cudaSuccess) return cuda_fail(c, e);
    if ((r = fft_frames(c, buf, B, CUFFT_INVERSE)) != OSOG_OK) return r;
    e = launch_sensor(c, B, buf, d_intensity, o->read_noise_sigma, o->shot_noise_photons, o->seed);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

int check_dic(const osog_ctx* c, const osog_dic* d)
{
    if (!d || d->struct_size != sizeof(osog_dic)) return OSOG_EINVAL;
    if (d->shear_x_px <= -c->W || d->shear_x_px >= c->W || d->shear_y_px <= -c->H || d->shear_y_px >= c->H) return OSOG_EINVAL;
    if (!(fabs(d->bias_rad) < 1.0e300)) return OSOG_EINVAL;
    return OSOG_OK;
}

// Eq. 5 on the B frames of U held in c->field (overwritten): see include/osog.h, osog_render_dic
// field: the exit wave (only read); nullptr = the context's own frame batch
int dic_stage(osog_ctx* c, const osog_optics* o, const osog_dic* d, float* d_dic, const float2* field = nullptr)
{
    if (!field) field = c->field;
    const int B = o->B;
    const double hw = (double)c->H * c->W;
    if (!c->work || !c->otf) {                       // first DIC call of this context: two more complex batches
        for (float2** buf : {&c->work, &c->otf}) {
            if (*buf) continue;
            cudaError_t ea = dalloc(buf, (size_t)c->max_frames * c->H * c->W, c);
            if (ea != cudaSuccess) { cudaGetLastError(); *buf = nullptr; return ea == cudaErrorMemoryAllocation ? OSOG_ENOMEM : cuda_fail(c, ea); }
        }
    }
    if (!c->otf_key) c->otf_key = new (std::nothrow) std::vector<double>();
    if (!c->otf_key) return OSOG_ENOMEM;
    const bool defocus = o->defocus_um != 0.0;
    cudaError_t e;
    int r;
    const bool fused = fused_optics_applies(c);      // power-of-two frames: the three fused kernels of optics.cu (below)
    // D = |U(r+ds) e^{i theta} - U(r-ds) e^{-i theta}|^2 and its spectrum
    if (!fused) {
        if ((e = launch_dic_shear(c, B, field, c->work, d->shear_x_px, d->shear_y_px, d->bias_rad)) != cudaSuccess) return cuda_fail(c, e);
        if ((r = fft_frames(c, c->work, B, CUFFT_FORWARD)) != OSOG_OK) return r;
    }
    // optical transfer function: P -> h_obj = F^-1{P} -> |h_obj|^2 -> F{.}; it depends on the optics alone, so it is kept
    // and rebuilt only when they change (the same stream orders the rebuild against earlier readers)
    std::vector<double> key = {(double)B, o->pitch_um, o->n_medium, o->defocus_um, (double)(o->pupil_enabled != 0)};
    for (int b = 0; b < B; ++b) {
        key.push_back(o->lambda_um[b]);
        key.push_back(o->pupil_enabled ? o->NA[b] : 0.0);
    }
    if (key != *c->otf_key) {
        c->otf_key->clear();
        if ((e = launch_pupil_fill(c, B, c->otf, o->pitch_um, defocus)) != cudaSuccess) return cuda_fail(c, e);
        if ((r = fft_frames(c, c->otf, B, CUFFT_INVERSE)) != OSOG_OK) return r;
        if ((e = launch_abs2(c, B, c->otf, 1.0 / (hw * hw))) != cudaSuccess) return cuda_fail(c, e);    // cuFFT's inverse is unnormalised
        if ((r = fft_frames(c, c->otf, B, CUFFT_FORWARD)) != OSOG_OK) return r;
        *c->otf_key = key;
    }
    // I = F^-1{ F{D} OTF }
    if (fused) {
        // row FFT of D (formed on the fly from the field) -> [column FFT, x OTF / (H W), inverse column FFT] of the columns inside
        // the OTF's support (twice the pupil's radius) -> inverse row FFT, real part, sensor
        if ((r = ensure_fused_optics(c)) != OSOG_OK) return r;
        e = launch_fused_dic(c, o, field, c->otf, c->spec_t, c->tw_w, c->tw_h, d->shear_x_px, d->shear_y_px, d->bias_rad, d_dic);
        return e == cudaSuccess ? OSOG_OK : cuda_fail(c, e);
    }
    if ((e = launch_cmul(c, B, c->work, c->otf, 1.0 / hw)) != cudaSuccess) return cuda_fail(c, e);
    if ((r = fft_frames(c, c->work, B, CUFFT_INVERSE)) != OSOG_OK) return r;
    if ((e = launch_sensor_real(c, B, c->work, d_dic, o->read_noise_sigma, o->shot_noise_photons, o->seed)) != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

}  // namespace

extern "C" {

int osog_tile_size(void) { return kTile; }

const char* osog_strerror(int code)
{
    switch (code) {
        case OSOG_OK: return "ok";
        case OSOG_EINVAL: return "invalid argument";
        case OSOG_ECUDA: return "CUDA or cuFFT failure";
        case OSOG_ECAPACITY: return "particle-tile pair list overflow";
        case OSOG_ENOMEM: return "out of memory";
        case OSOG_ELIMIT: return "beyond the fixed limits of osog_render_opd_static (particles, frames or tiles)";
        default: return "unknown error";
    }
}

int osog_last_cuda_error(const osog_ctx* ctx) { return ctx ? ctx->last_cuda_error : 0; }

int osog_destroy(osog_ctx* c)
{
    if (!c) return OSOG_EINVAL;
    DeviceGuard g(c->device);
    if (c->has_plan_one) cufftDestroy(c->plan_one);
    if (c->has_plan_batch) cufftDestroy(c->plan_batch);
    cudaFree(c->rec); cudaFree(c->rec2); cudaFree(c->tbox); cudaFree(c->pframe); cudaFree(c->count);
    cudaFree(c->list); cudaFree(c->meta); cudaFree(c->slices); cudaFree(c->offset); cudaFree(c->done); cudaFree(c->optics);
    cudaFree(c->status); cudaFree(c->field); cudaFree(c->work); cudaFree(c->otf); cudaFree(c->bf_h); cudaFree(c->spec_partial);
    cudaFree(c->spec_t); cudaFree(c->tw_w); if (c->tw_h != c->tw_w) cudaFree(c->tw_h);
    delete c->otf_key;
    delete c->guards;
    if (c->h_status) cudaFreeHost(c->h_status);
    delete c;
    return OSOG_OK;
}

int osog_create(osog_ctx** out, const osog_config* cfg)
{
    if (!out) return OSOG_EINVAL;
    *out = nullptr;
    if (!cfg || cfg->struct_size != sizeof(osog_config)) return OSOG_EINVAL;
    if (cfg->H < 1 || cfg->W < 1 || cfg->H > 32768 || cfg->W > 32768) return OSOG_EINVAL;
    if (cfg->max_frames < 1 || cfg->max_frames > 65535 || cfg->max_particles < 0 || cfg->max_pairs < 0) return OSOG_EINVAL;
    if (cfg->max_particles > 0x1fffffffll) return OSOG_EINVAL;       // 29-bit particle index in the survivor queues
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev) return OSOG_ECUDA;

    osog_ctx* c = new (std::nothrow) osog_ctx;
    if (!c) return OSOG_ENOMEM;
    std::memset(c, 0, sizeof(*c));
    c->device = cfg->device;
    c->last_has_ramp = -1;
    c->stream = static_cast<cudaStream_t>(cfg->stream);
    c->H = cfg->H; c->W = cfg->W; c->max_frames = cfg->max_frames;
    c->max_particles = cfg->max_particles;
    c->max_pairs = cfg->max_pairs > 0 ? cfg->max_pairs : 64 * cfg->max_particles + 1024;
    if (c->max_pairs > 0xfffffff0ll) c->max_pairs = 0xfffffff0ll;
    c->ntx = (c->W + kTile - 1) / kTile;
    c->nty = (c->H + kTile - 1) / kTile;
    c->max_tiles = (long long)c->max_frames * c->ntx * c->nty;
    if (c->max_tiles > 0x7fffffffll) { delete c; return OSOG_EINVAL; }
    c->count_stride = (c->max_tiles + 3) & ~3ll;
    // staging slice of one tile: about the mean list length the capacity allows, 32 .. 1,024 entries (1,024 = what
    // k_sort_cull sorts in shared memory); a longer list is rebuilt in order from the tile ranges, see k_sort_cull
    {
        long long cap = (c->max_pairs + c->max_tiles - 1) / c->max_tiles;
        cap = (cap + 3) & ~3ll;
        if (cap < 32) cap = 32;
        if (cap > 1024) cap = 1024;
        c->slice_cap = (int)cap;
    }

    DeviceGuard g(c->device);
    if (!g.ok) { delete c; return OSOG_ECUDA; }
    c->guards = new (std::nothrow) std::vector<std::pair<unsigned char*, size_t>>();
    const size_t np = (size_t)c->max_particles, npx = (size_t)c->H * c->W;
    cudaError_t e = cudaSuccess;
    auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
    A(dalloc(&c->rec, np * kRecWords, c));
    A(dalloc(&c->rec2, np * kPairWords, c));
    A(dalloc(&c->tbox, np, c));
    A(dalloc(&c->pframe, np, c));
    A(dalloc(&c->count, 2 * (size_t)c->count_stride, c));
    A(dalloc(&c->offset, (size_t)c->max_tiles + 4, c));
    A(dalloc(&c->done, 1, c));
    A(dalloc(&c->slices, (size_t)c->max_tiles * c->slice_cap, c));
    A(dalloc(&c->list, (size_t)c->max_pairs, c));
    A(dalloc(&c->meta, (size_t)c->max_pairs, c));
    A(dalloc(&c->optics, (size_t)c->max_frames, c));
    A(dalloc(&c->status, 2, c));
    A(dalloc(&c->field, (size_t)c->max_frames * npx, c));
    if (e == cudaSuccess) e = cudaMallocHost(reinterpret_cast<void**>(&c->h_status), sizeof(DeviceStatus));
    if (e == cudaSuccess) e = cudaMemset(c->status, 0, 2 * sizeof(DeviceStatus));
    if (e == cudaSuccess) e = cudaMemset(c->count, 0, sizeof(uint32_t) * 2 * (size_t)c->count_stride);
    if (e == cudaSuccess) e = cudaMemset(c->done, 0, sizeof(uint32_t));
    if (e != cudaSuccess) {
        const bool oom = e == cudaErrorMemoryAllocation;
        cudaGetLastError();
        osog_destroy(c);
        return oom ? OSOG_ENOMEM : OSOG_ECUDA;
    }
    int dims[2] = {c->H, c->W};
    if (cufftPlanMany(&c->plan_one, 2, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2C, 1) == CUFFT_SUCCESS) {
        c->has_plan_one = true;
        cufftSetStream(c->plan_one, c->stream);
    }
    if (c->max_frames > 1 &&
        cufftPlanMany(&c->plan_batch, 2, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2C, c->max_frames) == CUFFT_SUCCESS) {
        c->has_plan_batch = true;
        cufftSetStream(c->plan_batch, c->stream);
    }
    if (!c->has_plan_one) { osog_destroy(c); return OSOG_ECUDA; }
    *out = c;
    return OSOG_OK;
}

static int render_common(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, float* d_opd,
                         float2* d_field, bool unit_dn = false)
{
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    cudaError_t e = launch_binning(c, p, N, o, nullptr, unit_dn);
    if (e != cudaSuccess) return cuda_fail(c, e);
    const bool has_ramp = o->tilt_x_rad != 0.0 || o->tilt_y_rad != 0.0;
    e = launch_compose(c, o->B, has_ramp, d_opd, d_field);
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->last_has_ramp = has_ramp ? 1 : 0;             // osog_debug_recompose_field may re-run this composition
    c->scratch_dirty = false;                        // k_sort_cull cleared the counter / status slots of the next call
    return OSOG_OK;
}

int osog_render_opd(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, float* d_opd)
{
    const int r = check_call(c, p, N, o, d_opd);
    if (r != OSOG_OK) return r;
    return render_common(c, p, N, o, d_opd, nullptr);
}

int osog_render_field(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, float* d_field)
{
    const int r = check_call(c, p, N, o, d_field);
    if (r != OSOG_OK) return r;
    return render_common(c, p, N, o, nullptr, reinterpret_cast<float2*>(d_field));
}

int osog_render_intensity(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, float* d_intensity)
{
    int r = check_call(c, p, N, o, d_intensity);
    if (r != OSOG_OK) return r;
    if ((r = check_intensity(o)) != OSOG_OK) return r;
    if ((r = render_common(c, p, N, o, nullptr, c->field)) != OSOG_OK) return r;
    DeviceGuard g(c->device);
    return optics_stage(c, o, c->field, d_intensity);
}

int osog_field_to_intensity(osog_ctx* c, const osog_optics* o, const float* d_field, float* d_intensity)
{
    if (!c || !o || !d_field || !d_intensity || o->struct_size != sizeof(osog_optics)) return OSOG_EINVAL;
    if (o->B < 1 || o->B > c->max_frames || !o->lambda_um || !aligned16(d_field) || !aligned16(d_intensity)) return OSOG_EINVAL;
    if (!(o->pitch_um > 0.0)) return OSOG_EINVAL;
    for (int b = 0; b < o->B; ++b)
        if (!(o->lambda_um[b] > 0.0)) return OSOG_EINVAL;
    int r = check_intensity(o);
    if (r != OSOG_OK) return r;
    DeviceGuard g(c->device);
    cudaError_t e = upload_optics(c, o, nullptr);
    if (e != cudaSuccess) return cuda_fail(c, e);
    // the first transform reads the caller's field and writes the context's frame: no copy, the stage the product runs
    return optics_stage(c, o, c->field, d_intensity, reinterpret_cast<const float2*>(d_field));
}

int osog_render_dic(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, const osog_dic* d, float* d_dic)
{
    int r = check_call(c, p, N, o, d_dic);
    if (r != OSOG_OK) return r;
    if ((r = check_intensity(o)) != OSOG_OK) return r;
    if ((r = check_dic(c, d)) != OSOG_OK) return r;
    if ((r = render_common(c, p, N, o, nullptr, c->field)) != OSOG_OK) return r;
    DeviceGuard g(c->device);
    return dic_stage(c, o, d, d_dic);
}

int osog_render_brightfield(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, const osog_brightfield* bf,
                            float* d_intensity)
{
    int r = check_call(c, p, N, o, d_intensity);
    if (r != OSOG_OK) return r;
    if ((r = check_intensity(o)) != OSOG_OK) return r;
    if (!bf || bf->struct_size != sizeof(osog_brightfield)) return OSOG_EINVAL;
    if (!(bf->n_particle > 0.0) || !(bf->n_particle < 1.0e300) || !(o->n_medium > 0.0) || !(fabs(bf->delta_mu_per_um) < 1.0e300) ||
        !(fabs(bf->caustic_gain_um) < 1.0e300))
        return OSOG_EINVAL;
    DeviceGuard g(c->device);
    if (!c->bf_h) {                                  // first brightfield call of this context: one real frame batch
        const cudaError_t ea = dalloc(&c->bf_h, (size_t)c->max_frames * c->H * c->W, c);
        if (ea != cudaSuccess) { cudaGetLastError(); c->bf_h = nullptr; return ea == cudaErrorMemoryAllocation ? OSOG_ENOMEM : cuda_fail(c, ea); }
    }
    // height map (the hot path with unit index contrast), then the exit wave (the hot path proper); A multiplies U in place
    if ((r = render_common(c, p, N, o, c->bf_h, nullptr, true)) != OSOG_OK) return r;
    if ((r = render_common(c, p, N, o, nullptr, c->field)) != OSOG_OK) return r;
    const cudaError_t e = launch_brightfield(c, o->B, c->field, c->bf_h, o->pitch_um, o->n_medium, bf->n_particle,
                                             bf->delta_mu_per_um, bf->caustic_gain_um);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return optics_stage(c, o, c->field, d_intensity);
}

int osog_field_to_dic(osog_ctx* c, const osog_optics* o, const osog_dic* d, const float* d_field, float* d_dic)
{
    if (!c || !o || !d_field || !d_dic || o->struct_size != sizeof(osog_optics)) return OSOG_EINVAL;
    if (o->B < 1 || o->B > c->max_frames || !o->lambda_um || !aligned16(d_field) || !aligned16(d_dic)) return OSOG_EINVAL;
    if (!(o->pitch_um > 0.0)) return OSOG_EINVAL;
    for (int b = 0; b < o->B; ++b)
        if (!(o->lambda_um[b] > 0.0)) return OSOG_EINVAL;
    int r = check_intensity(o);
    if (r != OSOG_OK) return r;
    if ((r = check_dic(c, d)) != OSOG_OK) return r;
    DeviceGuard g(c->device);
    cudaError_t e = upload_optics(c, o, nullptr);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return dic_stage(c, o, d, d_dic, reinterpret_cast<const float2*>(d_field));      // (the stage only reads the field: no copy)
}

int osog_render_opd_atomic(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, float* d_opd)
{
    const int r = check_call(c, p, N, o, d_opd);
    if (r != OSOG_OK) return r;
    DeviceGuard g(c->device);
    cudaError_t e = launch_binning(c, p, N, o);      // records + bounding boxes (the tile lists are not used)
    if (e != cudaSuccess) return cuda_fail(c, e);
    e = launch_compose_atomic(c, N, o->B, d_opd);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

int osog_particle_obbs(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, float* d_obb)
{
    if (N == 0) return (c && p && o) ? OSOG_OK : OSOG_EINVAL;
    const int r = check_call(c, p, N, o, d_obb);
    if (r != OSOG_OK) return r;
    DeviceGuard g(c->device);
    cudaError_t e = launch_binning(c, p, N, o, d_obb);   // k_prepare alone; the tile lists it leaves are not used
    if (e != cudaSuccess) return cuda_fail(c, e);        // (scratch_dirty stays set: the next render call clears them)
    return OSOG_OK;
}

int osog_render_height(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, float* d_h, float* d_grad,
                       float* d_lap)
{
    int r = check_call(c, p, N, o, d_h);
    if (r != OSOG_OK) return r;
    if ((d_grad && !aligned16(d_grad)) || (d_lap && !aligned16(d_lap))) return OSOG_EINVAL;
    if ((r = render_common(c, p, N, o, d_h, nullptr, true)) != OSOG_OK) return r;     // the hot path with unit index contrast
    if (!d_grad && !d_lap) return OSOG_OK;
    DeviceGuard g(c->device);
    const cudaError_t e = launch_height_stencil(c, o->B, d_h, o->pitch_um, d_grad, d_lap);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

static int gbuffer_common(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, int32_t* d_top_id, float* d_depth,
                          float* d_normal)
{
    if (!d_top_id || !aligned16(d_top_id) || (d_normal && !aligned16(d_normal))) return OSOG_EINVAL;
    const int r = check_call(c, p, N, o, d_depth);
    if (r != OSOG_OK) return r;
    if (p->cz != nullptr && (reinterpret_cast<uintptr_t>(p->cz) & 3u)) return OSOG_EINVAL;
    DeviceGuard g(c->device);
    cudaError_t e = launch_binning(c, p, N, o);
    if (e != cudaSuccess) return cuda_fail(c, e);
    e = launch_gbuffer(c, o->B, o->B > 1 ? p->frame_start : nullptr, o->pitch_um, d_top_id, d_depth, d_normal);
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->scratch_dirty = false;
    return OSOG_OK;
}

int osog_render_gbuffer(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, int32_t* d_top_id, float* d_depth)
{
    return gbuffer_common(c, p, N, o, d_top_id, d_depth, nullptr);
}

int osog_render_gbuffer_normals(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, int32_t* d_top_id,
                                float* d_depth, float* d_normal)
{
    if (!d_normal) return OSOG_EINVAL;
    return gbuffer_common(c, p, N, o, d_top_id, d_depth, d_normal);
}

int osog_backward_intensity(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, const float* d_gI, float* d_gopd)
{
    if (!d_gI || !aligned16(d_gI)) return OSOG_EINVAL;
    int r = check_call(c, p, N, o, d_gopd);
    if (r != OSOG_OK) return r;
    if ((r = check_intensity(o)) != OSOG_OK) return r;
    if ((r = render_common(c, p, N, o, nullptr, c->field)) != OSOG_OK) return r;      // U, the exit wave
    DeviceGuard g(c->device);
    if (!c->work) {                                  // first call of this kind: a second complex batch
        const cudaError_t ea = dalloc(&c->work, (size_t)c->max_frames * c->H * c->W, c);
        if (ea != cudaSuccess) { cudaGetLastError(); c->work = nullptr; return ea == cudaErrorMemoryAllocation ? OSOG_ENOMEM : cuda_fail(c, ea); }
    }
    if (fused_optics_applies(c)) {                   // power-of-two frames: two passes of the three fused kernels (optics.cu)
        if ((r = ensure_fused_optics(c)) != OSOG_OK) return r;
        const cudaError_t ef = launch_fused_optics_adjoint(c, o, c->field, c->work, c->spec_t, c->tw_w, c->tw_h, d_gI, d_gopd);
        return ef == cudaSuccess ? OSOG_OK : cuda_fail(c, ef);
    }
    const int B = o->B;
    const bool defocus = o->defocus_um != 0.0;
    cudaError_t e = cudaMemcpyAsync(c->work, c->field, sizeof(float2) * (size_t)B * c->H * c->W, cudaMemcpyDeviceToDevice, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    // V = U * h_obj
    if ((r = fft_frames(c, c->work, B, CUFFT_FORWARD)) != OSOG_OK) return r;
    if ((e = launch_pupil(c, B, c->work, o->pitch_um, defocus)) != cudaSuccess) return cuda_fail(c, e);
    if ((r = fft_frames(c, c->work, B, CUFFT_INVERSE)) != OSOG_OK) return r;
    // g_V = G_I V;  g_U = F^-1{ conj(P) F{g_V} }
    if ((e = launch_mul_real(c, B, c->work, d_gI)) != cudaSuccess) return cuda_fail(c, e);
    if ((r = fft_frames(c, c->work, B, CUFFT_FORWARD)) != OSOG_OK) return r;
    if ((e = launch_pupil_conj(c, B, c->work, o->pitch_um, defocus)) != cudaSuccess) return cuda_fail(c, e);
    if ((r = fft_frames(c, c->work, B, CUFFT_INVERSE)) != OSOG_OK) return r;
    // dL/dOPD = (4 pi / lambda) Im(g_U conj(U))
    if ((e = launch_gopd(c, B, c->work, c->field, d_gopd)) != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

int osog_backward_np(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, const float* d_gopd, float* d_gnp)
{
    if (!d_gopd || !aligned16(d_gopd)) return OSOG_EINVAL;
    if (N == 0) return (c && p && o) ? OSOG_OK : OSOG_EINVAL;
    const int r = check_call(c, p, N, o, d_gnp);
    if (r != OSOG_OK) return r;
    if (o->topography_amplitude != 0.0) return OSOG_EINVAL;   // the gathers differentiate the smooth bodies (see osog.h)
    DeviceGuard g(c->device);
    cudaError_t e = launch_binning(c, p, N, o);      // records + bounding boxes (the tile lists are not used)
    if (e != cudaSuccess) return cuda_fail(c, e);    // (scratch_dirty stays set: the next render call clears them)
    e = launch_backward_np(c, N, d_gopd, d_gnp);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

int osog_backward_centre(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, const float* d_gopd, float* d_gc)
{
    if (!d_gopd || !aligned16(d_gopd)) return OSOG_EINVAL;
    if (N == 0) return (c && p && o) ? OSOG_OK : OSOG_EINVAL;
    const int r = check_call(c, p, N, o, d_gc);
    if (r != OSOG_OK) return r;
    if (o->topography_amplitude != 0.0) return OSOG_EINVAL;   // the gathers differentiate the smooth bodies (see osog.h)
    DeviceGuard g(c->device);
    cudaError_t e = launch_binning(c, p, N, o);      // records + bounding boxes (the tile lists are not used)
    if (e != cudaSuccess) return cuda_fail(c, e);    // (scratch_dirty stays set: the next render call clears them)
    e = launch_backward_centre(c, N, o->pitch_um, d_gopd, d_gc);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

int osog_spectral_loss(osog_ctx* c, int32_t B, const float* d_I, const float* d_I_target, double eps, double* d_loss, float* d_gI)
{
    if (!c || !d_I || !d_I_target || !d_loss || B < 1 || B > c->max_frames || !(eps > 0.0) || !(eps < 1.0e300)) return OSOG_EINVAL;
    if (!aligned16(d_I) || !aligned16(d_I_target) || (d_gI && !aligned16(d_gI))) return OSOG_EINVAL;
    DeviceGuard g(c->device);
    if (!c->work) {
        const cudaError_t ea = dalloc(&c->work, (size_t)c->max_frames * c->H * c->W, c);
        if (ea != cudaSuccess) { cudaGetLastError(); c->work = nullptr; return ea == cudaErrorMemoryAllocation ? OSOG_ENOMEM : cuda_fail(c, ea); }
    }
    const size_t nblk = ((size_t)c->H * c->W + 255) / 256;
    if (!c->spec_partial) {
        const cudaError_t ea = dalloc(&c->spec_partial, (size_t)c->max_frames * nblk, c);
        if (ea != cudaSuccess) { cudaGetLastError(); c->spec_partial = nullptr; return ea == cudaErrorMemoryAllocation ? OSOG_ENOMEM : cuda_fail(c, ea); }
    }
    c->last_has_ramp = -1;                           // the context's complex frame is overwritten
    cudaError_t e = launch_real_to_complex(c, B, d_I, d_I_target, c->field, c->work);
    if (e != cudaSuccess) return cuda_fail(c, e);
    int r;
    if ((r = fft_frames(c, c->field, B, CUFFT_FORWARD)) != OSOG_OK) return r;
    if ((r = fft_frames(c, c->work, B, CUFFT_FORWARD)) != OSOG_OK) return r;
    if ((e = launch_spectral_terms(c, B, c->field, c->work, eps, c->spec_partial, d_loss, d_gI != nullptr)) != cudaSuccess) return cuda_fail(c, e);
    if (!d_gI) return OSOG_OK;
    if ((r = fft_frames(c, c->field, B, CUFFT_FORWARD)) != OSOG_OK) return r;
    if ((e = launch_real_part(c, B, c->field, d_gI)) != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

int osog_backward_params(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, const float* d_gopd, float* d_gpar)
{
    if (!d_gopd || !aligned16(d_gopd)) return OSOG_EINVAL;
    if (N == 0) return (c && p && o) ? OSOG_OK : OSOG_EINVAL;
    const int r = check_call(c, p, N, o, d_gpar);
    if (r != OSOG_OK) return r;
    if (o->topography_amplitude != 0.0) return OSOG_EINVAL;   // the gathers differentiate the smooth bodies (see osog.h)
    DeviceGuard g(c->device);
    cudaError_t e = launch_binning(c, p, N, o);      // tile ranges, frames and pixel bounding boxes (the tile lists are not used)
    if (e != cudaSuccess) return cuda_fail(c, e);    // (scratch_dirty stays set: the next render call clears them)
    e = launch_backward_params(c, p, N, o->pitch_um, o->n_medium, d_gopd, d_gpar);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

int osog_backward_particles(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, const float* d_gopd, float* d_gnp,
                            float* d_gc, float* d_gpar)
{
    if (!d_gopd || !aligned16(d_gopd)) return OSOG_EINVAL;
    float* first = d_gnp ? d_gnp : (d_gc ? d_gc : d_gpar);       // at least one output
    if (!first) return OSOG_EINVAL;
    if (d_gc && (reinterpret_cast<uintptr_t>(d_gc) & 7u)) return OSOG_EINVAL;
    if (N == 0) return (c && p && o) ? OSOG_OK : OSOG_EINVAL;
    const int r = check_call(c, p, N, o, first);
    if (r != OSOG_OK) return r;
    if (o->topography_amplitude != 0.0) return OSOG_EINVAL;   // the gathers differentiate the smooth bodies (see osog.h)
    DeviceGuard g(c->device);
    cudaError_t e = launch_binning(c, p, N, o);      // tile ranges, frames and pixel bounding boxes (the tile lists are not used)
    if (e != cudaSuccess) return cuda_fail(c, e);
    e = launch_backward_params(c, p, N, o->pitch_um, o->n_medium, d_gopd, d_gpar, d_gnp, d_gc);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

int osog_render_opd_smem_atomic(osog_ctx* c, const osog_particles* p, int64_t N, const osog_optics* o, float* d_opd)
{
    const int r = check_call(c, p, N, o, d_opd);
    if (r != OSOG_OK) return r;
    DeviceGuard g(c->device);
    cudaError_t e = launch_binning(c, p, N, o);
    if (e != cudaSuccess) return cuda_fail(c, e);
    e = launch_compose_smem_atomic(c, o->B, d_opd);
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->scratch_dirty = false;
    return OSOG_OK;
}

int osog_debug_recompose_field(osog_ctx* c, float* d_field)
{
    if (!c || !d_field || !aligned16(d_field) || c->last_B < 1 || c->last_has_ramp < 0) return OSOG_EINVAL;
    DeviceGuard g(c->device);
    cudaError_t e = launch_compose(c, c->last_B, c->last_has_ramp != 0, nullptr, reinterpret_cast<float2*>(d_field), false);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

int osog_status(osog_ctx* c, uint32_t* status_bits, int64_t* pairs)
{
    if (!c) return OSOG_EINVAL;
    DeviceGuard g(c->device);
    cudaError_t e = cudaMemcpyAsync(c->h_status, c->status + c->status_idx, sizeof(DeviceStatus), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    const bool overflow = (c->h_status->bits & OSOG_WOVERFLOW) != 0u;
    if (status_bits) *status_bits = c->h_status->bits;
    if (pairs) *pairs = (int64_t)c->h_status->pairs;     // total of the device scan: on overflow, the max_pairs that suffices
    return overflow ? OSOG_ECAPACITY : OSOG_OK;
}

int osog_debug_poisson(osog_ctx* c, const float* d_lambda, int64_t n, uint64_t seed, uint32_t frame, int32_t* d_counts)
{
    if (!c || n < 0 || (n > 0 && (!d_lambda || !d_counts))) return OSOG_EINVAL;
    DeviceGuard g(c->device);
    const cudaError_t e = launch_poisson(c, d_lambda, (size_t)n, seed, frame, d_counts);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return OSOG_OK;
}

int osog_debug_check_guards(osog_ctx* c)
{
    if (!c || !c->guards) return OSOG_EINVAL;
    DeviceGuard g(c->device);
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    int bad = 0;
    std::vector<unsigned char> h(kGuardBytes);
    for (const auto& gb : *c->guards) {
        if ((e = cudaMemcpy(h.data(), gb.first, gb.second, cudaMemcpyDeviceToHost)) != cudaSuccess) return cuda_fail(c, e);
        for (size_t k = 0; k < gb.second; ++k)
            if (h[k] != kGuardByte) { ++bad; break; }
    }
    return bad;
}

int osog_debug_bins(osog_ctx* c, uint32_t* h_offset, uint32_t* h_list, int64_t cap, int64_t* n_tiles, int64_t* n_pairs)
{
    if (!c || cap < 0) return OSOG_EINVAL;
    uint32_t bits = 0;
    int64_t pairs = 0;
    const int r = osog_status(c, &bits, &pairs);
    if (r == OSOG_ECUDA || r == OSOG_EINVAL) return r;
    if (n_tiles) *n_tiles = c->last_tiles;
    if (n_pairs) *n_pairs = pairs;
    if (c->last_tiles <= 0 || (!h_offset && !h_list)) return r;
    DeviceGuard g(c->device);
    // the scan (offset) and the compact sorted lists are the device's own (k_prepare's scan, k_sort_cull's fill): plain copies
    const size_t nt = (size_t)c->last_tiles;
    cudaError_t e = cudaSuccess;
    if (h_offset) e = cudaMemcpy(h_offset, c->offset, sizeof(uint32_t) * (nt + 1), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(c, e);
    if (h_list && r == OSOG_OK && cap > 0) {
        const int64_t n = pairs < cap ? pairs : cap;
        e = cudaMemcpy(h_list, c->list, sizeof(uint32_t) * (size_t)n, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return cuda_fail(c, e);
    }
    return r;
}


// ---- osog_render_opd_static: the hot path without any allocation (osog.h) --------------------------------------------------
// All scratch of one call lives in ONE file-scope device array of a fixed, modest size; every GPU that loads the library
// holds it until exit.  In host code the array's name is only a stand-in: the device address is asked for once per device
// (cudaGetSymbolAddress with that device current) and carved into the scratch arrays of a static context, which is then
// handed to the same launch functions as a context made by osog_create.
constexpr long long kStaticMaxParticles = OSOG_STATIC_MAX_PARTICLES;
constexpr long long kStaticMaxTiles = OSOG_STATIC_MAX_TILES;
constexpr long long kStaticMaxPairs = OSOG_STATIC_MAX_PAIRS;
constexpr int kStaticMaxFrames = OSOG_STATIC_MAX_FRAMES;
constexpr int kStaticSliceCap = (int)(kStaticMaxPairs / kStaticMaxTiles);      // 256 entries per staging slice
constexpr int kStaticMaxDevices = 64;
constexpr size_t up256(size_t v) { return (v + 255) & ~(size_t)255; }
constexpr size_t kSoRec = 0;
constexpr size_t kSoRec2 = kSoRec + up256(sizeof(float) * kStaticMaxParticles * kRecWords);
constexpr size_t kSoTbox = kSoRec2 + up256(sizeof(float) * kStaticMaxParticles * kPairWords);
constexpr size_t kSoPframe = kSoTbox + up256(sizeof(int4) * kStaticMaxParticles);
constexpr size_t kSoCount = kSoPframe + up256(sizeof(int) * kStaticMaxParticles);
constexpr size_t kSoOffset = kSoCount + up256(sizeof(uint32_t) * 2 * kStaticMaxTiles);
constexpr size_t kSoDone = kSoOffset + up256(sizeof(uint32_t) * (kStaticMaxTiles + 4));
constexpr size_t kSoSlices = kSoDone + 256;
constexpr size_t kSoList = kSoSlices + up256(sizeof(uint32_t) * kStaticMaxTiles * kStaticSliceCap);
constexpr size_t kSoMeta = kSoList + up256(sizeof(uint32_t) * kStaticMaxPairs);
constexpr size_t kSoOptics = kSoMeta + up256(sizeof(uint16_t) * kStaticMaxPairs);
constexpr size_t kSoStatus = kSoOptics + up256(sizeof(FrameOptics) * kStaticMaxFrames);
constexpr size_t kStaticBytes = kSoStatus + 256;
static_assert(kStaticBytes <= OSOG_STATIC_SCRATCH_BYTES, "osog.h states the size of the static scratch");
static_assert(kStaticMaxTiles % 4 == 0 && kStaticSliceCap >= 32 && kStaticSliceCap <= 1024, "slice / scan layout");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

struct StaticSlot {
    bool ready;
    osog_ctx ctx;           // static storage: all zero until set up; never destroyed (it owns nothing)
};
static StaticSlot g_static_slot[kStaticMaxDevices];
static std::mutex g_static_mutex;

int osog_render_opd_static(int device, void* stream, int H, int W, const osog_particles* p, int64_t N, const osog_optics* o,
                           float* d_opd, uint32_t* d_status_bits)
{
    if (!p || !o || !d_opd || H < 1 || W < 1 || device < 0 || device >= kStaticMaxDevices) return OSOG_EINVAL;
    if (o->struct_size != sizeof(osog_optics) || o->B < 1 || N < 0) return OSOG_EINVAL;
    if (d_status_bits && (reinterpret_cast<uintptr_t>(d_status_bits) & 3u)) return OSOG_EINVAL;
    const long long ntx = ((long long)W + kTile - 1) / kTile, nty = ((long long)H + kTile - 1) / kTile;
    if (N > kStaticMaxParticles || o->B > kStaticMaxFrames || (long long)o->B * ntx * nty > kStaticMaxTiles) return OSOG_ELIMIT;
    std::lock_guard<std::mutex> lock(g_static_mutex);      // host side only: calls that overlap ON THE GPU still race (osog.h)
    DeviceGuard g(device);
    if (!g.ok) return OSOG_ECUDA;
    StaticSlot& slot = g_static_slot[device];
    osog_ctx* c = &slot.ctx;
    if (!slot.ready) {
        unsigned char* base = nullptr;                       // this device's copy of the array
        const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&base), g_static_scratch);
        if (e != cudaSuccess || !base) { c->last_cuda_error = (int)e; cudaGetLastError(); return OSOG_ECUDA; }
        c->device = device;
        c->max_frames = kStaticMaxFrames;
        c->max_particles = kStaticMaxParticles;
        c->max_pairs = kStaticMaxPairs;
        c->max_tiles = kStaticMaxTiles;
        c->count_stride = kStaticMaxTiles;
        c->slice_cap = kStaticSliceCap;
        c->rec = reinterpret_cast<float*>(base + kSoRec);
        c->rec2 = reinterpret_cast<float*>(base + kSoRec2);
        c->tbox = reinterpret_cast<int4*>(base + kSoTbox);
        c->pframe = reinterpret_cast<int*>(base + kSoPframe);
        c->count = reinterpret_cast<uint32_t*>(base + kSoCount);
        c->offset = reinterpret_cast<uint32_t*>(base + kSoOffset);
        c->done = reinterpret_cast<uint32_t*>(base + kSoDone);
        c->slices = reinterpret_cast<uint32_t*>(base + kSoSlices);
        c->list = reinterpret_cast<uint32_t*>(base + kSoList);
        c->meta = reinterpret_cast<uint16_t*>(base + kSoMeta);
        c->optics = reinterpret_cast<FrameOptics*>(base + kSoOptics);
        c->status = reinterpret_cast<DeviceStatus*>(base + kSoStatus);
        slot.ready = true;
    }
    c->stream = static_cast<cudaStream_t>(stream);
    c->H = H; c->W = W; c->ntx = (int)ntx; c->nty = (int)nty;
    c->last_has_ramp = -1;
    const int r = check_call(c, p, N, o, d_opd);
    if (r != OSOG_OK) return r;
    // The array keeps the last call's contents (possibly of another frame size, on another stream, or of a call that failed):
    // the tile counters of both slots, the scan ticket and the status words are cleared on this call's stream first.
    c->scratch_dirty = true;
    cudaError_t e = launch_binning(c, p, N, o, nullptr, false);
    if (e != cudaSuccess) return cuda_fail(c, e);
    e = launch_compose(c, o->B, false, d_opd, nullptr);
    if (e != cudaSuccess) return cuda_fail(c, e);
    if (d_status_bits) {
        e = cudaMemcpyAsync(d_status_bits, &(c->status + c->status_idx)->bits, sizeof(uint32_t), cudaMemcpyDeviceToDevice, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e);
    }
    return OSOG_OK;
}

}  // extern "C"
