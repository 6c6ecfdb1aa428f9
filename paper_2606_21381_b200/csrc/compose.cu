// H5-H7 of DESIGN.md: per-tile ordered composition.  One CTA per 32 x 32 pixel tile: sort the tile's
// particle list ascending (deterministic summation order), stage the particle records in shared memory with
// cp.async, let each warp cull the staged particles against its own 16 x 8 pixel sub-tile (ballot
// compaction), evaluate the ray-convex thickness for 4 pixels per lane, accumulate OPD per pixel in fp64
// registers, and write OPD and / or exp(i 2 pi OPD / lambda) * ramp straight from the registers.
#include "osog_internal.cuh"

namespace osog {

struct ComposeArgs {
    const float* rec32;
    const double* rec64;
    const uint32_t* offset;
    uint32_t* list;
    const FrameOptics* optics;
    const float2 *ramp_x, *ramp_y;
    const DeviceStatus* status;
    float* opd;
    float2* field;
    int H, W, ntx, nty;
    int ramp_y_on;
};

__device__ __forceinline__ float fast_sqrt(float x)
{
    float r;
    asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all()
{
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}

// ---- thickness kernels -----------------------------------------------------------------------------------------
// Ellipsoid (kind 0): w = 1 - d^T S d as a quadratic polynomial of the integer pixel offsets, evaluated in
// fp64 (2 DFMA per pixel after the per-row terms), then t = T0 sqrt(max(w, 0)) in fp32.  acc += dn T0 sqrt(w).
template <int NPX>
__device__ __forceinline__ void eval_ellipsoid(const float4* __restrict__ rec, double jd, double id, double (&acc)[NPX])
{
    const float4 h1 = rec[1];
    const double2 c01 = *reinterpret_cast<const double2*>(rec + 2);   // A, B
    const double2 c23 = *reinterpret_cast<const double2*>(rec + 3);   // C, D
    const double2 c45 = *reinterpret_cast<const double2*>(rec + 4);   // E, F1
    const double2 c67 = *reinterpret_cast<const double2*>(rec + 5);   // jc, ic
    const double K = (double)h1.y;
    const double dj = jd - c67.x, di = id - c67.y;
    const double b1 = fma(c01.y, di, c23.y);
    const double c1 = fma(-fma(c23.x, di, c45.x), di, c45.y);
#pragma unroll
    for (int k = 0; k < NPX; ++k) {
        const double djk = dj + (double)k;
        const double g = fma(c01.x, djk, b1);
        const float w = (float)fma(-djk, g, c1);
        const float t = fast_sqrt(fmaxf(w, 0.0f));
        acc[k] = fma((double)t, K, acc[k]);
    }
}

// Prism, fp64, one pixel: the 6 slabs from the fp64 coefficients (exit_k = Cx - U dj - V di, enter_k = Cn - ...).
__device__ __noinline__ double prism_t64(const double* __restrict__ r64, uint32_t vmask, double dj, double di)
{
    double ex = 1.0e300, en = -1.0e300;
    for (int q = 0; q < 6; ++q) {
        const double2 uv = *reinterpret_cast<const double2*>(r64 + 4 * q);
        const double2 xn = *reinterpret_cast<const double2*>(r64 + 4 * q + 2);
        const double m = fma(uv.x, dj, uv.y * di);
        if ((vmask >> q) & 1u) {
            if (fabs(m + xn.x) > xn.y) return 0.0;     // outside a vertical slab: empty chord
        } else {
            const double e = xn.x - m, n = xn.y - m;
            ex = e < ex ? e : ex;
            en = n > en ? n : en;
        }
    }
    const double t = ex - en;
    return t > 0.0 ? t : 0.0;
}

// Prism (kind 1): 6 slabs in fp32; the first ns slabs are the steep ones.  A pixel where a steep slab is (within
// the margin) the active entry or exit face is re-evaluated in fp64 ("precision").
template <int NPX>
__device__ __forceinline__ void eval_prism(const float4* __restrict__ rec, const double* __restrict__ rec64,
                                           float jf, float fi, double (&acc)[NPX])
{
    const float4 h0 = rec[0];
    const float4 h1 = rec[1];
    const uint32_t flags = __float_as_uint(h1.x);
    const int ns = (flags >> 8) & 7;
    const float margin = h1.z;
    const float dj = jf - h0.x, di = fi - h0.y;
    float exs[NPX], ens[NPX], exr[NPX], enr[NPX];
#pragma unroll
    for (int k = 0; k < NPX; ++k) { exs[k] = 3.0e38f; ens[k] = -3.0e38f; exr[k] = 3.0e38f; enr[k] = -3.0e38f; }
    int q = 0;
#pragma unroll 1
    for (; q < ns; ++q) {
        const float4 s = rec[2 + q];                   // U, V, Cx, Cn
        const float ek = fmaf(-s.y, di, s.z), nk = fmaf(-s.y, di, s.w);
#pragma unroll
        for (int k = 0; k < NPX; ++k) {
            const float djk = dj + (float)k;
            exs[k] = fminf(exs[k], fmaf(-s.x, djk, ek));
            ens[k] = fmaxf(ens[k], fmaf(-s.x, djk, nk));
        }
    }
#pragma unroll 1
    for (; q < 6; ++q) {
        const float4 s = rec[2 + q];
        const float ek = fmaf(-s.y, di, s.z), nk = fmaf(-s.y, di, s.w);
#pragma unroll
        for (int k = 0; k < NPX; ++k) {
            const float djk = dj + (float)k;
            exr[k] = fminf(exr[k], fmaf(-s.x, djk, ek));
            enr[k] = fmaxf(enr[k], fmaf(-s.x, djk, nk));
        }
    }
    float t[NPX];
    bool any = false;
    unsigned fmask = 0u;
#pragma unroll
    for (int k = 0; k < NPX; ++k) {
        t[k] = fminf(exs[k], exr[k]) - fmaxf(ens[k], enr[k]);
        bool f = false;
        if (ns > 0) {
            f = (t[k] > -2.0f * margin) && (exs[k] < exr[k] + margin || ens[k] > enr[k] - margin);
            f = f || (flags & kFlagAllF64);
        }
        if (f) fmask |= 1u << k;
        any = any || f;
        t[k] = fmaxf(t[k], 0.0f);
    }
    const double dn = (double)h1.y;
    if (any) {
        const uint32_t id = __float_as_uint(h1.w);
        const double* r64 = rec64 + (size_t)id * kRec64Doubles;
        const double djd = (double)dj, did = (double)di;
#pragma unroll
        for (int k = 0; k < NPX; ++k) {
            if ((fmask >> k) & 1u) acc[k] = fma(prism_t64(r64, flags >> 16, djd + (double)k, did), dn, acc[k]);
            else acc[k] = fma((double)t[k], dn, acc[k]);
        }
    } else {
#pragma unroll
        for (int k = 0; k < NPX; ++k) acc[k] = fma((double)t[k], dn, acc[k]);
    }
}

// ---- list ordering ----------------------------------------------------------------------------------------------
// In-place ascending sort of list[0..L) in GLOBAL memory by one CTA (only for lists longer than kSortCap):
// bitonic network in its "all comparators ascending" form, so that virtual +inf padding beyond L never moves.
__device__ void sort_global(uint32_t* a, uint32_t L)
{
    uint32_t P = 1;
    while (P < L) P <<= 1;
    for (uint32_t k = 2; k <= P; k <<= 1) {
        for (uint32_t j = k >> 1; j > 0; j >>= 1) {
            for (uint32_t t = threadIdx.x; t < (P >> 1); t += blockDim.x) {
                uint32_t lo, hi;
                if (j == (k >> 1)) {                       // first step of a merge: mirror inside the block of size k
                    const uint32_t blk = t / j, r = t % j;
                    lo = blk * k + r;
                    hi = blk * k + (k - 1 - r);
                } else {
                    lo = (t / j) * (2 * j) + (t % j);
                    hi = lo + j;
                }
                if (hi < L) {
                    const uint32_t x = a[lo], y = a[hi];
                    if (x > y) { a[lo] = y; a[hi] = x; }
                }
            }
            __threadfence_block();
            __syncthreads();
        }
    }
}

constexpr int kWarps = kComposeThreads / 32;

template <bool OPD, bool FIELD, bool RAMP>
__global__ void __launch_bounds__(kComposeThreads) k_compose_tile(const ComposeArgs a)
{
    __shared__ __align__(16) float4 s_rec[kChunk * 8];          // staged 128-byte records
    __shared__ uint32_t s_ids[kSortCap];                        // this tile's list, ascending
    __shared__ uint8_t s_surv[kWarps][kChunk];                  // per-warp survivors of the sub-tile cull

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int tpf = a.ntx * a.nty;
    const int tile = blockIdx.x;
    const int b = tile / tpf, rt = tile - b * tpf;
    const int ty = rt / a.ntx, tx = rt - ty * a.ntx;

    const bool overflow = (a.status->bits & OSOG_WOVERFLOW) != 0u;
    const uint32_t beg = a.offset[tile];
    const uint32_t L = overflow ? 0u : a.offset[tile + 1] - beg;
    uint32_t* glist = a.list + beg;

    // ---- H4 (second half): canonical order ------------------------------------------------------------------
    const bool in_smem = L <= (uint32_t)kSortCap;
    if (in_smem) {
        uint32_t* s_in = reinterpret_cast<uint32_t*>(s_rec);    // kChunk * 32 words >= kSortCap
        for (uint32_t k = tid; k < L; k += kComposeThreads) s_in[k] = glist[k];
        __syncthreads();
        for (uint32_t k = tid; k < L; k += kComposeThreads) {
            const uint32_t v = s_in[k];
            uint32_t r = 0;
            for (uint32_t m = 0; m < L; ++m) r += s_in[m] < v ? 1u : 0u;
            s_ids[r] = v;
            glist[r] = v;                                        // write the sorted segment back (osog_debug_bins)
        }
        __syncthreads();
    } else {
        sort_global(glist, L);
    }

    // ---- pixel ownership ----------------------------------------------------------------------------------------
    const int wx0 = tx * kTile + (wid & 1) * 16, wy0 = ty * kTile + (wid >> 1) * 8;   // warp sub-tile origin
    const int j = wx0 + (lane & 3) * 4, i = wy0 + (lane >> 2);
    const float jf = (float)j, fi = (float)i;
    const double jd = (double)j, id = (double)i;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};

    for (uint32_t c0 = 0; c0 < L; c0 += kChunk) {
        const int nC = (int)min((uint32_t)kChunk, L - c0);
        if (c0 > 0) __syncthreads();                             // everyone is done with the previous chunk
        for (int u = tid; u < nC * 8; u += kComposeThreads) {
            const uint32_t pid = in_smem ? s_ids[c0 + (u >> 3)] : glist[c0 + (u >> 3)];
            cp_async16(&s_rec[u], a.rec32 + (size_t)pid * kRecWords + (u & 7) * 4);
        }
        cp_async_wait_all();
        __syncthreads();
        // warp-level cull: keep the staged particles whose pixel bounding box meets this warp's 16 x 8 sub-tile
        int ns = 0;
        for (int base = 0; base < nC; base += 32) {
            const int k = base + lane;
            bool keep = false;
            if (k < nC) {
                const float4 h0 = s_rec[k * 8];
                const uint32_t bx = __float_as_uint(h0.z), by = __float_as_uint(h0.w);
                const int pj0 = bx & 0xffff, pj1 = bx >> 16, pi0 = by & 0xffff, pi1 = by >> 16;
                keep = pj0 <= wx0 + 15 && pj1 >= wx0 && pi0 <= wy0 + 7 && pi1 >= wy0;
            }
            const unsigned m = __ballot_sync(0xffffffffu, keep);
            if (keep) s_surv[wid][ns + __popc(m & ((1u << lane) - 1u))] = (uint8_t)k;
            ns += __popc(m);
        }
        __syncwarp();
        for (int s = 0; s < ns; ++s) {
            const float4* rec = &s_rec[(int)s_surv[wid][s] * 8];
            const uint32_t flags = __float_as_uint(rec[1].x);
            if (flags & kFlagPrism) eval_prism<4>(rec, a.rec64, jf, fi, acc);
            else eval_ellipsoid<4>(rec, jd, id, acc);
        }
    }

    // ---- H6/H7: write-out straight from the registers --------------------------------------------------------------
    if (i >= a.H || j >= a.W) return;
    const size_t row = ((size_t)b * a.H + i) * a.W;
    const bool vec = ((a.W & 3) == 0);                           // then j + 3 < W and the row base is 16-byte aligned
    if (OPD) {
        if (vec) {
            *reinterpret_cast<float4*>(a.opd + row + j) =
                overflow ? make_float4(0.f, 0.f, 0.f, 0.f)
                         : make_float4((float)acc[0], (float)acc[1], (float)acc[2], (float)acc[3]);
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (j + k < a.W) a.opd[row + j + k] = overflow ? 0.0f : (float)acc[k];
        }
    }
    if (FIELD) {
        const double inv_lambda = a.optics[b].inv_lambda;
        float2 u[4];
        float2 ry = make_float2(1.0f, 0.0f);
        if (RAMP && a.ramp_y_on) ry = a.ramp_y[(size_t)b * a.H + i];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            double turns = acc[k] * inv_lambda;                  // Eq. 2: phase = 2 pi OPD / lambda, kept in turns
            turns -= rint(turns);
            float s, c;
            sincospif(2.0f * (float)turns, &s, &c);
            if (RAMP && j + k < a.W) {
                float2 r = a.ramp_x[(size_t)b * a.W + j + k];
                if (a.ramp_y_on) r = make_float2(r.x * ry.x - r.y * ry.y, r.x * ry.y + r.y * ry.x);
                const float c2 = c * r.x - s * r.y, s2 = c * r.y + s * r.x;
                c = c2; s = s2;
            }
            u[k] = overflow ? make_float2(0.f, 0.f) : make_float2(c, s);
        }
        float2* out = a.field + row + j;
        if (vec) {
            reinterpret_cast<float4*>(out)[0] = make_float4(u[0].x, u[0].y, u[1].x, u[1].y);
            reinterpret_cast<float4*>(out)[1] = make_float4(u[2].x, u[2].y, u[3].x, u[3].y);
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (j + k < a.W) out[k] = u[k];
        }
    }
}

cudaError_t launch_compose(osog_ctx* c, long long N, int B, bool has_ramp, float* d_opd, float2* d_field)
{
    (void)N;
    ComposeArgs a;
    a.rec32 = c->rec32; a.rec64 = c->rec64; a.offset = c->offset; a.list = c->list; a.optics = c->optics;
    a.ramp_x = c->ramp_x; a.ramp_y = c->ramp_y; a.status = c->status;
    a.opd = d_opd; a.field = d_field;
    a.H = c->H; a.W = c->W; a.ntx = c->ntx; a.nty = c->nty;
    a.ramp_y_on = 1;
    const unsigned grid = (unsigned)((long long)B * c->ntx * c->nty);
    const dim3 blk(kComposeThreads);
    if (d_opd != nullptr && d_field == nullptr) k_compose_tile<true, false, false><<<grid, blk, 0, c->stream>>>(a);
    else if (d_opd == nullptr && !has_ramp) k_compose_tile<false, true, false><<<grid, blk, 0, c->stream>>>(a);
    else if (d_opd == nullptr && has_ramp) k_compose_tile<false, true, true><<<grid, blk, 0, c->stream>>>(a);
    else if (!has_ramp) k_compose_tile<true, true, false><<<grid, blk, 0, c->stream>>>(a);
    else k_compose_tile<true, true, true><<<grid, blk, 0, c->stream>>>(a);
    return cudaGetLastError();
}

// ---- measured alternative: paper-style scatter-add with global atomics ------------------------
// One warp per particle walks the particle's pixel bounding box and atomicAdd's (n_p - n_m) t into the frame.
// Summation order, hence the last bits, depend on scheduling: NOT deterministic.  The frame must be zeroed first.
__global__ void __launch_bounds__(256) k_compose_atomic(const float* __restrict__ rec32, const double* __restrict__ rec64,
                                                        const int4* __restrict__ tbox, const int* __restrict__ pframe,
                                                        long long N, int H, int W, float* __restrict__ opd)
{
    const long long n = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (n >= N) return;
    if (tbox[n].x > tbox[n].y) return;
    const float4* rec = reinterpret_cast<const float4*>(rec32 + (size_t)n * kRecWords);
    const float4 h0 = rec[0];
    const uint32_t bx = __float_as_uint(h0.z), by = __float_as_uint(h0.w);
    const int j0 = bx & 0xffff, j1 = bx >> 16, i0 = by & 0xffff, i1 = by >> 16;
    const uint32_t flags = __float_as_uint(rec[1].x);
    const int bw = j1 - j0 + 1, np = bw * (i1 - i0 + 1);
    float* frame = opd + (size_t)pframe[n] * H * W;
    for (int q = lane; q < np; q += 32) {
        const int i = i0 + q / bw, j = j0 + q % bw;
        double acc[1] = {0.0};
        if (flags & kFlagPrism) {
            eval_prism<1>(rec, rec64, (float)j, (float)i, acc);
        } else {
            eval_ellipsoid<1>(rec, (double)j, (double)i, acc);
        }
        const float v = (float)acc[0];
        if (v != 0.0f) atomicAdd(&frame[(size_t)i * W + j], v);
    }
}

cudaError_t launch_compose_atomic(osog_ctx* c, long long N, int B, float* d_opd)
{
    cudaError_t e = cudaMemsetAsync(d_opd, 0, sizeof(float) * (size_t)B * c->H * c->W, c->stream);
    if (e != cudaSuccess || N == 0) return e;
    const long long threads = N * 32;
    k_compose_atomic<<<(unsigned)((threads + 255) / 256), 256, 0, c->stream>>>(c->rec32, c->rec64, c->tbox, c->pframe, N,
                                                                              c->H, c->W, d_opd);
    return cudaGetLastError();
}

}  // namespace osog
