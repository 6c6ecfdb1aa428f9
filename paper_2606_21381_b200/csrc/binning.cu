// H1-H4 of DESIGN.md: per-particle preparation (fp64), bounding box -> tile range -> count (H2), exclusive scan of the
// per-tile counts (H3, warp shuffles, by the last binning block to finish), and the first half of the fill (H4): the
// atomic that counts a (particle, tile) pair also returns its slot in the tile's staging slice.  k_sort_cull
// (compose.cu) then moves every tile's entries, in ascending particle index, to offset[tile] of the compact CSR list.
// Integer results must equal the oracle's binning bit for bit (B1-B4).
#include "osog_internal.cuh"

namespace osog {

struct PrepArgs {
    const float *cx, *cy, *cz, *qw, *qx, *qy, *qz, *d0, *d1, *d2, *n_p;   // cz may be nullptr (all zero)
    const uint8_t* kind;
    const int32_t* frame_start;   // device [B+1] or nullptr
    long long N;
    int B, H, W, ntx, nty;
    double pitch, n_medium;
    float* rec;
    float* rec2;
    int4* tbox;
    int* pframe;
    uint32_t* count;              // this call's slot of the per-tile counters (all zero on entry)
    uint32_t* slices;             // [tiles][slice_cap] staging slices (unsorted; entries beyond slice_cap are not stored)
    int slice_cap;
    uint32_t* offset;             // [tiles + 1] exclusive scan of count (H3), written by the last binning block
    uint32_t* done;               // number of binning blocks that have finished (0 on entry, reset by the last one)
    long long max_pairs;          // capacity of the CSR list: a larger total sets OSOG_WOVERFLOW
    float* obb;                   // [N][6] oriented-bounding-box labels (osog_particle_obbs), or nullptr
    int unit_dn;                  // 1: index contrast n_p - n_medium replaced by 1 (height map of the G-buffer)
    FrameOptics* optics;
    DeviceStatus* status;
    OpticsChunk oc;               // frames 0 .. min(B, kOpticsChunk)-1 by value
};

__device__ __forceinline__ bool finite_f(float v) { return fabsf(v) <= 3.402823466e38f; }   // false for NaN / inf

constexpr int kPrepThreads = 128;

// ---- binning role of k_prepare (H2 + H4): one particle per thread, list appends balanced over the warp -------------------
// B1-B2 (fp64): half extents of the projection, inclusive pixel range padded by 2^-10 px, clamped to the frame; B3: tile
// range.  H4: the (particle, tile) pairs of the warp's 32 particles are dealt out evenly to its lanes (prefix sum of the
// tile counts + a binary search in shared memory), so that every lane has about the same number of list appends and
// all of them are in flight at once: the atomic on the tile's counter returns the slot of the tile's slice.
__device__ __forceinline__ void binning_role(const PrepArgs& a, long long n)
{
    __shared__ int s_pre[kPrepThreads / 32][33];
    __shared__ int4 s_box[kPrepThreads / 32][32];      // tx0, tile columns, ty0, particle index
    __shared__ uint32_t s_t0[kPrepThreads / 32][32];   // first tile of the particle's frame
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int4 tb = make_int4(1, 0, 1, 0);                 // empty tile range
    int b = 0;
    if (n < a.N) {
        const float fcx = a.cx[n], fcy = a.cy[n], fqw = a.qw[n], fqx = a.qx[n], fqy = a.qy[n], fqz = a.qz[n];
        const float fd0 = a.d0[n], fd1 = a.d1[n], fd2 = a.d2[n], fnp = a.n_p[n];
        const unsigned kind = a.kind[n];
        const bool valid = finite_f(fcx) && finite_f(fcy) && finite_f(fqw) && finite_f(fqx) && finite_f(fqy) && finite_f(fqz) &&
                           finite_f(fd0) && finite_f(fd1) && finite_f(fd2) && finite_f(fnp) &&
                           fd0 > 0.0f && fd1 > 0.0f && fd2 > 0.0f && kind <= 1u;
        if (a.frame_start != nullptr) {              // largest b with frame_start[b] <= n
            int lo = 0, hi = a.B;
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if ((long long)a.frame_start[mid] <= n) lo = mid; else hi = mid;
            }
            b = lo;
        }
        a.pframe[n] = b;
        if (!valid) {
            atomicOr(&a.status->bits, OSOG_WBADPARTICLE);
        } else {
            const double p = a.pitch;
            const double cx = fcx, cy = fcy;
            const double w = fqw, x = fqx, y = fqy, z = fqz;
            // rows x and y of the Hamilton active rotation body -> world, no renormalisation (reading A4)
            const double R00 = 1.0 - 2.0 * (y * y + z * z), R01 = 2.0 * (x * y - w * z), R02 = 2.0 * (x * z + w * y);
            const double R10 = 2.0 * (x * y + w * z), R11 = 1.0 - 2.0 * (x * x + z * z), R12 = 2.0 * (y * z - w * x);
            const double e0 = fd0, e1 = fd1, e2 = fd2;
            // B1: half extents of the projection
            double hx, hy;
            if (kind == 0u) {
                hx = sqrt(R00 * R00 * e0 * e0 + R01 * R01 * e1 * e1 + R02 * R02 * e2 * e2);
                hy = sqrt(R10 * R10 * e0 * e0 + R11 * R11 * e1 * e1 + R12 * R12 * e2 * e2);
            } else {
                const double hs = 0.5 * e0, hl = 0.5 * e1, ap = 0.5 * e1 + e2;
                hx = fabs(R02 * ap);
                hy = fabs(R12 * ap);
#pragma unroll
                for (int v = 0; v < 4; ++v) {        // (+-s/2, +-s/2, +L/2); the -L/2 half mirrors it through the centre
                    const double sx = (v & 1) ? -hs : hs, sy = (v & 2) ? -hs : hs;
                    hx = fmax(hx, fabs(R00 * sx + R01 * sy + R02 * hl));
                    hy = fmax(hy, fabs(R10 * sx + R11 * sy + R12 * hl));
                }
            }
            // B2: inclusive pixel range, padded by 2^-10 px, clamped to the frame
            const double fj0 = ceil((cx - hx) / p - 0.5 - kBBoxPadPx), fj1 = floor((cx + hx) / p - 0.5 + kBBoxPadPx);
            const double fi0 = ceil((cy - hy) / p - 0.5 - kBBoxPadPx), fi1 = floor((cy + hy) / p - 0.5 + kBBoxPadPx);
            const double big = 1073741824.0;
            if (fabs(fj0) <= 1.7976931348623157e308 && fabs(fj1) <= 1.7976931348623157e308 &&
                fabs(fi0) <= 1.7976931348623157e308 && fabs(fi1) <= 1.7976931348623157e308) {   // else: not listed (as the oracle)
                const int j0 = max(0, min(a.W, (int)fmin(fmax(fj0, -big), big)));
                const int j1 = max(-1, min(a.W - 1, (int)fmin(fmax(fj1, -big), big)));
                const int i0 = max(0, min(a.H, (int)fmin(fmax(fi0, -big), big)));
                const int i1 = max(-1, min(a.H - 1, (int)fmin(fmax(fi1, -big), big)));
                if (j0 <= j1 && i0 <= i1) {
                    tb = make_int4(j0 / kTile, j1 / kTile, i0 / kTile, i1 / kTile);      // B3
                    // words 0, 1, 6, 7 of the record: centre in pixel-index coordinates and the packed pixel bounding box
                    float* r32 = a.rec + (size_t)n * kRecWords;
                    uint32_t* r32u = reinterpret_cast<uint32_t*>(r32);
                    const double ip = 1.0 / p;
                    r32[0] = (float)(cx * ip - 0.5);
                    r32[1] = (float)(cy * ip - 0.5);
                    r32u[6] = (uint32_t)j0 | ((uint32_t)j1 << 16);
                    r32u[7] = (uint32_t)i0 | ((uint32_t)i1 << 16);
                }
            }
        }
        a.tbox[n] = tb;
    }
    // ---- H4: deal the warp's (particle, tile) pairs out to its lanes
    const int tw = tb.y - tb.x + 1;
    const int nt = tb.x > tb.y ? 0 : tw * (tb.w - tb.z + 1);
    int incl = nt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += v;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    s_pre[wid][lane] = incl - nt;
    if (lane == 31) s_pre[wid][32] = total;
    s_box[wid][lane] = make_int4(tb.x, tw, tb.z, (int)(uint32_t)n);
    s_t0[wid][lane] = (uint32_t)((size_t)b * a.ntx * a.nty);
    __syncwarp();
    const uint32_t cap = (uint32_t)a.slice_cap;
    for (int k0 = 0; k0 < total; k0 += 32 * 8) {
        uint32_t t[8], pos[8], id[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int k = k0 + q * 32 + lane;
            if (k < total) {
                int s = 0;                                       // largest s with pre[s] <= k (lanes without tiles share the
#pragma unroll                                                   // prefix of their successor and are never picked)
                for (int step = 16; step > 0; step >>= 1)
                    if (s_pre[wid][s + step] <= k) s += step;
                const int4 bx = s_box[wid][s];
                const int local = k - s_pre[wid][s];
                const int dy = local / bx.y, dx = local - dy * bx.y;
                t[q] = s_t0[wid][s] + (uint32_t)((bx.z + dy) * a.ntx + bx.x + dx);
                id[q] = (uint32_t)bx.w;
                pos[q] = atomicAdd(&a.count[t[q]], 1u);
            }
        }
#pragma unroll
        for (int q = 0; q < 8; ++q)
            if (k0 + q * 32 + lane < total && pos[q] < cap) a.slices[(size_t)t[q] * cap + pos[q]] = id[q];
    }
}

// ---- H3: exclusive scan of the per-tile counts, by ONE block (the last binning block to finish) ------------------------
// Every thread sums a contiguous chunk of tiles (independent 128-bit loads, all in flight), the chunk sums are scanned
// across the block with warp shuffles (inclusive shuffle scan per warp, the warp totals through shared memory), then
// every thread walks its chunk again and writes offset[t].  Also: total pair count, longest list, capacity check.
__device__ void scan_counts(const PrepArgs& a)
{
    __shared__ unsigned long long s_warp[kPrepThreads / 32];
    __shared__ uint32_t s_max[kPrepThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long long tiles = (long long)a.B * a.ntx * a.nty;
    long long chunk = (tiles + kPrepThreads - 1) / kPrepThreads;
    chunk = (chunk + 3) & ~3ll;                                   // multiple of 4: the 128-bit loads stay aligned
    const long long t0 = min(tiles, (long long)threadIdx.x * chunk), t1 = min(tiles, t0 + chunk);
    const uint32_t* cnt = a.count;
    unsigned long long sum = 0;
    uint32_t mx = 0;
    long long t = t0;
    for (; t + 4 <= t1; t += 4) {                                 // L2 reads: the counters were written by atomics
        const uint4 v = __ldcg(reinterpret_cast<const uint4*>(cnt + t));
        sum += (unsigned long long)v.x + v.y + v.z + v.w;
        mx = max(max(mx, v.x), max(v.y, max(v.z, v.w)));
    }
    for (; t < t1; ++t) { const uint32_t v = __ldcg(cnt + t); sum += v; mx = max(mx, v); }
    // block-wide exclusive scan of the chunk sums
    unsigned long long incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned long long v = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += v;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, d));
    if (lane == 31) s_warp[wid] = incl;
    if (lane == 0) s_max[wid] = mx;
    __syncthreads();
    unsigned long long base = 0, total = 0;
    uint32_t mall = 0;
#pragma unroll
    for (int w = 0; w < kPrepThreads / 32; ++w) {
        if (w < wid) base += s_warp[w];
        total += s_warp[w];
        mall = max(mall, s_max[w]);
    }
    unsigned long long run = base + incl - sum;                   // exclusive prefix of this thread's chunk
    for (t = t0; t + 4 <= t1; t += 4) {
        const uint4 v = __ldcg(reinterpret_cast<const uint4*>(cnt + t));
        uint4 o;
        o.x = (uint32_t)min(run, 0xffffffffull); run += v.x;
        o.y = (uint32_t)min(run, 0xffffffffull); run += v.y;
        o.z = (uint32_t)min(run, 0xffffffffull); run += v.z;
        o.w = (uint32_t)min(run, 0xffffffffull); run += v.w;
        *reinterpret_cast<uint4*>(a.offset + t) = o;
    }
    for (; t < t1; ++t) { a.offset[t] = (uint32_t)min(run, 0xffffffffull); run += __ldcg(cnt + t); }
    if (threadIdx.x == 0) {
        a.offset[tiles] = (uint32_t)min(total, 0xffffffffull);
        a.status->pairs = total;
        a.status->max_count = mall;
        if (total > (unsigned long long)a.max_pairs) atomicOr(&a.status->bits, OSOG_WOVERFLOW);
        *a.done = 0u;                                             // ready for the next call
    }
}

// ---- record role of k_prepare (H1): EIGHT lanes per particle ------------------------------------------------------------
// The derived record of a prism is a long fp64 dependency chain (rotation, 6 slab normals, slope ranking, a division and
// an exact-grid split per slab, the oriented box): one thread per particle made k_prepare the latency-bound head of the
// whole step.  Here the 8 lanes of a group all form the short common part (rotation, normals, slopes) and then split the
// rest: lanes 0..5 one slab each (rank, coefficients, (hi, lo) pairs), lane 6 the oriented box and the header, lane 7 the
// reference pixel / height bound / chord scale.  An ellipsoid uses lanes 0 (quadratic), 1 (oriented box), 7.
__device__ __forceinline__ void record_role(const PrepArgs& a, long long n, int l8, unsigned gmask)
{
    if (n >= a.N) return;
    const float fcx = a.cx[n], fcy = a.cy[n], fqw = a.qw[n], fqx = a.qx[n], fqy = a.qy[n], fqz = a.qz[n];
    const float fd0 = a.d0[n], fd1 = a.d1[n], fd2 = a.d2[n], fnp = a.n_p[n];
    const unsigned kind = a.kind[n];
    const bool valid = finite_f(fcx) && finite_f(fcy) && finite_f(fqw) && finite_f(fqx) && finite_f(fqy) && finite_f(fqz) &&
                 finite_f(fd0) && finite_f(fd1) && finite_f(fd2) && finite_f(fnp) &&
                 fd0 > 0.0f && fd1 > 0.0f && fd2 > 0.0f && kind <= 1u;
    if (!valid) {                                // flagged by the binning role
        if (a.obb != nullptr && l8 < 6) a.obb[(size_t)n * 6 + l8] = __int_as_float(0x7fc00000);
        return;
    }
    const double p = a.pitch;
    const double cx = fcx, cy = fcy;
    const double w = fqw, x = fqx, y = fqy, z = fqz;
    // Hamilton active rotation body -> world, no renormalisation (reading A4)
    const double R00 = 1.0 - 2.0 * (y * y + z * z), R01 = 2.0 * (x * y - w * z), R02 = 2.0 * (x * z + w * y);
    const double R10 = 2.0 * (x * y + w * z), R11 = 1.0 - 2.0 * (x * x + z * z), R12 = 2.0 * (y * z - w * x);
    const double R20 = 2.0 * (x * z - w * y), R21 = 2.0 * (y * z + w * x), R22 = 1.0 - 2.0 * (x * x + y * y);
    const double e0 = fd0, e1 = fd1, e2 = fd2;

    float* r32 = a.rec + (size_t)n * kRecWords;
    uint32_t* r32u = reinterpret_cast<uint32_t*>(r32);
    const double ip = 1.0 / p;
    // Coordinates are pixel offsets from pixel (jc, ic): dx = p dj + ox
    const double jc = fmin(fmax(floor(cx * ip), -1.0e6), 1.0e6);      // reference pixel: any nearby pixel will do
    const double ic = fmin(fmax(floor(cy * ip), -1.0e6), 1.0e6);
    const double ox = (jc + 0.5) * p - cx, oy = (ic + 0.5) * p - cy;
    const double dn = a.unit_dn ? 1.0 : (double)fnp - a.n_medium;
    double* r64 = reinterpret_cast<double*>(r32 + 16);
    // upper bound of the chord's top relative to the centre (word 14; G-buffer: a particle whose cz + bound lies below every
    // top already found in a sub-tile is skipped; padded for the not-quite-orthogonal R of reading A4), and the chord scale
    // (word 15): the power of two s with s * chord <= 1/2 for every chord of the body (chord <= 2 zmax): the composition
    // evaluates s * t with a saturating subtraction (clamp to [0, 1] for free) and folds 1 / s into the index contrast
    double zmax;
    if (kind == 0u) {
        zmax = sqrt(R20 * R20 * e0 * e0 + R21 * R21 * e1 * e1 + R22 * R22 * e2 * e2);
    } else {
        const double hs = 0.5 * e0, hl = 0.5 * e1;
        zmax = fabs(R22) * (hl + e2);
        zmax = fmax(zmax, fabs(R20) * hs + fabs(R21) * hs + fabs(R22) * hl);
    }
    int ex2 = ((__double2hiint(2.0 * zmax * (1.0 + 1.0e-5) + 2.0e-6) >> 20) & 0x7ff) - 1022;     // 2 zmax < 2^ex2
    ex2 = min(max(ex2 + 1, -60), 60);
    const float tscf = __int_as_float((127 - ex2) << 23);
    if (l8 == 7) {
        r32u[11] = (uint32_t)n;
        reinterpret_cast<int*>(r32)[12] = (int)jc;
        reinterpret_cast<int*>(r32)[13] = (int)ic;
        r32[14] = __double2float_ru(zmax * (1.0 + 1.0e-5) + 1.0e-6);
        r32[15] = tscf;
    }
    // Words 2..5: oriented box of the silhouette (unit axis with a_x >= 0, half lengths > 0); their sign bits carry the
    // evaluation code of the particle (0 ellipsoid, 1 + number of steep slabs, 4 all-fp64): bit 0 in the sign of
    // the first half length, bit 1 in the second, bit 2 in the sign of a_x.
    const double cull_pad = 1.0 / 64.0;          // px; covers the fp32 rounding of the cull test

    if (kind == 0u) {
        if (l8 > 1) return;
        // M = R diag(1/a^2, 1/b^2, 1/c^2) R^T; chord of {q^T M q <= 1} along z at (dx, dy):
        // t = T0 sqrt(1 - d^T S d), S = Schur complement of M_zz, T0 = 2 / sqrt(M_zz)   (H5)
        const double i0s = 1.0 / (e0 * e0), i1s = 1.0 / (e1 * e1), i2s = 1.0 / (e2 * e2);
        const double Mxx = R00 * i0s * R00 + R01 * i1s * R01 + R02 * i2s * R02;
        const double Mxy = R00 * i0s * R10 + R01 * i1s * R11 + R02 * i2s * R12;
        const double Mxz = R00 * i0s * R20 + R01 * i1s * R21 + R02 * i2s * R22;
        const double Myy = R10 * i0s * R10 + R11 * i1s * R11 + R12 * i2s * R12;
        const double Myz = R10 * i0s * R20 + R11 * i1s * R21 + R12 * i2s * R22;
        const double Mzz = R20 * i0s * R20 + R21 * i1s * R21 + R22 * i2s * R22;
        const double iMzz = 1.0 / Mzz;
        const double Sxx = Mxx - Mxz * Mxz * iMzz, Sxy = Mxy - Mxz * Myz * iMzz, Syy = Myy - Myz * Myz * iMzz;
        if (l8 == 0) {
            const double T0 = 2.0 * rsqrt(Mzz);
            // w(dj, di) = F1 - (A dj^2 + B dj di + C di^2 + D dj + E di)
            const double cA = Sxx * p * p, cB = 2.0 * Sxy * p * p, cC = Syy * p * p;
            const double cD = 2.0 * p * (Sxx * ox + Sxy * oy), cE = 2.0 * p * (Sxy * ox + Syy * oy);
            const double cF = 1.0 - (Sxx * ox * ox + 2.0 * Sxy * ox * oy + Syy * oy * oy);
            r64[0] = cA; r64[1] = cB; r64[2] = cC; r64[3] = cD; r64[4] = cE; r64[5] = cF;
            r64[6] = jc;
            r64[7] = ic;
            // Words 40..53: the same quadratic for the composition kernel as (hi, lo) float pairs on an exact grid: hi is a
            // multiple of q = 2^(e - 22) where 2^e bounds every intermediate of the Horner evaluation over the pixels the
            // kernel can ask for (|dj| <= Rj, |di| <= Ri), so the fp32 FMAs on the hi parts are exact (integers times q below
            // 2^24 q); lo = the remainder, fp32.  Signs arranged for w = F + (E + Cn ndi) ndi + (D + Bn ndi + An ndj) ndj with
            // ndj = -(j - jc), ndi = -(i - ic): An = -A, Bn = -B, Cn = -C.
            const double det = Sxx * Syy - Sxy * Sxy;
            const double Rj = sqrt(fmax(Syy / det, 0.0)) * ip + 20.0, Ri = sqrt(fmax(Sxx / det, 0.0)) * ip + 20.0;
            double Mb = 1.0 + fabs(cF) + (fabs(cC) * Ri + fabs(cE)) * Ri + (fabs(cA) * Rj + fabs(cB) * Ri + fabs(cD)) * Rj;
            if (!(Mb < 1.0e30)) Mb = 1.0e30;                   // degenerate shape: the grid is coarse, the result stays finite
            const int eb = ((__double2hiint(Mb) >> 20) & 0x7ff) - 1022;                     // Mb < 2^eb
            const double cq = __hiloint2double(((eb - 22 + 52 + 1023) << 20) | 0x80000, 0);  // 1.5 * 2^52 * q, q = 2^(eb - 22)
            const double v[6] = {-cA, -cB, -cC, cD, cE, cF};
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                const double hi = (v[k] + cq) - cq;
                r32[40 + 2 * k] = (float)hi;
                r32[41 + 2 * k] = (float)(v[k] - hi);
            }
            r32[52] = (float)jc;
            r32[53] = (float)ic;
            r32u[8] = 0u;
            r32[9] = (float)(dn * T0);
            // chord midpoint z = -(M_xz dx + M_yz dy) / M_zz as Z0 + Zx dj + Zy di, and T0 (G-buffer only)
            r64[8] = -(Mxz * ox + Myz * oy) * iMzz;
            r64[9] = -Mxz * p * iMzz;
            r64[10] = -Myz * p * iMzz;
            r64[11] = T0;
            return;
        }
        // lane 1: oriented box of the silhouette ellipse {d^T S d <= 1}: principal axes of S
        const double hd = 0.5 * (Sxx - Syy), rad = sqrt(hd * hd + Sxy * Sxy), mid = 0.5 * (Sxx + Syy);
        const double lmin = fmax(mid - rad, 1.0e-300), lmax = mid + rad;
        double vx = Sxy, vy = lmin - Sxx;        // eigenvector of the small eigenvalue = long axis
        if (fabs(lmin - Syy) > fabs(vy)) { vx = lmin - Syy; vy = Sxy; }
        const double vn2 = vx * vx + vy * vy;
        double ivn = rsqrt(vn2);
        if (!(vn2 > 1.0e-280)) { vx = 1.0; vy = 0.0; ivn = 1.0; }
        if (vx < 0.0) { vx = -vx; vy = -vy; }
        r32[2] = fabsf((float)(vx * ivn));
        r32[3] = (float)(vy * ivn);
        r32[4] = (float)(rsqrt(lmin) * ip * (1.0 + 1.0e-5) + cull_pad);
        r32[5] = (float)(rsqrt(lmax) * ip * (1.0 + 1.0e-5) + cull_pad);
        r32[10] = a.cz != nullptr ? a.cz[n] : 0.0f;          // centre height (G-buffer depth map only)
        if (a.obb != nullptr) {                  // label (reading A23): principal-axis box of the silhouette ellipse, no padding
            float* ob = a.obb + (size_t)n * 6;
            ob[0] = (float)(cx * ip - 0.5); ob[1] = (float)(cy * ip - 0.5);
            ob[2] = (float)(vx * ivn); ob[3] = (float)(vy * ivn);
            ob[4] = (float)(rsqrt(lmin) * ip); ob[5] = (float)(rsqrt(lmax) * ip);
        }
        return;
    }

    // ---- capped tetragonal prism: 12 half-spaces = 6 centrally symmetric slabs  |n_k . x| <= b_k  (Eq. 1) ----
    // Everything below is fully unrolled with constant indices (registers, no local memory); slabs are written to the
    // record in order of decreasing slope |n_xy| / |n_z| (rank by cross-multiplied comparisons, no division).
    const double s = e0, L = e1, hc = e2;
    const double hs2 = 0.5 * s;
    const double bcap = hc * s * 0.5 + s * L * 0.25;
    double nx[6], ny[6], nz[6], h2[6], z2[6];
    // body normals (1,0,0), (0,1,0), (hc,0,s/2), (hc,0,-s/2), (0,hc,s/2), (0,hc,-s/2) rotated to the world frame
    nx[0] = R00; ny[0] = R10; nz[0] = R20;
    nx[1] = R01; ny[1] = R11; nz[1] = R21;
    nx[2] = R00 * hc + R02 * hs2; ny[2] = R10 * hc + R12 * hs2; nz[2] = R20 * hc + R22 * hs2;
    nx[3] = R00 * hc - R02 * hs2; ny[3] = R10 * hc - R12 * hs2; nz[3] = R20 * hc - R22 * hs2;
    nx[4] = R01 * hc + R02 * hs2; ny[4] = R11 * hc + R12 * hs2; nz[4] = R21 * hc + R22 * hs2;
    nx[5] = R01 * hc - R02 * hs2; ny[5] = R11 * hc - R12 * hs2; nz[5] = R21 * hc - R22 * hs2;
    const double g0sq = (double)kSteepSlope * (double)kSteepSlope, gasq = kAllF64Slope * kAllF64Slope;
    int ns = 0;
    bool allf64 = false;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        h2[k] = nx[k] * nx[k] + ny[k] * ny[k];
        z2[k] = nz[k] * nz[k];
        ns += (nz[k] == 0.0 || h2[k] > g0sq * z2[k]) ? 1 : 0;
        allf64 = allf64 || nz[k] == 0.0 || h2[k] > gasq * z2[k];
    }
    if (ns > 2) allf64 = true;                   // more than two steep slabs: rare, every pixel goes to fp64
    uint32_t vbit = 0u;
    if (l8 < 6) {
        // this lane's slab k = l8 (selected with constant indices: the arrays stay in registers)
        double nxk = nx[0], nyk = ny[0], nzk = nz[0], h2k = h2[0], z2k = z2[0];
#pragma unroll
        for (int k = 1; k < 6; ++k)
            if (k == l8) { nxk = nx[k]; nyk = ny[k]; nzk = nz[k]; h2k = h2[k]; z2k = z2[k]; }
        int q = 0;                                   // rank of the slab: number of slabs steeper than it (ties: lower index first)
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            const double lhs = h2[j] * z2k, rhs = h2k * z2[j];      // slope_j > slope_k  <=>  lhs > rhs
            q += (j != l8 && (lhs > rhs || (lhs == rhs && j < l8))) ? 1 : 0;
        }
        const double bk = l8 < 2 ? hs2 : bcap;
        double o0, o1, o2, o3;
        if (nzk == 0.0) {
            // vertical face pair: no z bound; the line is inside the slab iff |n_x dx + n_y dy| <= b
            o0 = nxk * p; o1 = nyk * p; o2 = nxk * ox + nyk * oy; o3 = bk;
            vbit = 1u << (16 + q);
        } else {
            const double r = (nzk > 0.0 ? 1.0 : -1.0) / fabs(nzk);  // sigma / |n_z|
            const double W0 = r * (nxk * ox + nyk * oy), Cb = bk * fabs(r);
            o0 = r * nxk * p;                         // U:  exit_k = Cx - U dj - V di
            o1 = r * nyk * p;                         // V:  enter_k = Cn - U dj - V di
            o2 = Cb - W0;                             // Cx
            o3 = -Cb - W0;                            // Cn
        }
        double2* o4 = reinterpret_cast<double2*>(r64 + 4 * q);
        o4[0] = make_double2(o0, o1);
        o4[1] = make_double2(o2, o3);
        // The slab once more for the composition kernel, scaled by the chord scale s (word 15) and split into (hi, lo)
        // float pairs on an exact grid: hi = multiple of q_k = 2^(e_k - 22) with 2^e_k above every intermediate of
        // C - U oj - V oi for all sub-tile origins (oj, oi) the kernel can ask for (|oj| + |oi| <= the body's diameter in
        // pixels + 64), so the kernel's fp32 FMAs on the hi parts are exact and hi + lo reproduces the fp64 re-basing to
        // ~2^-47 of that bound.  Layout per slab: (U_h, V_h, Cx_h, Cn_h), (U_l, V_l, Cx_l, Cn_l).
        const double reach = (1.5 * s + L + 2.0 * hc) * ip + 64.0;
        double mb = fmax(fabs(o2), fabs(o3)) + reach * (fabs(o0) + fabs(o1));
        if (!(mb < 1.0e30)) mb = 1.0e30;
        const int eb = ((__double2hiint(mb) >> 20) & 0x7ff) - 1022;                      // mb < 2^eb
        const double cq = __hiloint2double(((eb - 22 + 52 + 1023) << 20) | 0x80000, 0);   // 1.5 * 2^52 * q, q = 2^(eb - 22)
        const double h0 = (o0 + cq) - cq, h1 = (o1 + cq) - cq, h2s = (o2 + cq) - cq, h3s = (o3 + cq) - cq;
        float4* pw = reinterpret_cast<float4*>(a.rec2 + (size_t)n * kPairWords) + 2 * q;
        pw[0] = make_float4((float)h0 * tscf, (float)h1 * tscf, (float)h2s * tscf, (float)h3s * tscf);
        pw[1] = make_float4((float)(o0 - h0) * tscf, (float)(o1 - h1) * tscf, (float)(o2 - h2s) * tscf, (float)(o3 - h3s) * tscf);
    }
    // which ranks hold a vertical slab: OR over the group's lanes
#pragma unroll
    for (int d = 1; d < 8; d <<= 1) vbit |= __shfl_xor_sync(gmask, vbit, d);
    if (l8 != 6) return;
    uint32_t flags = kFlagPrism | vbit | ((uint32_t)ns << 8);
    if (allf64) flags |= kFlagAllF64;
    // oriented box of the silhouette: along the projected long axis (body z) and across it, over the 10 vertices
    double ax = R02, ay = R12;
    const double an = sqrt(ax * ax + ay * ay);
    if (an > 1.0e-12) { ax /= an; ay /= an; } else { ax = 1.0; ay = 0.0; }
    const double hs = hs2, hl = 0.5 * L, ap = 0.5 * L + hc;
    double ha = fabs((R02 * ax + R12 * ay) * ap), hb = fabs((-R02 * ay + R12 * ax) * ap);
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        const double sx = (v & 1) ? -hs : hs, sy = (v & 2) ? -hs : hs;
        const double px = R00 * sx + R01 * sy + R02 * hl, py = R10 * sx + R11 * sy + R12 * hl;
        ha = fmax(ha, fabs(px * ax + py * ay));
        hb = fmax(hb, fabs(-px * ay + py * ax));
    }
    if (ax < 0.0) { ax = -ax; ay = -ay; }
    const uint32_t code = allf64 ? 4u : 1u + (uint32_t)ns;
    r32u[2] = (__float_as_uint((float)ax) & 0x7fffffffu) | ((code >> 2) << 31);
    r32[3] = (float)ay;
    r32u[4] = __float_as_uint((float)(ha * ip * (1.0 + 1.0e-5) + cull_pad)) | ((code & 1u) << 31);
    r32u[5] = __float_as_uint((float)(hb * ip * (1.0 + 1.0e-5) + cull_pad)) | (((code >> 1) & 1u) << 31);
    r32u[8] = flags;
    r32[9] = (float)dn;
    r32[10] = a.cz != nullptr ? a.cz[n] : 0.0f;              // centre height (G-buffer depth map only)
    if (a.obb != nullptr) {                      // label (reading A23): box along the projected long axis, no padding
        float* ob = a.obb + (size_t)n * 6;
        ob[0] = (float)(cx * ip - 0.5); ob[1] = (float)(cy * ip - 0.5);
        ob[2] = (float)ax; ob[3] = (float)ay;
        ob[4] = (float)(ha * ip); ob[5] = (float)(hb * ip);
    }
}

constexpr int kRecPerBlock = kPrepThreads / 8;     // particles per record-role block

// Grid layout (blocks of 128 threads): [0, nbin) binning role, one particle per thread (nbin = max(1, ceil(N / 128)): the
// scan needs a block even when N = 0); [nbin, nbin + nrec) record role, 16 particles per block, 8 lanes each, the block's
// particles permuted so that prisms come first (its warps are then uniform in the code path they take, except one mixed
// warp per block).  nrec = ceil(N / 16).
__global__ void __launch_bounds__(kPrepThreads, 6) k_prepare(const PrepArgs a)
{
    pdl_trigger();                               // k_sort_cull's CTAs may become resident (they wait for this grid to finish)
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long nb = (a.N + kPrepThreads - 1) / kPrepThreads;
    const long long nbin = nb > 0 ? nb : 1;
    const long long nrec = (a.N + kRecPerBlock - 1) / kRecPerBlock;

    if (gid < a.B && gid < kOpticsChunk) a.optics[gid] = a.oc.f[gid];

    if ((long long)blockIdx.x >= nbin + nrec) return;          // blocks that only upload optics (B > blocks * threads)

    if ((long long)blockIdx.x < nbin) {
        // ---- H2 + first half of H4: binning role, one particle per thread
        binning_role(a, (long long)blockIdx.x * kPrepThreads + threadIdx.x);
        // H3: the last binning block to get here scans the counts (the record role blocks are still busy: off the critical path)
        __shared__ bool s_last;
        __threadfence();                                          // this block's counter atomics before its done-ticket
        __syncthreads();
        if (threadIdx.x == 0) s_last = atomicAdd(a.done, 1u) == (uint32_t)(nbin - 1);
        __syncthreads();
        if (s_last) {
            __threadfence();
            scan_counts(a);
        }
        return;
    }

    // ---- H1: record role, 8 lanes per particle; group g of the block takes the g-th particle in "prisms first" order
    const int lane = threadIdx.x & 31;
    const long long n0 = (long long)(blockIdx.x - nbin) * kRecPerBlock;
    const long long np_ = n0 + (lane & (kRecPerBlock - 1));
    const bool is_prism = np_ < a.N && a.kind[np_] == 1u;
    const unsigned mp = __ballot_sync(0xffffffffu, is_prism) & ((1u << kRecPerBlock) - 1u);
    const int g = threadIdx.x >> 3, npr = __popc(mp);
    const int slot = g < npr ? (int)__fns(mp, 0, g + 1) : (int)__fns(~mp & ((1u << kRecPerBlock) - 1u), 0, g - npr + 1);
    record_role(a, n0 + slot, threadIdx.x & 7, 0xffu << (lane & 24));
}

__global__ void k_set_optics(FrameOptics* optics, const OpticsChunk oc)
{
    const int k = threadIdx.x;
    if (k < oc.count) optics[oc.first + k] = oc.f[k];
}

static FrameOptics frame_optics(const osog_ctx* c, const osog_optics* o, int b)
{
    FrameOptics f;
    const double lam = o->lambda_um[b];
    f.inv_lambda = 1.0 / lam;
    f.fx0_pitch = sin(o->tilt_x_rad) / lam * o->pitch_um;
    f.fy0_pitch = sin(o->tilt_y_rad) / lam * o->pitch_um;
    f.pupil_thresh = -1;
    if (o->pupil_enabled && o->NA != nullptr) {
        const double r = o->NA[b] * o->pitch_um / lam;
        const double t = floor(r * r * ((double)c->H * c->H) * ((double)c->W * c->W));
        f.pupil_thresh = t >= 9.0e18 ? -1 : (long long)t;     // a radius beyond every bin is all-pass
    }
    f.defocus_um = o->defocus_um;
    const double q = o->n_medium / lam;
    f.nm_over_lambda_sq = q * q;
    const double rp = o->n_medium * o->pitch_um / lam;
    const double tp = floor(rp * rp * ((double)c->H * c->H) * ((double)c->W * c->W));
    f.prop_thresh = tp >= 9.0e18 ? -1 : (long long)tp;
    f.pad_ = 0.0;
    return f;
}

cudaError_t upload_optics(osog_ctx* c, const osog_optics* o, OpticsChunk* first)
{
    const int B = o->B;
    for (int s = 0; s < B; s += kOpticsChunk) {
        OpticsChunk oc;
        oc.first = s;
        oc.count = min(kOpticsChunk, B - s);
        for (int k = 0; k < oc.count; ++k) oc.f[k] = frame_optics(c, o, s + k);
        for (int k = oc.count; k < kOpticsChunk; ++k) oc.f[k] = oc.f[0];
        if (s == 0 && first != nullptr) *first = oc;
        if (s > 0 || first == nullptr) {
            k_set_optics<<<1, kOpticsChunk, 0, c->stream>>>(c->optics, oc);
            cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return e;
        }
    }
    return cudaSuccess;
}

cudaError_t launch_binning(osog_ctx* c, const osog_particles* p, long long N, const osog_optics* o, float* d_obb, bool unit_dn)
{
    const int B = o->B;
    const long long tiles = (long long)B * c->ntx * c->nty;
    c->last_B = B;
    c->last_tiles = tiles;
    c->last_N = N;
    c->last_frame_start = B > 1 ? p->frame_start : nullptr;
    c->last_has_ramp = -1;                           // set again by a call that runs the sort and a field-capable composition
    c->last_topo = o->topography_amplitude;
    c->last_seed = o->seed;
    cudaError_t e;
    // Invariant kept by the kernels themselves (no memset nodes in the steady state): the counter slot and the status
    // slot of this call are all zero on entry (cleared by the previous call's k_sort_cull, which works on the other
    // slot).  After a failed or atomic-variant call: clear explicitly.
    if (c->scratch_dirty) {
        if ((e = cudaMemsetAsync(c->count, 0, sizeof(uint32_t) * 2 * (size_t)c->count_stride, c->stream)) != cudaSuccess) return e;
        if ((e = cudaMemsetAsync(c->status, 0, 2 * sizeof(DeviceStatus), c->stream)) != cudaSuccess) return e;
        if ((e = cudaMemsetAsync(c->done, 0, sizeof(uint32_t), c->stream)) != cudaSuccess) return e;
        c->slot_tiles[0] = c->slot_tiles[1] = 0;
    }
    c->scratch_dirty = true;
    c->status_idx ^= 1;
    c->slot_tiles[c->status_idx] = tiles;
    DeviceStatus* status = c->status + c->status_idx;

    PrepArgs a;
    a.cx = p->cx; a.cy = p->cy; a.cz = p->cz; a.qw = p->qw; a.qx = p->qx; a.qy = p->qy; a.qz = p->qz;
    a.d0 = p->d0; a.d1 = p->d1; a.d2 = p->d2; a.n_p = p->n_p; a.kind = p->kind;
    a.frame_start = B > 1 ? p->frame_start : nullptr;
    a.N = N; a.B = B; a.H = c->H; a.W = c->W; a.ntx = c->ntx; a.nty = c->nty;
    a.pitch = o->pitch_um; a.n_medium = o->n_medium;
    a.rec = c->rec; a.rec2 = c->rec2; a.tbox = c->tbox; a.pframe = c->pframe;
    a.count = c->count + (size_t)c->status_idx * c->count_stride; a.slices = c->slices; a.slice_cap = c->slice_cap;
    a.offset = c->offset; a.done = c->done; a.max_pairs = c->max_pairs;
    a.obb = d_obb;
    a.unit_dn = unit_dn ? 1 : 0;
    a.optics = c->optics; a.status = status;
    if ((e = upload_optics(c, o, &a.oc)) != cudaSuccess) return e;

    const int threads = kPrepThreads;
    const long long nb = (N + threads - 1) / threads;
    const long long nrec = (N + kRecPerBlock - 1) / kRecPerBlock;
    long long blocks = (nb > 0 ? nb : 1) + nrec;
    if (blocks * threads < B) blocks = (B + threads - 1) / threads;     // the first threads also upload the optics
    k_prepare<<<(unsigned)blocks, threads, 0, c->stream>>>(a);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    return cudaSuccess;
}

}  // namespace osog
