// H4 (second half) - H7 of DESIGN.md: per-tile ordered composition, two kernels.
// k_sort_cull, two warps per 32 x 32 pixel tile:
//   1. fill the tile's segment of the CSR list (at offset[tile], the device scan of k_prepare) in ascending particle
//      index (deterministic summation order): rank sort of the tile's staging slice, or, for a list longer than the
//      slice, an ordered re-scan of the particles' tile ranges,
//   2. per list entry, test the particle's pixel bounding box and oriented box against the tile's eight 16 x 8 pixel
//      sub-tiles: 8-bit mask + evaluation code of the record -> meta.
// k_compose_tile, two CTAs of four warps per tile, every warp independent (no barrier, no shared list):
//   3. per warp (one sub-tile, 4 x 1 pixels per lane): walk the sorted list in batches of 32 entries and queue those whose
//      mask bit is set; whenever 32 survivors are queued (or the list ends) every lane prepares ONE survivor: it re-bases
//      a prism's fp64 slab coefficients to the sub-tile origin (rounding to fp32 only there), finds by an interval test
//      which exit / entry planes can be active anywhere in the sub-tile, and picks the evaluation class,
//   4. all lanes walk the prepared survivors class by class (one branch-free loop per class): ray-convex thickness from
//      the re-based coefficients (packed fp32 FMA and 3-input min/max for the prism slabs, two-float fp32 quadratic + fp32
//      sqrt for the ellipsoid), OPD accumulated per pixel in fp32 partial sums that are flushed to fp64 registers,
//   5. write OPD and / or exp(i 2 pi OPD / lambda) * ramp straight from the registers.
#include <type_traits>

#include "osog_internal.cuh"

namespace osog {

struct ComposeArgs {
    const float* rec;
    const float* rec2;           // prism slab coefficients as (hi, lo) float pairs (k_prepare)
    const uint32_t* offset;      // [tiles + 1] exclusive scan of the per-tile list lengths (k_prepare)
    const uint32_t* list;        // CSR list, every tile's segment sorted by k_sort_cull
    const uint16_t* meta;        // per list entry
    const FrameOptics* optics;
    const DeviceStatus* status;
    float* opd;
    float2* field;
    int H, W, ntx, nty;
    float topo_amp;              // micro-topography (reading A29): the height map is multiplied by 1 + topo_amp * eta(pixel); 0 = off
    unsigned long long seed;
};

constexpr int kWarps = kComposeThreads / 32;
constexpr int kSlotStride4 = 11;                   // survivor slot stride in float4 (10 used, odd stride: conflict-free lane-per-slot writes)
constexpr int kQueue = 64;                         // survivor queue entries per warp (32 being processed + up to 31 waiting)
#ifndef OSOG_CTA_SPLIT
#define OSOG_CTA_SPLIT 2
#endif
constexpr int kCtaSplit = OSOG_CTA_SPLIT;             // compose CTAs per tile (each takes kWarps / kCtaSplit sub-tiles)
constexpr int kCtaWarps = kWarps / kCtaSplit;
constexpr int kSmemSlots = kCtaWarps * 32 * kSlotStride4 * 16;
constexpr int kSmemBytes = kSmemSlots + kCtaWarps * 2 * kQueue * 4;   // k_compose_tile: per-warp survivor slots + two survivor queues

// ---- small PTX helpers ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float fast_sqrt(float x)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));    // one MUFU.SQRT (no denormal fix-up: w < 1e-38 -> t = 0)
    return r;
}
__device__ __forceinline__ float min3(float a, float b, float c)
{
    float r;
    asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}
__device__ __forceinline__ float max3(float a, float b, float c)
{
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}
// packed fp32 FMA (Blackwell FFMA2): d = a * b + c on both halves, one issue slot for two FMAs
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c)
{
    unsigned long long ra, rb, rc, rd;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(b.x), "f"(b.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rc) : "f"(c.x), "f"(c.y));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(ra), "l"(rb), "l"(rc));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(rd));
    return d;
}
// saturating fp32 add / subtract: the result is clamped to [0, 1] by the FMA pipe (NaN -> 0), no separate min / max
__device__ __forceinline__ float sub_sat(float a, float b)
{
    float r;
    asm("sub.sat.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ float add_sat(float a, float b)
{
    float r;
    asm("add.sat.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b));
    return r;
}
// ---- fp64 prism evaluation (refinement of flagged pixels, and the atomic variant) -------------------------------------
// r64: 24 doubles (U, V, Cx, Cn per slab, relative to pixel (jc, ic)); dj, di: pixel offsets from (jc, ic).
__device__ __noinline__ double prism_t64(const double* r64, uint32_t vmask, double dj, double di)
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

// ---- preparation of one prism survivor by ONE lane (32 survivors are prepared at once, one per lane) --------------------
// Evaluation classes of a prepared survivor:
constexpr uint32_t kClsFull = 1u /* 1 + steep slabs: 1, 2, 3 */, kClsF64 = 4u, kClsPair = 5u, kClsLin = 6u, kClsNone = 7u;
// For each of the 6 slabs: re-base its coefficients from the particle's reference pixel (jc, ic) to the warp's sub-tile
// origin (wx0, wy0) and round to fp32 there: all later fp32 arithmetic uses pixel offsets 0..15 / 0..7 (DESIGN.md section
// 6).  The re-basing itself runs in fp32 on the record's exact-grid (hi, lo) pairs (k_prepare; already scaled by the
// particle's chord scale s, s t <= 1/2): the FMAs on the hi parts are exact, so hi + lo carries the fp64 result.  Then an
// interval test over the sub-tile: exit plane k takes values in [emin_k, emax_k]; it can be the lowest exit plane somewhere
// only if emin_k <= min_q emax_q (likewise for the entry planes with max / min).  If the lowest possible exit lies below
// the highest possible entry everywhere, the prism does not touch the sub-tile at all (kClsNone).  If at most two exit and
// two entry planes remain, they are copied into a compact block (kClsPair: 2 + 2 planes instead of 6 + 6 per pixel).
// A steep slab (slope > kSteepSlope; the first NS slabs of the record) is stored again as (hi, lo) pairs, now on the
// finer grid of the sub-tile: hi = multiple of q = 2^(e - 21), 2^e > every intermediate of  C - U lx - V ly  over the
// sub-tile, so the evaluation's fp32 FMAs on the hi parts are exact and hi + lo is good to 2^-24 relative of the (small)
// result; the class with the lo-part FMAs (1 + NS) is only taken when a steep plane survives the interval test.
// Slot layout (float4 units; one 128-bit store per slab, conflict-free across the lanes' slots): 0..5 = (Ex, En, U, V) of slab
// 0..5 (hi parts for steep slabs), 6 = (-, dn / s, -, particle index), 7 and 8 = lo parts (Ex, En, U, V) of slab 0 and 1; or,
// class kClsPair, 7..9 = Cx_a Cx_b Ux_a Ux_b | Vx_a Vx_b Cn_c Cn_d | Un_c Un_d Vn_c Vn_d (exit planes a, b; entry planes c, d).
// An ellipsoid slot holds the record's words 40..53 in float4 0..3.
__device__ __forceinline__ uint32_t prep_prism(float4* __restrict__ slot, const float4* __restrict__ rec, const float4* __restrict__ pairs,
                                               int wx0, int wy0)
{
    float* sw = reinterpret_cast<float*>(slot);
    const float4 h2 = __ldg(rec + 2);                                  // flags, dn, cz, index
    const int4 h3 = __ldg(reinterpret_cast<const int4*>(rec + 3));     // jc, ic, zmax, chord scale
    sw[25] = h2.y * __int_as_float(0x7f000000 - h3.w);                 // dn / s: s is a power of two, so 1 / s is an exponent flip (exact)
    const float oj = (float)(wx0 - h3.x), oi = (float)(wy0 - h3.y);    // exact small integers
    const int ns = (int)((__float_as_uint(h2.x) >> 8) & 7u);
    float emin[6], nmax[6];
    float xlow = __int_as_float(0x7f800000), nhigh = __int_as_float(0xff800000);   // min_q emax_q, max_q nmin_q
#pragma unroll
    for (int q = 0; q < 6; ++q) {
        const float4 h = __ldg(pairs + 2 * q), l = __ldg(pairs + 2 * q + 1);       // U, V, Cx, Cn: hi parts | lo parts
        const float mh = fmaf(h.x, oj, h.y * oi);                      // exact (grid multiples below 2^24 q)
        const float ml = fmaf(l.x, oj, l.y * oi);
        const float xh = h.z - mh, nh = h.w - mh;                      // exact
        const float xl = l.z - ml, nl = l.w - ml;
        float exf = xh + xl, enf = nh + nl, uf = h.x + l.x, vf = h.y + l.y;   // one rounding each: the fp64 value in fp32
        if (q < 2 && q < ns) {                                         // steep slab: (hi, lo) once more, on the sub-tile's grid
            const float mb = fmaxf(fabsf(exf), fabsf(enf)) + 15.0f * fabsf(uf) + 7.0f * fabsf(vf);
            const int e = (int)(__float_as_uint(mb) >> 23) - 126;      // mb < 2^e
            const float cq = __int_as_float(((e + 129) << 23) | 0x400000);   // 1.5 * 2^23 * q, q = 2^(e - 21)
            const float exh = (exf + cq) - cq, enh = (enf + cq) - cq, uh = (uf + cq) - cq, vh = (vf + cq) - cq;
            slot[7 + q] = make_float4((xh - exh) + xl, (nh - enh) + nl, (h.x - uh) + l.x, (h.y - vh) + l.y);
            exf = exh; enf = enh; uf = uh; vf = vh;
        }
        slot[q] = make_float4(exf, enf, uf, vf);
        // value range of  C - U lx - V ly  over lx in [0, 15], ly in [0, 7]: centre value -+ half range, padded for the
        // fp32 roundings of this block and of the evaluation (a few ulp of the largest magnitude involved)
        const float ec = fmaf(-3.5f, vf, fmaf(-7.5f, uf, exf));
        const float hr = fmaf(3.5f, fabsf(vf), 7.5f * fabsf(uf));
        const float d = enf - exf;
        const float hrp = fmaf(1.0e-6f, (fabsf(exf) + fabsf(enf)) + hr, hr);
        const float lo_x = ec - hrp, hi_x = ec + hrp;
        emin[q] = lo_x;
        nmax[q] = hi_x + d;
        xlow = fminf(xlow, hi_x);
        nhigh = fmaxf(nhigh, lo_x + d);
    }
    if (!(xlow > nhigh)) return kClsNone;                              // empty chord everywhere in the sub-tile
    uint32_t mx = 0u, mn = 0u;                                         // planes that can be active somewhere
#pragma unroll
    for (int q = 0; q < 6; ++q) {
        mx |= emin[q] <= xlow ? (1u << q) : 0u;
        mn |= nmax[q] >= nhigh ? (1u << q) : 0u;
    }
    if ((mx | mn) & ((1u << ns) - 1u)) return kClsFull + (uint32_t)ns; // a steep plane matters here: lo-part classes
    if (__popc(mx) > 2 || __popc(mn) > 2) return kClsFull;
    const int a0 = __ffs(mx) - 1, c0 = __ffs(mn) - 1;
    if (__popc(mx) == 1 && __popc(mn) == 1) {                          // one exit and one entry plane: s t is one plane, clamped
        const float4 sa = slot[a0], sc = slot[c0];
        slot[7] = make_float4(sa.x - sc.y, sa.z - sc.z, sa.w - sc.w, 0.0f);
        return kClsLin;
    }
    const uint32_t mx1 = mx & (mx - 1u), mn1 = mn & (mn - 1u);
    const int a1 = mx1 ? __ffs(mx1) - 1 : a0, c1 = mn1 ? __ffs(mn1) - 1 : c0;      // a single plane is simply used twice
    const float4 sa = slot[a0], sb = slot[a1], sc = slot[c0], sd = slot[c1];
    slot[7] = make_float4(sa.x, sb.x, sa.z, sb.z);
    slot[8] = make_float4(sa.w, sb.w, sc.y, sd.y);
    slot[9] = make_float4(sc.z, sd.z, sc.w, sd.w);
    return kClsPair;
}

// ---- sub-tile cull (tile_meta below): does the particle (header words 0..7: centre, oriented box, packed pixel bounding
// box) touch a 16 x 8 pixel sub-tile?  Bounding-box overlap, then a separating-axis test against the oriented box of the
// silhouette (which contains it by construction).
// evaluation code in the sign bits of the (positive) half lengths and of a_x (a_x >= 0 by construction)
__device__ __forceinline__ uint32_t header_code(const float4 h0, const float4 h1)
{
    return (__float_as_uint(h1.x) >> 31) | ((__float_as_uint(h1.y) >> 31) << 1) | ((__float_as_uint(h0.z) >> 31) << 2);
}

// ---- thickness, 4 pixels of one row per lane --------------------------------------------------------------------------
struct LaneGeom {
    float2 nlx[4];     // (-lx_k, -lx_k), lx_k = 4 (lane & 3) + k : pixel column offset inside the warp sub-tile
    float2 nly;        // (-ly, -ly),     ly = lane >> 2
    float xf, yf;      // absolute pixel column of this lane's first pixel, and its row (exact small integers)
};

// Ellipsoid (kind 0): w = 1 - d^T S d as a quadratic polynomial of the pixel offsets from (jc, ic), from the record's
// (hi, lo) coefficient pairs (k_prepare): Horner in packed fp32, exact on the hi halves, so w = hi + lo is good to
// ~2^-47 of the largest intermediate (the precision the outline needs: t ~ sqrt(w)) without any fp64 instruction;
// the saturating add clamps w to [0, 1] (w <= 1 by construction); pend += (dn T0) sqrt(w).
__device__ __forceinline__ void eval_ellipsoid(const float4* __restrict__ slot, const LaneGeom& g, float (&pend)[4])
{
    const float4 c0 = slot[0], c1 = slot[1], c2 = slot[2];      // An, Bn | Cn, D | E, F  (each as hi, lo)
    const float4 c3 = slot[3];                                   // jc, ic
    const float K = slot[6].y;
    const float ndi = c3.y - g.yf, ndj0 = c3.x - g.xf;           // -(i - ic), -(j - jc): exact small integers
    const float2 ndi2 = make_float2(ndi, ndi);
    const float2 t1 = ffma2(make_float2(c1.x, c1.y), ndi2, make_float2(c2.x, c2.y));    // E + C di
    const float2 wr = ffma2(t1, ndi2, make_float2(c2.z, c2.w));                          // F - (E + C di) di
    const float2 gr = ffma2(make_float2(c0.z, c0.w), ndi2, make_float2(c1.z, c1.w));    // D + B di
    const float2 an = make_float2(c0.x, c0.y);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float ndj = ndj0 - (float)k;
        const float2 ndj2 = make_float2(ndj, ndj);
        const float2 sl = ffma2(an, ndj2, gr);                   // D + B di + A dj
        const float2 w2 = ffma2(sl, ndj2, wr);                   // w = F - (E + C di) di - (D + B di + A dj) dj
        const float t = fast_sqrt(add_sat(w2.x, w2.y));
        pend[k] = fmaf(t, K, pend[k]);
    }
}

// Prism whose every pixel goes to fp64 (a vertical face, a slab steeper than kAllF64Slope, or > 2 steep slabs): rare.
// One pixel per call; returns dn * t (by value, so that the accumulators stay in registers).
__device__ __noinline__ double prism_f64_px(const float4* __restrict__ rec, double xd, double yd)
{
    const int4 h3 = __ldg(reinterpret_cast<const int4*>(rec + 3));
    const float4 h2 = __ldg(rec + 2);
    return (double)h2.y * prism_t64(reinterpret_cast<const double*>(rec + 4), __float_as_uint(h2.x) >> 16,
                                    xd - (double)h3.x, yd - (double)h3.y);
}

// Prism (kind 1): 6 slabs, exit_k = Ex_k - U_k lx - V_k ly, enter_k = En_k - U_k lx - V_k ly from the re-based, scaled
// fp32 coefficients (packed FFMA2: the exit and the entry plane of one slab per instruction, they share U and V),
// s t = sat(min_k exit_k - max_k enter_k) with 3-input
// min / max and a saturating subtraction.  The first NS (<= 2) slabs are steep (slope > kSteepSlope): their values are
// the exact hi-part FMAs plus a packed lo-part FMA (one FFMA2 + 2 FADD per pixel and steep slab), no fp64.
template <int NS>
__device__ __forceinline__ void eval_prism(const float4* __restrict__ slot, const LaneGeom& g, float (&pend)[4])
{
    const float4 s0 = slot[0], s1 = slot[1], s2 = slot[2], s3 = slot[3], s4 = slot[4], s5 = slot[5];   // (Ex, En, U, V) per slab
    const float dn = slot[6].y;
    // row terms: (exit, entry) value of every slab at this lane's row, column offset 0
    const float2 r0 = ffma2(make_float2(s0.w, s0.w), g.nly, make_float2(s0.x, s0.y));
    const float2 r1 = ffma2(make_float2(s1.w, s1.w), g.nly, make_float2(s1.x, s1.y));
    const float2 r2 = ffma2(make_float2(s2.w, s2.w), g.nly, make_float2(s2.x, s2.y));
    const float2 r3 = ffma2(make_float2(s3.w, s3.w), g.nly, make_float2(s3.x, s3.y));
    const float2 r4 = ffma2(make_float2(s4.w, s4.w), g.nly, make_float2(s4.x, s4.y));
    const float2 r5 = ffma2(make_float2(s5.w, s5.w), g.nly, make_float2(s5.x, s5.y));
    float2 l0 = make_float2(0.f, 0.f), ul0 = l0, l1 = l0, ul1 = l0;   // lo parts of the steep slabs: (exit, entry) row terms, U
    if (NS > 0) {
        const float4 l = slot[7];
        l0 = ffma2(make_float2(l.w, l.w), g.nly, make_float2(l.x, l.y));
        ul0 = make_float2(l.z, l.z);
    }
    if (NS > 1) {
        const float4 l = slot[8];
        l1 = ffma2(make_float2(l.w, l.w), g.nly, make_float2(l.x, l.y));
        ul1 = make_float2(l.z, l.z);
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        float2 p0 = ffma2(make_float2(s0.z, s0.z), g.nlx[k], r0), p1 = ffma2(make_float2(s1.z, s1.z), g.nlx[k], r1);
        const float2 p2 = ffma2(make_float2(s2.z, s2.z), g.nlx[k], r2), p3 = ffma2(make_float2(s3.z, s3.z), g.nlx[k], r3);
        const float2 p4 = ffma2(make_float2(s4.z, s4.z), g.nlx[k], r4), p5 = ffma2(make_float2(s5.z, s5.z), g.nlx[k], r5);
        if (NS > 0) {
            const float2 lo = ffma2(ul0, g.nlx[k], l0);
            p0.x += lo.x;
            p0.y += lo.y;
        }
        if (NS > 1) {
            const float2 lo = ffma2(ul1, g.nlx[k], l1);
            p1.x += lo.x;
            p1.y += lo.y;
        }
        const float ex = fminf(min3(p0.x, p1.x, p2.x), min3(p3.x, p4.x, p5.x));
        const float en = fmaxf(max3(p0.y, p1.y, p2.y), max3(p3.y, p4.y, p5.y));
        pend[k] = fmaf(sub_sat(ex, en), dn, pend[k]);
    }
}

// Prism of which at most two exit and two entry planes can be active in this sub-tile (prep_prism): 2 + 2 plane values,
// one min, one max per pixel.  Same fp32 coefficients as the full evaluation, so the result is the same number.
__device__ __forceinline__ void eval_prism_pair(const float4* __restrict__ slot, const LaneGeom& g, float (&pend)[4])
{
    const float4 a = slot[7], b = slot[8], c = slot[9];
    const float dn = slot[6].y;
    const float2 xr = ffma2(make_float2(b.x, b.y), g.nly, make_float2(a.x, a.y));
    const float2 nr = ffma2(make_float2(c.z, c.w), g.nly, make_float2(b.z, b.w));
    const float2 xu = make_float2(a.z, a.w), nu = make_float2(c.x, c.y);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float2 e = ffma2(xu, g.nlx[k], xr), n = ffma2(nu, g.nlx[k], nr);
        pend[k] = fmaf(sub_sat(fminf(e.x, e.y), fmaxf(n.x, n.y)), dn, pend[k]);
    }
}

// Prism of which one exit and one entry plane can be active in this sub-tile: s t = sat(D - Du lx - Dv ly), one saturating
// FMA per pixel.
__device__ __forceinline__ float ffma_sat(float a, float b, float c)
{
    float d;
    asm("fma.rn.sat.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}
__device__ __forceinline__ void eval_prism_lin(const float4* __restrict__ slot, const LaneGeom& g, float (&pend)[4])
{
    const float4 a = slot[7];
    const float dn = slot[6].y;
    const float r = fmaf(a.z, g.nly.x, a.x);
#pragma unroll
    for (int k = 0; k < 4; ++k) pend[k] = fmaf(ffma_sat(a.y, g.nlx[k].x, r), dn, pend[k]);
}

// The evaluation loops add into fp32 partial sums; every kFlush survivors (and at the end of a class) these are widened
// and added to the fp64 per-pixel accumulators: one widening conversion + DADD per pixel and kFlush particles.
constexpr int kFlush = 8;
__device__ __forceinline__ void flush(float (&pend)[4], double (&acc)[4])
{
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        acc[k] += (double)pend[k];
        pend[k] = 0.0f;
    }
}

// all lanes evaluate the survivors whose bit is set in `m` (slot = survivor index), ascending, flushing every kFlush
template <class Eval>
__device__ __forceinline__ void run_class(unsigned m, const float4* __restrict__ my_slots, float (&pend)[4], double (&acc)[4], Eval eval)
{
#pragma unroll 1
    while (m) {
#pragma unroll 1
        for (int q = 0; q < kFlush && m; ++q) {
            const int r = __ffs(m) - 1;
            m &= m - 1u;
            eval(my_slots + r * kSlotStride4);
        }
        flush(pend, acc);
    }
}

// ---- H4 (second half) + tile-level cull: two WARPS per tile ------------------------------------------------------------
// Fills the tile's CSR segment list[offset[tile] .. offset[tile + 1]) in ascending particle index (the canonical,
// deterministic summation order) and writes one 16-bit word per list entry: bits 0..7 = which of the tile's 8 warp
// sub-tiles (16 x 8 pixels) the particle can touch (bounding box + oriented-box test), bits 8..10 = the evaluation code of
// the record.  k_compose_tile then needs no barrier.
// Rank sort (ids are unique inside a tile): the tile's staging slice is copied to shared memory, every lane counts the
// ids smaller than its own with broadcast 128-bit reads; the record header loads of the cull are issued first so that
// their latency hides behind the counting.  A list longer than the staging slice (a crowded tile) is rebuilt instead from
// the particles' tile ranges (tbox, written by k_prepare): the two warps walk the frame's particles from both ends in
// index order and keep those whose range contains the tile, which yields the ascending list directly.
constexpr int kWarpSortCap = 1024;                 // largest staging slice (4 KB of shared memory per tile)
#ifndef OSOG_SORT_WARPS
#define OSOG_SORT_WARPS 2
#endif
constexpr int kSortWarps = OSOG_SORT_WARPS;        // warps that share one tile in k_sort_cull (power of two <= kWarps)

// r += (a < v): one compare and one predicated add
__device__ __forceinline__ void count_less(uint32_t& r, uint32_t a, uint32_t v)
{
    asm("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %1, %2;\n\t@p add.u32 %0, %0, 1;\n\t}" : "+r"(r) : "r"(a), "r"(v));
}

// All eight sub-tile tests of one list entry at once: sub-tile (wx, wy) has origin (x0 + 16 wx, y0 + 8 wy) and centre
// offset (7.5, 3.5); it is kept iff its pixel range overlaps the particle's pixel bounding box and its centre's
// projections on the two box axes are within half length + the sub-tile's own half extent along that axis.
__device__ __forceinline__ uint32_t tile_meta(const float4 h0, const float4 h1, int tx, int ty)
{
    const uint32_t bx = __float_as_uint(h1.z), by = __float_as_uint(h1.w);
    const int pj0 = bx & 0xffff, pj1 = bx >> 16, pi0 = by & 0xffff, pi1 = by >> 16;
    const int x0 = tx * kTile, y0 = ty * kTile;
    const float axx = fabsf(h0.z), ayy = h0.w, ha = fabsf(h1.x), hb = fabsf(h1.y);
    const float ta = ha + (7.5f * axx + 3.5f * fabsf(ayy)), tb = hb + (7.5f * fabsf(ayy) + 3.5f * axx);
    const float ddx0 = (float)x0 + 7.5f - h0.x, ddy0 = (float)y0 + 3.5f - h0.y;
    uint32_t mask = 0;
#pragma unroll
    for (int wy = 0; wy < 4; ++wy) {
        const bool row_ok = pi0 <= y0 + 8 * wy + 7 && pi1 >= y0 + 8 * wy;
        const float ddy = ddy0 + (float)(8 * wy);
#pragma unroll
        for (int wx = 0; wx < 2; ++wx) {
            const bool col_ok = pj0 <= x0 + 16 * wx + 15 && pj1 >= x0 + 16 * wx;
            const float ddx = ddx0 + (float)(16 * wx);
            const float pa = fabsf(ddx * axx + ddy * ayy), pb = fabsf(ddy * axx - ddx * ayy);
            mask |= (row_ok && col_ok && pa <= ta && pb <= tb) ? (1u << (2 * wy + wx)) : 0u;
        }
    }
    return mask | (header_code(h0, h1) << 8);
}

struct SortArgs {
    const float* recs;
    const int4* tbox;             // [N] tile ranges of the particles (tx0 > tx1: not listed)
    const int32_t* frame_start;   // device [B + 1] or nullptr (one frame)
    long long N;
    const uint32_t* count;        // this call's per-tile list lengths
    uint32_t* count_next;         // the other counter slot, cleared here for the next call
    const uint32_t* offset;       // [tiles + 1] device scan
    const uint32_t* slices;       // [tiles][slice_cap] unsorted staging slices
    int slice_cap;
    uint32_t* list;               // CSR list (output)
    uint16_t* meta;               // (output)
    const DeviceStatus* status;
    DeviceStatus* status_next;
    int ntx, nty, n_tiles, n_clear;
};

__global__ void __launch_bounds__(kComposeThreads) k_sort_cull(const SortArgs a)
{
    __shared__ __align__(16) uint32_t s_all[(kWarps / kSortWarps) * kWarpSortCap];
    pdl_trigger();                                               // k_compose_tile's CTAs may become resident
    pdl_wait();                                                  // k_prepare has finished: counts, offsets, slices, records are visible
    // kSortWarps warps per tile: they stage the list together in one shared slice, each ranks / culls every kSortWarps-th group of 32 entries
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int half = wid % kSortWarps;                           // this warp's part of the tile's work
    const int tile = (blockIdx.x * kWarps + wid) / kSortWarps;
    if (blockIdx.x == 0 && threadIdx.x == 0) {                   // the other status slot belongs to the next call
        a.status_next->bits = 0u; a.status_next->max_count = 0u; a.status_next->pairs = 0ull;
    }
    const uint32_t L = tile < a.n_tiles ? a.count[tile] : 0u;
    if (tile < a.n_clear && lane == 0 && half == 0) a.count_next[tile] = 0u;    // every counter the other slot's last user touched
    if (L == 0u || (a.status->bits & OSOG_WOVERFLOW) != 0u) return;   // empty, or more pairs than the CSR list holds (frames are zero-filled)
    const uint32_t beg = a.offset[tile];
    uint32_t* glist = a.list + beg;
    uint16_t* gmeta = a.meta + beg;
    const int tpf = a.ntx * a.nty;
    const int b = tile / tpf, rt = tile - b * tpf;
    const int ty = rt / a.ntx, tx = rt - ty * a.ntx;
    const float4* recs4 = reinterpret_cast<const float4*>(a.recs);
    if (L <= (uint32_t)a.slice_cap) {
        const uint32_t* slice = a.slices + (size_t)tile * a.slice_cap;
        uint32_t* s = s_all + (wid / kSortWarps) * kWarpSortCap; // the tile's warps share one slice
        const uint32_t L4 = (L + 3u) & ~3u;
        for (uint32_t k = lane + 32 * half; k < L4; k += 32 * kSortWarps) s[k] = k < L ? slice[k] : 0xffffffffu;
        asm volatile("bar.sync %0, %1;" ::"r"(1 + wid / kSortWarps), "n"(32 * kSortWarps) : "memory");   // tile barrier: the list is staged
        for (uint32_t k = lane + 32 * half; k < L; k += 32 * kSortWarps) {
            const uint32_t v = s[k];
            const float4* rec = recs4 + (size_t)v * (kRecWords / 4);
            const float4 h0 = __ldg(rec), h1 = __ldg(rec + 1);   // cxp, cyp, ax, ay | ha, hb, bbx, bby
            uint32_t r = 0, r1 = 0;                               // two chains of predicated adds
            const uint4* s4 = reinterpret_cast<const uint4*>(s);
            for (uint32_t m = 0; m < L4 / 4; ++m) {
                const uint4 q = s4[m];
                count_less(r, q.x, v); count_less(r1, q.y, v); count_less(r, q.z, v); count_less(r1, q.w, v);
            }
            r += r1;
            glist[r] = v;                                        // H4: the sorted CSR segment (also what osog_debug_bins returns)
            gmeta[r] = (uint16_t)tile_meta(h0, h1, tx, ty);
        }
        return;
    }
    // ---- crowded tile: the slice holds only part of the list.  Rebuild it in order from the tile ranges: warp 0 walks the
    // frame's particles upwards from the first and fills the segment from its front, warp 1 walks downwards from the last
    // and fills from the back; together they find exactly L particles whose range contains (tx, ty).
    long long p_lo = 0, p_hi = a.N;
    if (a.frame_start != nullptr) { p_lo = a.frame_start[b]; p_hi = a.frame_start[b + 1]; }
    const long long p_mid = p_lo + (p_hi - p_lo) / (kSortWarps == 1 ? 1 : 2);
    const unsigned lt = (1u << lane) - 1u;
    if (half == 0) {
        uint32_t pos = 0;
        for (long long base = p_lo; base < p_mid; base += 32) {
            const long long n = base + lane;
            bool in = false;
            if (n < p_mid) { const int4 tb = __ldg(a.tbox + n); in = tb.x <= tx && tx <= tb.y && tb.z <= ty && ty <= tb.w; }
            const unsigned m = __ballot_sync(0xffffffffu, in);
            if (in) glist[pos + __popc(m & lt)] = (uint32_t)n;
            pos += __popc(m);
        }
    } else if (half == 1) {
        uint32_t pos = L;
        for (long long top = p_hi; top > p_mid; top -= 32) {
            const long long n = top - 32 + lane;                 // lanes ascending inside the chunk [top - 32, top)
            bool in = false;
            if (n >= p_mid) { const int4 tb = __ldg(a.tbox + n); in = tb.x <= tx && tx <= tb.y && tb.z <= ty && ty <= tb.w; }
            const unsigned m = __ballot_sync(0xffffffffu, in);
            pos -= __popc(m);
            if (in) glist[pos + __popc(m & lt)] = (uint32_t)n;
        }
    }
    asm volatile("bar.sync %0, %1;" ::"r"(1 + wid / kSortWarps), "n"(32 * kSortWarps) : "memory");   // the segment is complete
    for (uint32_t k = lane + 32 * half; k < L; k += 32 * kSortWarps) {
        const float4* rec = recs4 + (size_t)glist[k] * (kRecWords / 4);
        gmeta[k] = (uint16_t)tile_meta(__ldg(rec), __ldg(rec + 1), tx, ty);
    }
}

static cudaError_t launch_sort_cull(osog_ctx* c, unsigned grid, bool pdl)
{
    SortArgs a;
    a.recs = c->rec; a.tbox = c->tbox; a.frame_start = c->last_frame_start; a.N = c->last_N;
    a.count = c->count + (size_t)c->status_idx * c->count_stride;
    a.count_next = c->count + (size_t)(c->status_idx ^ 1) * c->count_stride;
    a.offset = c->offset; a.slices = c->slices; a.slice_cap = c->slice_cap; a.list = c->list; a.meta = c->meta;
    a.status = c->status + c->status_idx; a.status_next = c->status + (c->status_idx ^ 1);
    a.ntx = c->ntx; a.nty = c->nty; a.n_tiles = (int)grid;
    const long long n_clear = c->slot_tiles[c->status_idx ^ 1];
    a.n_clear = (int)n_clear;
    const unsigned cover = (unsigned)(n_clear > (long long)grid ? n_clear : (long long)grid);
    const dim3 g((kSortWarps * cover + kWarps - 1) / kWarps), blk(kComposeThreads);
    cudaError_t e;
    if (pdl) {
        e = launch_pdl(k_sort_cull, g, blk, 0, c->stream, a);
    } else {
        k_sort_cull<<<g, blk, 0, c->stream>>>(a);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) c->slot_tiles[c->status_idx ^ 1] = 0;
    return e;
}

// Micro-topography (reading A29): every thickness at a pixel is multiplied by 1 + amp * eta, eta ~ N(0, 1) white per
// pixel (Philox stream 2 of (seed, frame, pixel)), hence so is the OPD sum.  Out of line: it runs once per pixel, rarely.
__device__ __noinline__ double topo_factor(unsigned long long seed, uint32_t frame, uint32_t pixel, float amp)
{
    return 1.0 + (double)(amp * philox_normal(seed, frame, pixel, 2u));
}

// ---- H5-H7: every warp is independent (no barrier, no shared list): it walks its tile's sorted list in batches of 32
template <bool OPD, bool FIELD, bool RAMP>
__global__ void __launch_bounds__(kCtaWarps * 32, 4 * kCtaSplit) k_compose_tile(const ComposeArgs a)
{
    extern __shared__ __align__(16) unsigned char smem[];
    float4* s_slots = reinterpret_cast<float4*>(smem);                            // per-warp survivor slots

    const int tid = threadIdx.x, lane = tid & 31;
    const int wid = (tid >> 5) + kCtaWarps * (int)(blockIdx.x % kCtaSplit);     // sub-tile of the tile
    const int tx = (int)blockIdx.x / kCtaSplit, ty = (int)blockIdx.y, b = (int)blockIdx.z;   // grid = (ntx * split, nty, B)
    const int tile = (b * a.nty + ty) * a.ntx + tx;
    pdl_wait();                                                  // k_sort_cull (and all before it) has finished

    const bool overflow = (a.status->bits & OSOG_WOVERFLOW) != 0u;
    const uint32_t beg = a.offset[tile];
    const uint32_t L = overflow ? 0u : a.offset[tile + 1] - beg;
    const uint32_t* __restrict__ glist = a.list + beg;
    const uint16_t* __restrict__ gmeta = a.meta + beg;

    // ---- pixel ownership ------------------------------------------------------------------------------------------------
    const int wx0 = tx * kTile + (wid & 1) * 16, wy0 = ty * kTile + (wid >> 1) * 8;   // warp sub-tile origin
    const int lx = (lane & 3) * 4, ly = lane >> 2;
    const int j = wx0 + lx, i = wy0 + ly;
    LaneGeom g;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        g.nlx[k] = make_float2(-(float)(lx + k), -(float)(lx + k));
    }
    g.nly = make_float2(-(float)ly, -(float)ly);
    g.xf = (float)j;
    g.yf = (float)i;
    float4* my_slots = s_slots + (tid >> 5) * 32 * kSlotStride4;
    // two survivor queues per warp: prisms (particle index | record code << 29) and ellipsoids (particle index)
    uint32_t* queue_p = reinterpret_cast<uint32_t*>(smem + kSmemSlots) + (tid >> 5) * (2 * kQueue);
    uint32_t* queue_e = queue_p + kQueue;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    float pend[4] = {0.0f, 0.0f, 0.0f, 0.0f};

    const float4* recs4 = reinterpret_cast<const float4*>(a.rec);
    const unsigned lt = (1u << lane) - 1u;
    int nqp = 0, nqe = 0;                                        // queued prisms / ellipsoids (warp-uniform)
    // The list is read one entry per lane at the top of each batch.  Measured alternatives (profiles/r2_compose_ncu.md): a register
    // prefetch of the next batch (its two registers spill at 64 registers and the spill store waits for the load: no gain) and
    // cp.async staging of the next batch's particle indices and meta words in shared memory (137.2 against 133.9 us: not kept).
    for (uint32_t base = 0; base < L; base += 32) {
        // ---- lane <-> list entry base + lane: survivors of this warp's sub-tile join their kind's queue, in list order ---------
        const uint32_t kq = base + lane;
        const uint32_t meta = kq < L ? gmeta[kq] : 0u, pid = kq < L ? glist[kq] : 0u;
        const bool keep = ((meta >> wid) & 1u) != 0u;
        const uint32_t code = meta >> 8;
        const unsigned mkp = __ballot_sync(0xffffffffu, keep && code != 0u), mke = __ballot_sync(0xffffffffu, keep && code == 0u);
        if (keep) {
            if (code != 0u) queue_p[nqp + __popc(mkp & lt)] = (pid & 0x1fffffffu) | (code << 29);
            else queue_e[nqe + __popc(mke & lt)] = pid;
        }
        nqp += __popc(mkp);
        nqe += __popc(mke);
        __syncwarp();
        const bool last = base + 32 >= L;
        // ---- 32 prisms queued (or the list has ended): one lane prepares one prism, then all lanes evaluate them class by class;
        // fixed, data-defined summation order: 2 + 2 plane prisms, full prisms, one / two steep slabs, all-fp64 prisms, each class
        // in ascending list position
        while (nqp >= 32 || (last && nqp > 0)) {
            const int n = min(nqp, 32);
            uint32_t cls = kClsNone;
            if (lane < n) {
                const uint32_t ent = queue_p[lane];
                const uint32_t spid = ent & 0x1fffffffu;
                cls = ent >> 29;                                     // record code: 1..3 prism, 4 all-fp64 prism
                float4* sl = my_slots + lane * kSlotStride4;
                reinterpret_cast<uint32_t*>(sl)[27] = spid;
                if (cls != kClsF64)
                    cls = prep_prism(sl, recs4 + (size_t)spid * (kRecWords / 4),
                                     reinterpret_cast<const float4*>(a.rec2 + (size_t)spid * kPairWords), wx0, wy0);
            }
            const unsigned ml = __ballot_sync(0xffffffffu, cls == kClsLin);
            const unsigned mp = __ballot_sync(0xffffffffu, cls == kClsPair);
            const unsigned m1 = __ballot_sync(0xffffffffu, cls == kClsFull);
            const unsigned m2 = __ballot_sync(0xffffffffu, cls == kClsFull + 1u);
            const unsigned m3 = __ballot_sync(0xffffffffu, cls == kClsFull + 2u);
            const unsigned m4 = __ballot_sync(0xffffffffu, cls == kClsF64);
            uint32_t moved = 0u;                                     // the next queue entries move to the front
            if (32 + lane < nqp) moved = queue_p[32 + lane];
            __syncwarp();
            if (32 + lane < nqp) queue_p[lane] = moved;
            nqp -= n;
            run_class(ml, my_slots, pend, acc, [&](const float4* slot) { eval_prism_lin(slot, g, pend); });
            run_class(mp, my_slots, pend, acc, [&](const float4* slot) { eval_prism_pair(slot, g, pend); });
            run_class(m1, my_slots, pend, acc, [&](const float4* slot) { eval_prism<0>(slot, g, pend); });
            run_class(m2, my_slots, pend, acc, [&](const float4* slot) { eval_prism<1>(slot, g, pend); });
            run_class(m3, my_slots, pend, acc, [&](const float4* slot) { eval_prism<2>(slot, g, pend); });
#pragma unroll 1
            for (unsigned m = m4; m; m &= m - 1u) {
                const float4* slot = my_slots + (__ffs(m) - 1) * kSlotStride4;
                const float4* rec = recs4 + (size_t)__float_as_uint(slot[6].w) * (kRecWords / 4);
#pragma unroll
                for (int k = 0; k < 4; ++k) acc[k] += prism_f64_px(rec, (double)(g.xf + (float)k), (double)g.yf);
            }
            __syncwarp();
        }
        // ---- 32 ellipsoids queued (or the list has ended): every lane copies one record's fp32 (hi, lo) coefficients into its
        // slot, then all lanes evaluate slots 0 .. n-1 in order
        while (nqe >= 32 || (last && nqe > 0)) {
            const int n = min(nqe, 32);
            if (lane < n) {
                const float4* rec = recs4 + (size_t)queue_e[lane] * (kRecWords / 4);
                float4* sl = my_slots + lane * kSlotStride4;
                const float4 c0 = __ldg(rec + 10), c1 = __ldg(rec + 11), c2 = __ldg(rec + 12), c3 = __ldg(rec + 13);
                const float K = __ldg(reinterpret_cast<const float*>(rec) + 9);
                sl[0] = c0; sl[1] = c1; sl[2] = c2; sl[3] = c3;
                reinterpret_cast<float*>(sl)[25] = K;
            }
            uint32_t moved = 0u;
            if (32 + lane < nqe) moved = queue_e[32 + lane];
            __syncwarp();
            if (32 + lane < nqe) queue_e[lane] = moved;
            nqe -= n;
            const float4* slot = my_slots;
#pragma unroll 1
            for (int left = n; left > 0; left -= kFlush) {
#pragma unroll 1
                for (int q = min(left, kFlush); q > 0; --q, slot += kSlotStride4) eval_ellipsoid(slot, g, pend);
                flush(pend, acc);
            }
            __syncwarp();
        }
    }

    // ---- H6/H7: write-out straight from the registers ----------------------------------------------------------------------
    if (i >= a.H || j >= a.W) return;
    if (a.topo_amp != 0.0f) {
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (j + k < a.W) acc[k] *= topo_factor(a.seed, (uint32_t)b, (uint32_t)(i * a.W + j + k), a.topo_amp);
    }
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
        float2* out = a.field + row + j;
        if (overflow) {                                              // warp-uniform: the frame is zero-filled
            if (vec) {
                reinterpret_cast<float4*>(out)[0] = make_float4(0.f, 0.f, 0.f, 0.f);
                reinterpret_cast<float4*>(out)[1] = make_float4(0.f, 0.f, 0.f, 0.f);
            } else {
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (j + k < a.W) out[k] = make_float2(0.f, 0.f);
            }
            return;
        }
        // Eq. 2 with the oblique-illumination ramp: U = exp(i 2 pi (OPD / lambda + fx0 x_j + fy0 y_i)).  The
        // three terms are added in turns, in fp64, and reduced to [-1/2, 1/2] before the one fp32 sincos per pixel (no ramp
        // tables, no complex multiplications).
        const FrameOptics* fo = a.optics + b;
        const double inv_lambda = fo->inv_lambda;
        double ramp0 = 0.0, ramp_dx = 0.0;
        if (RAMP) {
            ramp_dx = fo->fx0_pitch;
            ramp0 = fma(ramp_dx, (double)j + 0.5, fo->fy0_pitch * ((double)i + 0.5));
        }
        // sin(pi x), cos(pi x) for |x| <= 1 (the reduced phase, in half turns): k = nearest integer to 2 x, r = x - k / 2 in
        // [-1/4, 1/4], Taylor polynomials of sin(pi r) (through r^9) and cos(pi r) (through r^8): truncation errors 2e-9 and
        // 2.5e-8, far below the fp32 rounding of the result; then the quadrant rotation by k.  Packed Horner coefficients of
        // sin(pi r) / r and cos(pi r):
        const float2 c3 = make_float2(0.0821458866f, 0.235330630f), c2 = make_float2(-0.599264529f, -1.33526277f);
        const float2 c1 = make_float2(2.55016404f, 4.05871213f), c0 = make_float2(-5.16771278f, -4.93480220f);
        const float2 cc = make_float2(3.14159265f, 1.0f);
        float2 u[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            double turns = fma(acc[k], inv_lambda, RAMP ? fma(ramp_dx, (double)k, ramp0) : 0.0);
            turns -= rint(turns);
            const float x = 2.0f * (float)turns;                     // angle / pi, in [-1, 1]
            const float kf = rintf(x + x);
            const int q = (int)kf;
            const float r = fmaf(kf, -0.5f, x);
            const float r2 = r * r;
            const float2 rr = make_float2(r2, r2);
            float2 pq = ffma2(rr, c3, c2);
            pq = ffma2(rr, pq, c1);
            pq = ffma2(rr, pq, c0);
            pq = ffma2(rr, pq, cc);
            float sp = pq.x * r, cp = pq.y;
            if (q & 1) { const float t = sp; sp = cp; cp = -t; }
            if (q & 2) { sp = -sp; cp = -cp; }
            u[k] = make_float2(cp, sp);
        }
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

template <bool OPD, bool FIELD, bool RAMP>
static cudaError_t launch_variant(const ComposeArgs& a, int B, cudaStream_t stream)
{
    // opt in to > 48 KB dynamic shared memory (cheap, idempotent; per device, so done on every launch)
    cudaError_t e = cudaFuncSetAttribute(k_compose_tile<OPD, FIELD, RAMP>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         kSmemBytes);
    if (e != cudaSuccess) return e;
    return launch_pdl(k_compose_tile<OPD, FIELD, RAMP>, dim3(a.ntx * kCtaSplit, a.nty, B), dim3(kCtaWarps * 32), (size_t)kSmemBytes, stream, a);
}

// sort_first = false: the lists of the last call are already sorted and culled (osog_debug_recompose_field)
cudaError_t launch_compose(osog_ctx* c, int B, bool has_ramp, float* d_opd, float2* d_field, bool sort_first)
{
    ComposeArgs a;
    a.rec = c->rec; a.rec2 = c->rec2; a.offset = c->offset; a.list = c->list; a.meta = c->meta;
    a.optics = c->optics;
    a.status = c->status + c->status_idx;
    a.opd = d_opd; a.field = d_field;
    a.H = c->H; a.W = c->W; a.ntx = c->ntx; a.nty = c->nty;
    a.topo_amp = (float)c->last_topo; a.seed = c->last_seed;
    const unsigned grid = (unsigned)((long long)B * c->ntx * c->nty);
    if (sort_first) {
        const cudaError_t e = launch_sort_cull(c, grid, true);
        if (e != cudaSuccess) return e;
    }
    if (d_opd != nullptr && d_field == nullptr) return launch_variant<true, false, false>(a, B, c->stream);
    if (d_opd == nullptr && !has_ramp) return launch_variant<false, true, false>(a, B, c->stream);
    if (d_opd == nullptr && has_ramp) return launch_variant<false, true, true>(a, B, c->stream);
    if (!has_ramp) return launch_variant<true, true, false>(a, B, c->stream);
    return launch_variant<true, true, true>(a, B, c->stream);
}

// ---- measured alternative: paper-style scatter-add with global atomics ----------------------------
// One warp per particle walks the particle's pixel bounding box and atomicAdd's (n_p - n_m) t into the frame (fp64
// thickness per pixel, fp32 atomics).  Summation order, hence the last bits, depend on scheduling: NOT deterministic.
// The frame must be zeroed first.
__global__ void __launch_bounds__(256) k_compose_atomic(const float* __restrict__ recs, const int4* __restrict__ tbox,
                                                        const int* __restrict__ pframe, long long N, int H, int W,
                                                        float* __restrict__ opd)
{
    const long long n = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (n >= N) return;
    if (tbox[n].x > tbox[n].y) return;
    const float4* rec = reinterpret_cast<const float4*>(recs + (size_t)n * kRecWords);
    const float4 h1 = rec[1], h2 = rec[2];
    const int4 h3 = *reinterpret_cast<const int4*>(rec + 3);
    const uint32_t bx = __float_as_uint(h1.z), by = __float_as_uint(h1.w);
    const int j0 = bx & 0xffff, j1 = bx >> 16, i0 = by & 0xffff, i1 = by >> 16;
    const uint32_t flags = __float_as_uint(h2.x);
    const double* c = reinterpret_cast<const double*>(rec + 4);
    const double K = (double)h2.y;
    const int bw = j1 - j0 + 1, np = bw * (i1 - i0 + 1);
    float* frame = opd + (size_t)pframe[n] * H * W;
    for (int q = lane; q < np; q += 32) {
        const int i = i0 + q / bw, j = j0 + q % bw;
        const double dj = (double)(j - h3.x), di = (double)(i - h3.y);
        double v;
        if (flags & kFlagPrism) {
            v = K * prism_t64(c, flags >> 16, dj, di);
        } else {
            const double w = c[5] - fma(fma(c[0], dj, fma(c[1], di, c[3])), dj, fma(c[2], di, c[4]) * di);
            v = K * (double)fast_sqrt(fmaxf((float)w, 0.0f));
        }
        const float f = (float)v;
        if (f != 0.0f) atomicAdd(&frame[(size_t)i * W + j], f);
    }
}

// ---- G-buffer extras (reading A24): depth map and instance-id map -----------------------------------
// One CTA of 8 warps per tile, warp = 16 x 8 pixel sub-tile, lane = 4 x 1 pixels (the layout of the composition).  Every
// warp walks the tile's sorted list, skips the entries whose sub-tile mask bit is clear, and for the others evaluates the
// top of the chord in fp64 straight from the record: the decision "which particle is on top" is taken in the precision
// the oracle takes it in.  Ascending list order and a strict comparison give ties to the smallest index.
// NORMAL: also the slope (dz/dx, dz/dy) of the owner's top surface (the analytic height gradient of the visible surface,
// PAPER.md:76, 92): the active exit plane's -n_x / n_z = -U / p for a prism, the derivative of the upper root of the quadric
// for an ellipsoid: d/ddj (Z0 + Zx dj + Zy di + T0 sqrt(w) / 2) / p.
constexpr int kGbCap = 512;                        // longest list that k_gbuffer_tile ranks front to back (10 KB of shared memory)
template <bool NORMAL>
__global__ void __launch_bounds__(kComposeThreads) k_gbuffer_tile(const float* __restrict__ recs, const uint32_t* __restrict__ offset,
                                                                const uint32_t* __restrict__ list, const uint16_t* __restrict__ meta,
                                                                const DeviceStatus* __restrict__ status,
                                                                const int32_t* __restrict__ frame_start, int ntx, int nty, int H,
                                                                int W, double inv_pitch, int32_t* __restrict__ top_id,
                                                                float* __restrict__ depth, float2* __restrict__ normal)
{
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int tile = blockIdx.x, tpf = ntx * nty;
    const int b = tile / tpf, rt = tile - b * tpf;
    const int ty = rt / ntx, tx = rt - ty * ntx;
    const int j = tx * kTile + (wid & 1) * 16 + (lane & 3) * 4, i = ty * kTile + (wid >> 1) * 8 + (lane >> 2);
    const uint32_t beg = offset[tile];
    const uint32_t L = (status->bits & OSOG_WOVERFLOW) ? 0u : offset[tile + 1] - beg;
    const uint32_t* glist = list + beg;
    const uint16_t* gmeta = meta + beg;
    const uint32_t first = frame_start != nullptr ? (uint32_t)frame_start[b] : 0u;
    double best[4] = {0.0, 0.0, 0.0, 0.0};
    int32_t who[4] = {-1, -1, -1, -1};
    float2 slope[4] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
    float floor_all = __int_as_float(0xff800000);                // -inf: nothing can be skipped yet
    // Front to back: the tile's entries are ranked by the upper bound cz + zmax of their tops (descending; ties in list order)
    // in shared memory, so that a warp can STOP at the first entry whose bound lies below every top it has found, instead of
    // skipping such entries one by one.  Lists longer than kGbCap keep the list order (the skip test still applies).
    __shared__ uint32_t s_pid[2][kGbCap];
    __shared__ float s_key[2][kGbCap];
    __shared__ uint16_t s_meta[2][kGbCap];
    const bool sorted = L <= (uint32_t)kGbCap;                   // CTA-uniform
    if (sorted) {
        for (uint32_t k = tid; k < L; k += kComposeThreads) {
            const uint32_t pid = glist[k];
            const float4* rec = reinterpret_cast<const float4*>(recs + (size_t)pid * kRecWords);
            const float czf = __ldg(rec + 2).z;
            const float key = czf + __int_as_float(__ldg(reinterpret_cast<const int4*>(rec + 3)).z);
            s_pid[0][k] = pid;
            s_key[0][k] = fabsf(czf) <= 3.402823466e38f ? key : __int_as_float(0xff800000);   // non-finite height: last (and skipped below)
            s_meta[0][k] = gmeta[k];
        }
        __syncthreads();
        for (uint32_t k = tid; k < L; k += kComposeThreads) {
            const float key = s_key[0][k];
            uint32_t r = 0;
            for (uint32_t q = 0; q < L; ++q) {
                const float kq = s_key[0][q];
                r += (kq > key || (kq == key && q < k)) ? 1u : 0u;
            }
            s_pid[1][r] = s_pid[0][k];
            s_key[1][r] = key;
            s_meta[1][r] = s_meta[0][k];
        }
        __syncthreads();
    }
    for (uint32_t k = 0; k < L; ++k) {
        uint32_t pid, mk;
        if (sorted) {
            if (s_key[1][k] < floor_all) break;                  // no later entry can reach any pixel of this warp
            pid = s_pid[1][k];
            mk = s_meta[1][k];
        } else {
            pid = glist[k];
            mk = gmeta[k];
        }
        if (((mk >> wid) & 1u) == 0u) continue;                  // warp-uniform
        const float4* rec = reinterpret_cast<const float4*>(recs + (size_t)pid * kRecWords);
        const float4 h2 = __ldg(rec + 2);
        const int4 h3 = __ldg(reinterpret_cast<const int4*>(rec + 3));
        const float czf = h2.z;
        if (!(fabsf(czf) <= 3.402823466e38f)) continue;          // non-finite height: no entry in the depth map
        // no point of this particle lies above cz + zmax: skip it when every pixel of the sub-tile already has a higher top
        if (czf + __int_as_float(h3.z) < floor_all) continue;
        const uint32_t flags = __float_as_uint(h2.x);
        const double* c = reinterpret_cast<const double*>(rec + 4);
        const double di = (double)(i - h3.y), dj0 = (double)(j - h3.x);
        // Bound of this particle's top over THIS sub-tile (16 x 8 pixels): a prism's top is the lowest exit plane, so it lies
        // below every exit plane's maximum over the rectangle (lanes 0..5 take one slab each); an ellipsoid's top is the chord's
        // midplane plus at most half the longest chord.  Tighter than cz + zmax wherever the sub-tile only sees the particle's flank.
        if (floor_all > __int_as_float(0xff800000)) {
            const double djc = (double)(tx * kTile + (wid & 1) * 16 - h3.x) + 7.5, dic = (double)(ty * kTile + (wid >> 1) * 8 - h3.y) + 3.5;
            double bnd;
            if (flags & kFlagPrism) {
                bnd = 1.0e300;
                if (lane < 6 && (((flags >> 16) >> lane) & 1u) == 0u) {
                    const double2 uv = *reinterpret_cast<const double2*>(c + 4 * lane);
                    bnd = c[4 * lane + 2] - uv.x * djc - uv.y * dic + 7.5 * fabs(uv.x) + 3.5 * fabs(uv.y);
                }
#pragma unroll
                for (int d = 1; d < 8; d <<= 1) bnd = fmin(bnd, __shfl_xor_sync(0xffffffffu, bnd, d));
                bnd = __shfl_sync(0xffffffffu, bnd, 0);
            } else {
                bnd = c[8] + c[9] * djc + c[10] * dic + 7.5 * fabs(c[9]) + 3.5 * fabs(c[10]) + 0.5 * c[11];
            }
            if ((double)czf + bnd + 1.0e-9 * (1.0 + fabs(bnd)) < (double)floor_all) continue;
        }
        double zx[4];
        bool hit[4];
        double sxs[4] = {0.0, 0.0, 0.0, 0.0}, sys[4] = {0.0, 0.0, 0.0, 0.0};    // slope of this particle's top (NORMAL only)
        if (flags & kFlagPrism) {
            // slab by slab for the lane's four pixels: coefficients loaded and the row term formed once per slab
            const uint32_t vmask = flags >> 16;
            double ex[4] = {1.0e300, 1.0e300, 1.0e300, 1.0e300}, en[4] = {-1.0e300, -1.0e300, -1.0e300, -1.0e300};
            bool out[4] = {false, false, false, false};
            auto slabs = [&](auto vert) {                        // vert: the prism has a vertical slab (rare; its tests leave the common code)
#pragma unroll
            for (int sl = 0; sl < 6; ++sl) {
                const double2 uv = *reinterpret_cast<const double2*>(c + 4 * sl);
                const double2 xn = *reinterpret_cast<const double2*>(c + 4 * sl + 2);
                const double r = uv.y * di;
                if (decltype(vert)::value && ((vmask >> sl) & 1u)) {   // vertical slab (warp-uniform branch)
#pragma unroll
                    for (int q = 0; q < 4; ++q) out[q] = out[q] || fabs(fma(uv.x, dj0 + (double)q, r) + xn.x) > xn.y;
                } else {
                    const double cx = xn.x - r, cn = xn.y - r;
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const double m = uv.x * (dj0 + (double)q);
                        const double e = cx - m, n = cn - m;
                        if (NORMAL && e < ex[q]) { sxs[q] = -uv.x; sys[q] = -uv.y; }    // the active exit plane so far
                        ex[q] = e < ex[q] ? e : ex[q];
                        en[q] = n > en[q] ? n : en[q];
                    }
                }
            }
            };
            if (vmask) slabs(std::true_type{}); else slabs(std::false_type{});
#pragma unroll
            for (int q = 0; q < 4; ++q) { hit[q] = !out[q] && ex[q] - en[q] > 0.0; zx[q] = ex[q]; }
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const double dj = dj0 + (double)q;
                const double w = c[5] - fma(fma(c[0], dj, fma(c[1], di, c[3])), dj, fma(c[2], di, c[4]) * di);
                hit[q] = w > 0.0;
                const double sq = sqrt(fmax(w, 0.0));
                zx[q] = fma(c[9], dj, fma(c[10], di, c[8])) + 0.5 * c[11] * sq;
                if (NORMAL && hit[q]) {
                    const double k4 = 0.25 * c[11] / sq;            // d(T0 sqrt(w) / 2) = T0 dw / (4 sqrt(w))
                    sxs[q] = c[9] - k4 * (2.0 * c[0] * dj + c[1] * di + c[3]);
                    sys[q] = c[10] - k4 * (c[1] * dj + 2.0 * c[2] * di + c[4]);
                }
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const double top = (double)czf + zx[q];
            // strictly higher, or equally high with the smaller index (front-to-back order does not visit indices ascending)
            if (hit[q] && (who[q] < 0 || top > best[q] || (top == best[q] && (int32_t)(pid - first) < who[q]))) {
                best[q] = top; who[q] = (int32_t)(pid - first);
                if (NORMAL) slope[q] = make_float2((float)(sxs[q] * inv_pitch), (float)(sys[q] * inv_pitch));
            }
        }
        // lowest top over the warp's 128 pixels, rounded down (-inf while some pixel has no owner)
        float lo = __int_as_float(0x7f800000);
#pragma unroll
        for (int q = 0; q < 4; ++q)                             // (pixels outside the frame never get an owner: they do not count)
            if (j + q < W && i < H) lo = fminf(lo, who[q] < 0 ? __int_as_float(0xff800000) : __double2float_rd(best[q]));
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, d));
        floor_all = lo - 1.0e-5f;                                // margin for the float sum cz + zmax
    }
    if (i >= H) return;
    const size_t row = ((size_t)b * H + i) * W;
#pragma unroll
    for (int q = 0; q < 4; ++q)
        if (j + q < W) {
            top_id[row + j + q] = who[q];
            depth[row + j + q] = who[q] < 0 ? 0.0f : (float)best[q];
            if (NORMAL) normal[row + j + q] = who[q] < 0 ? make_float2(0.f, 0.f) : slope[q];
        }
}

cudaError_t launch_gbuffer(osog_ctx* c, int B, const int32_t* d_frame_start, double pitch, int32_t* d_top_id, float* d_depth,
                           float* d_normal)
{
    const unsigned grid = (unsigned)((long long)B * c->ntx * c->nty);
    const cudaError_t e = launch_sort_cull(c, grid, false);
    if (e != cudaSuccess) return e;
    if (d_normal != nullptr)
        k_gbuffer_tile<true><<<grid, kComposeThreads, 0, c->stream>>>(c->rec, c->offset, c->list, c->meta, c->status + c->status_idx,
                                                                     d_frame_start, c->ntx, c->nty, c->H, c->W, 1.0 / pitch, d_top_id,
                                                                     d_depth, reinterpret_cast<float2*>(d_normal));
    else
        k_gbuffer_tile<false><<<grid, kComposeThreads, 0, c->stream>>>(c->rec, c->offset, c->list, c->meta, c->status + c->status_idx,
                                                                      d_frame_start, c->ntx, c->nty, c->H, c->W, 1.0 / pitch, d_top_id,
                                                                      d_depth, nullptr);
    return cudaGetLastError();
}

// ---- measured alternative: tile lists + shared-memory atomics (north_star's "accumulate in shared memory") -------------
// One CTA per 32 x 32 tile keeps the tile's OPD in shared memory; one warp per listed particle walks the part of the
// particle's pixel bounding box that lies in the tile and atomicAdd's (n_p - n_m) t into it (fp64 thickness per pixel, fp32
// shared-memory atomics).  The order in which the warps reach a pixel depends on scheduling: NOT deterministic in the last
// bits, and the sum is fp32.  Kept to be measured against the ordered register accumulation of k_compose_tile.
__global__ void __launch_bounds__(kComposeThreads) k_compose_smem_atomic(const float* __restrict__ recs, const uint32_t* __restrict__ offset,
                                                                       const uint32_t* __restrict__ list,
                                                                       const DeviceStatus* __restrict__ status, int ntx, int nty,
                                                                       int H, int W, float* __restrict__ opd)
{
    __shared__ float s_acc[kTile * kTile];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int tile = blockIdx.x, tpf = ntx * nty;
    const int b = tile / tpf, rt = tile - b * tpf;
    const int ty = rt / ntx, tx = rt - ty * ntx;
    const int x0 = tx * kTile, y0 = ty * kTile;
    for (int k = tid; k < kTile * kTile; k += kComposeThreads) s_acc[k] = 0.0f;
    __syncthreads();
    const uint32_t beg = offset[tile];
    const uint32_t L = (status->bits & OSOG_WOVERFLOW) ? 0u : offset[tile + 1] - beg;
    const uint32_t* glist = list + beg;
    for (uint32_t k = wid; k < L; k += kWarps) {
        const float4* rec = reinterpret_cast<const float4*>(recs + (size_t)glist[k] * kRecWords);
        const float4 h1 = __ldg(rec + 1), h2 = __ldg(rec + 2);
        const int4 h3 = __ldg(reinterpret_cast<const int4*>(rec + 3));
        const uint32_t bx = __float_as_uint(h1.z), by = __float_as_uint(h1.w);
        const int j0 = max((int)(bx & 0xffff), x0), j1 = min((int)(bx >> 16), x0 + kTile - 1);
        const int i0 = max((int)(by & 0xffff), y0), i1 = min((int)(by >> 16), y0 + kTile - 1);
        const uint32_t flags = __float_as_uint(h2.x);
        const double* c = reinterpret_cast<const double*>(rec + 4);
        const double K = (double)h2.y;
        const int bw = j1 - j0 + 1, np = bw * (i1 - i0 + 1);
        for (int q = lane; q < np; q += 32) {
            const int i = i0 + q / bw, j = j0 + q % bw;
            const double dj = (double)(j - h3.x), di = (double)(i - h3.y);
            double v;
            if (flags & kFlagPrism) {
                v = K * prism_t64(c, flags >> 16, dj, di);
            } else {
                const double w = c[5] - fma(fma(c[0], dj, fma(c[1], di, c[3])), dj, fma(c[2], di, c[4]) * di);
                v = K * (double)fast_sqrt(fmaxf((float)w, 0.0f));
            }
            const float f = (float)v;
            if (f != 0.0f) atomicAdd(&s_acc[(i - y0) * kTile + (j - x0)], f);
        }
    }
    __syncthreads();
    for (int k = tid; k < kTile * kTile; k += kComposeThreads) {
        const int i = y0 + k / kTile, j = x0 + k % kTile;
        if (i < H && j < W) opd[((size_t)b * H + i) * W + j] = s_acc[k];
    }
}

// runs k_sort_cull first (it fills the CSR list and keeps the counter / status invariants)
cudaError_t launch_compose_smem_atomic(osog_ctx* c, int B, float* d_opd)
{
    const unsigned grid = (unsigned)((long long)B * c->ntx * c->nty);
    const cudaError_t e = launch_sort_cull(c, grid, false);
    if (e != cudaSuccess) return e;
    k_compose_smem_atomic<<<grid, kComposeThreads, 0, c->stream>>>(c->rec, c->offset, c->list, c->status + c->status_idx,
                                                                  c->ntx, c->nty, c->H, c->W, d_opd);
    return cudaGetLastError();
}

// ---- first step of the backward pass: dL/dn_p[n] = sum_px G[px] t_n[px] ----------------
// The OPD sum is linear in n_p, so its adjoint in n_p is a gather: one warp per particle walks the particle's pixel
// bounding box (thickness in fp64 from the record), lane q takes pixels q, q + 32, ... in row-major order of the box and
// a shuffle tree adds the 32 partial sums: a fixed order, so the result is reproducible bit for bit.
__global__ void __launch_bounds__(256) k_backward_np(const float* __restrict__ recs, const int4* __restrict__ tbox,
                                                     const int* __restrict__ pframe, long long N, int H, int W,
                                                     const float* __restrict__ gopd, float* __restrict__ gnp)
{
    const long long n = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (n >= N) return;
    double acc = 0.0;
    if (tbox[n].x <= tbox[n].y) {                                // listed: valid and on the canvas (else the gradient is 0)
        const float4* rec = reinterpret_cast<const float4*>(recs + (size_t)n * kRecWords);
        const float4 h1 = rec[1], h2 = rec[2];
        const int4 h3 = *reinterpret_cast<const int4*>(rec + 3);
        const uint32_t bx = __float_as_uint(h1.z), by = __float_as_uint(h1.w);
        const int j0 = bx & 0xffff, j1 = bx >> 16, i0 = by & 0xffff, i1 = by >> 16;
        const uint32_t flags = __float_as_uint(h2.x);
        const double* c = reinterpret_cast<const double*>(rec + 4);
        const int bw = j1 - j0 + 1, np = bw * (i1 - i0 + 1);
        const float* g = gopd + (size_t)pframe[n] * H * W;
        int i = i0 + lane / bw, j = j0 + lane % bw;
        if (flags & kFlagPrism) {
            double2 uv[6], xn[6];                                // the record's slabs in registers for the whole walk
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                uv[q] = *reinterpret_cast<const double2*>(c + 4 * q);
                xn[q] = *reinterpret_cast<const double2*>(c + 4 * q + 2);
            }
            const uint32_t vmask = flags >> 16;
            auto walk = [&](auto vert) {                         // vert: the prism has a vertical slab (rare; its tests leave the common loop)
            for (int q = lane; q < np; q += 32) {
                const double dj = (double)(j - h3.x), di = (double)(i - h3.y);
                const double gv = (double)g[(size_t)i * W + j];
                j += 32;
                while (j > j1) { j -= bw; ++i; }
                double ex = 1.0e300, en = -1.0e300;
                bool out = false;
#pragma unroll
                for (int s = 0; s < 6; ++s) {
                    const double m = fma(uv[s].x, dj, uv[s].y * di);
                    if (decltype(vert)::value && ((vmask >> s) & 1u)) {
                        out = out || fabs(m + xn[s].x) > xn[s].y;
                    } else {
                        const double e = xn[s].x - m, f = xn[s].y - m;
                        ex = e < ex ? e : ex;
                        en = f > en ? f : en;
                    }
                }
                const double t = ex - en;
                if (!out && t > 0.0) acc = fma(gv, t, acc);
            }
            };
            if (vmask) walk(std::true_type{}); else walk(std::false_type{});
        } else {
            const double c0 = c[0], c1 = c[1], c2 = c[2], c3 = c[3], c4 = c[4], c5 = c[5], T0 = c[11];
            for (int q = lane; q < np; q += 32) {
                const double dj = (double)(j - h3.x), di = (double)(i - h3.y);
                const double gv = (double)g[(size_t)i * W + j];
                j += 32;
                while (j > j1) { j -= bw; ++i; }
                const double w = c5 - fma(fma(c0, dj, fma(c1, di, c3)), dj, fma(c2, di, c4) * di);
                acc = fma(gv, T0 * sqrt(fmax(w, 0.0)), acc);     // T0 sqrt(w)
            }
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if (lane == 0) gnp[n] = (float)acc;
}

// Second step: dL/d(cx, cy)[n] = -(n_p - n_m) sum_px G[px] grad t_n[px].  Same gather as k_backward_np; the gradient in
// um^-1 is the gradient in pixel offsets divided by the pitch.  Ellipsoid: t = T0 sqrt(w), w the record's quadratic,
// grad t = T0 grad w / (2 sqrt(w)).  record word 9 holds dn (prism) or dn T0 (ellipsoid).
__global__ void __launch_bounds__(256) k_backward_centre(const float* __restrict__ recs, const int4* __restrict__ tbox,
                                                         const int* __restrict__ pframe, long long N, int H, int W,
                                                         double inv_pitch, const float* __restrict__ gopd,
                                                         float2* __restrict__ gc)
{
    __shared__ double2 s_uv[256 / 32][6];                        // per warp: (U, V) of the prism's slabs, looked up by active-slab index
    const long long n = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (n >= N) return;
    double ax = 0.0, ay = 0.0, scale = 0.0;
    if (tbox[n].x <= tbox[n].y) {
        const float4* rec = reinterpret_cast<const float4*>(recs + (size_t)n * kRecWords);
        const float4 h1 = rec[1], h2 = rec[2];
        const int4 h3 = *reinterpret_cast<const int4*>(rec + 3);
        const uint32_t bx = __float_as_uint(h1.z), by = __float_as_uint(h1.w);
        const int j0 = bx & 0xffff, j1 = bx >> 16, i0 = by & 0xffff, i1 = by >> 16;
        const uint32_t flags = __float_as_uint(h2.x);
        const double* c = reinterpret_cast<const double*>(rec + 4);
        const int bw = j1 - j0 + 1, np = bw * (i1 - i0 + 1);
        const float* g = gopd + (size_t)pframe[n] * H * W;
        scale = -(double)h2.y * inv_pitch;                       // -dn / p  (ellipsoid: -dn T0 / p, T0 folded in below)
        int i = i0 + lane / bw, j = j0 + lane % bw;
        if (flags & kFlagPrism) {
            double2 uv[6], xn[6];                                // the record's slabs in registers for the whole walk
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                uv[q] = *reinterpret_cast<const double2*>(c + 4 * q);
                xn[q] = *reinterpret_cast<const double2*>(c + 4 * q + 2);
            }
            const uint32_t vmask = flags >> 16;
            if (lane < 6) s_uv[wid][lane] = *reinterpret_cast<const double2*>(c + 4 * lane);
            __syncwarp();
            auto walk = [&](auto vert) {                         // vert: the prism has a vertical slab (rare; its tests leave the common loop)
            for (int q = lane; q < np; q += 32) {
                const double dj = (double)(j - h3.x), di = (double)(i - h3.y);
                const double gv = (double)g[(size_t)i * W + j];
                j += 32;
                while (j > j1) { j -= bw; ++i; }
                // t = exit - enter on the active planes (arg min / arg max), exit_k = Cx_k - U_k dj - V_k di:
                // dt/ddj = -(U_e - U_f), dt/ddi = -(V_e - V_f); 0 where the chord is empty
                double ex = 1.0e300, en = -1.0e300;
                int ke = 0, kf = 0;                              // active slabs (their slopes are looked up in shared memory)
                bool out = false;
#pragma unroll
                for (int s = 0; s < 6; ++s) {
                    const double m = fma(uv[s].x, dj, uv[s].y * di);
                    if (decltype(vert)::value && ((vmask >> s) & 1u)) {
                        out = out || fabs(m + xn[s].x) > xn[s].y;
                    } else {
                        const double e = xn[s].x - m, f = xn[s].y - m;
                        if (e < ex) { ex = e; ke = s; }
                        if (f > en) { en = f; kf = s; }
                    }
                }
                if (!out && ex - en > 0.0) {
                    const double2 se = s_uv[wid][ke], sf = s_uv[wid][kf];
                    ax = fma(gv, sf.x - se.x, ax);
                    ay = fma(gv, sf.y - se.y, ay);
                }
            }
            };
            if (vmask) walk(std::true_type{}); else walk(std::false_type{});
        } else {
            const double c0 = c[0], c1 = c[1], c2 = c[2], c3 = c[3], c4 = c[4], c5 = c[5];
            for (int q = lane; q < np; q += 32) {
                const double dj = (double)(j - h3.x), di = (double)(i - h3.y);
                const double gv = (double)g[(size_t)i * W + j];
                j += 32;
                while (j > j1) { j -= bw; ++i; }
                const double w = c5 - fma(fma(c0, dj, fma(c1, di, c3)), dj, fma(c2, di, c4) * di);
                const double r = w > 0.0 ? 0.5 * rsqrt(w) : 0.0;  // (the record's K = dn T0 supplies T0)
                ax = fma(gv, -(2.0 * c0 * dj + c1 * di + c3) * r, ax);
                ay = fma(gv, -(c1 * dj + 2.0 * c2 * di + c4) * r, ay);
            }
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        ax += __shfl_xor_sync(0xffffffffu, ax, d);
        ay += __shfl_xor_sync(0xffffffffu, ay, d);
    }
    if (lane == 0) gc[n] = make_float2((float)(scale * ax), (float)(scale * ay));
}

// ---- third step of the backward pass: dL/d(d0, d1, d2, qw, qx, qy, qz)[n] =
// (n_p - n_m) sum_px G[px] dt_n/dtheta[px].  The shape parameters enter through the rotation and the body's planes / quadric,
// which the derived record no longer shows, so this kernel works from the particle columns themselves, all in fp64:
//   ellipsoid: M = R D R^T; per parameter dM = dR D R^T + R dD R^T + R D dR^T (once per particle); per pixel
//              disc = Bq^2 - A C, t = 2 sqrt(disc) / A, dt = d(disc) / (A sqrt(disc)) - 2 sqrt(disc) dA / A^2;
//   prism:     per pixel the active exit / entry planes e, f of the 12 world planes (arg min / arg max of
//              z_k = (b_k - n_x dx - n_y dy) / n_z); dz_k = (db_k - dn_x dx - dn_y dy - z_k dn_z) / n_z with
//              dn = dR n_hat (rotation) or R dn_hat (dimensions); dt = dz_e - dz_f.
// Same gather as k_backward_np: one warp per particle over its pixel bounding box, fixed order (reproducible bits).
struct ParamGradArgs {
    const float *cx, *cy, *qw, *qx, *qy, *qz, *d0, *d1, *d2, *n_p;
    const uint8_t* kind;
    const float* recs;
    const int4* tbox;
    const int* pframe;
    long long N;
    int H, W;
    double pitch, n_medium;
    const float* gopd;
    float* gpar;                  // [N][7], or nullptr
    float* gnp;                   // [N] dL/dn_p, or nullptr    (osog_backward_particles: the same moments give all three)
    float2* gc;                   // [N] dL/d(cx, cy), or nullptr
};

// body-frame plane k of the capped prism (0, 1: +-x; 2, 3: +-y; 4..7: (+-hc, 0, +-s/2); 8..11: (0, +-hc, +-s/2)) and its
// derivatives in (s, L, hc)
__device__ __forceinline__ void prism_plane(int k, double s, double L, double hc, double nb[3], double* b, double dnb[3][3], double db[3])
{
#pragma unroll
    for (int p = 0; p < 3; ++p) { db[p] = 0.0; dnb[p][0] = dnb[p][1] = dnb[p][2] = 0.0; }
    nb[0] = nb[1] = nb[2] = 0.0;
    if (k < 4) {
        nb[k >> 1] = (k & 1) ? -1.0 : 1.0;
        *b = 0.5 * s;
        db[0] = 0.5;
        return;
    }
    const int lat = k < 8 ? 0 : 1;                 // lateral component that carries +-hc
    const int kk = (k - 4) & 3;
    const double sl = (kk & 1) ? -1.0 : 1.0, sz = (kk & 2) ? -1.0 : 1.0;
    nb[lat] = sl * hc;
    nb[2] = sz * 0.5 * s;
    *b = hc * s * 0.5 + s * L * 0.25;
    db[0] = 0.5 * hc + 0.25 * L; db[1] = 0.25 * s; db[2] = 0.5 * s;
    dnb[2][lat] = sl;                              // d / dhc
    dnb[0][2] = sz * 0.5;                          // d / ds
}

// The per-pixel derivative is LINEAR in a few per-pixel quantities, so the pixel loop only accumulates moments and the
// seven parameters are formed once per particle:
//   prism, pixel with active exit plane e and entry plane f:  dz_k/dtheta = (db_k - dn_x dx - dn_y dy - z_k dn_z) / n_z, so
//     sum_px G dt/dtheta = sum_k sgn_k (db_k S0_k - dn_x Sx_k - dn_y Sy_k - dn_z Sz_k) / n_z,k  with the moments
//     (S0, Sx, Sy)_k = sum over the pixels where plane k is active of G (1, dx, dy), Sz_k = zc_k S0_k - za_k Sx_k - zb_k Sy_k,
//     sgn = +1 for exit planes (n_z > 0), -1 for entry planes.  36 moments per lane, in shared memory (lane-private columns).
//   ellipsoid, w = G / sqrt(disc):  sum_px G dt/dtheta = (2 <Bq dBq> - dA <C> - A <dC>) / A - 2 dA sum(G sqrt(disc)) / A^2,
//     <.> = sum_px w (.), every bracket a quadratic form in (dx, dy): moments sum w (1, dx^2, dx dy, dy^2) and sum G sqrt(disc).
constexpr int kPgThreads = 128;
__global__ void __launch_bounds__(kPgThreads, 4) k_backward_params(const ParamGradArgs a)
{
    __shared__ double s_mom[kPgThreads / 32][36][32];            // prism moments: [plane * 3 + (0, x, y)][lane]
    const long long n = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (n >= a.N) return;
    double acc[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    double gt = 0.0, gcx = 0.0, gcy = 0.0;          // sum G t, sum G dt/dcx, sum G dt/dcy
    double dn_idx = 0.0;
    if (a.tbox[n].x <= a.tbox[n].y) {              // listed: valid and on the canvas (else the gradient is 0)
        const float4* rec = reinterpret_cast<const float4*>(a.recs + (size_t)n * kRecWords);
        const float4 h1 = rec[1];
        const uint32_t bx = __float_as_uint(h1.z), by = __float_as_uint(h1.w);
        const int j0 = bx & 0xffff, j1 = bx >> 16, i0 = by & 0xffff, i1 = by >> 16;
        const int bw = j1 - j0 + 1, np = bw * (i1 - i0 + 1);
        const float* g = a.gopd + (size_t)a.pframe[n] * a.H * a.W;
        const double cx = a.cx[n], cy = a.cy[n], w = a.qw[n], x = a.qx[n], y = a.qy[n], z = a.qz[n];
        const double e[3] = {(double)a.d0[n], (double)a.d1[n], (double)a.d2[n]};
        dn_idx = (double)a.n_p[n] - a.n_medium;
        const double R[9] = {1.0 - 2.0 * (y * y + z * z), 2.0 * (x * y - w * z), 2.0 * (x * z + w * y),
                             2.0 * (x * y + w * z), 1.0 - 2.0 * (x * x + z * z), 2.0 * (y * z - w * x),
                             2.0 * (x * z - w * y), 2.0 * (y * z + w * x), 1.0 - 2.0 * (x * x + y * y)};
        const double dR[4][9] = {{0.0, -2.0 * z, 2.0 * y, 2.0 * z, 0.0, -2.0 * x, -2.0 * y, 2.0 * x, 0.0},
                                 {0.0, 2.0 * y, 2.0 * z, 2.0 * y, -4.0 * x, -2.0 * w, 2.0 * z, 2.0 * w, -4.0 * x},
                                 {-4.0 * y, 2.0 * x, 2.0 * w, 2.0 * x, 0.0, 2.0 * z, -2.0 * w, 2.0 * z, -4.0 * y},
                                 {-4.0 * z, -2.0 * w, 2.0 * x, 2.0 * w, -4.0 * z, 2.0 * y, 2.0 * x, 2.0 * y, 0.0}};
        if (a.kind[n] == 0u) {
            const double D[3] = {1.0 / (e[0] * e[0]), 1.0 / (e[1] * e[1]), 1.0 / (e[2] * e[2])};
            // symmetric 3 x 3 as (xx, xy, yy, xz, yz, zz)
            const int ra[6] = {0, 0, 1, 0, 1, 2}, rb[6] = {0, 1, 1, 2, 2, 2};
            double M[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) {
                M[c] = 0.0;
#pragma unroll
                for (int k = 0; k < 3; ++k) M[c] += R[3 * ra[c] + k] * D[k] * R[3 * rb[c] + k];
            }
            double m0 = 0.0, mxx = 0.0, mxy = 0.0, myy = 0.0, ms = 0.0, mx = 0.0, my = 0.0;
            int i = i0 + lane / bw, j = j0 + lane % bw;
            for (int q = lane; q < np; q += 32) {
                const double dx = (j + 0.5) * a.pitch - cx, dy = (i + 0.5) * a.pitch - cy;
                const double gv = (double)g[(size_t)i * a.W + j];
                j += 32;
                while (j > j1) { j -= bw; ++i; }
                const double A = M[5], Bq = M[3] * dx + M[4] * dy, C = M[0] * dx * dx + 2.0 * M[1] * dx * dy + M[2] * dy * dy - 1.0;
                const double disc = Bq * Bq - A * C;
                if (!(disc > 0.0)) continue;
                const double sq = sqrt(disc);
                const double wq = gv / sq;
                m0 += wq;
                mxx = fma(wq, dx * dx, mxx);
                mxy = fma(wq, dx * dy, mxy);
                myy = fma(wq, dy * dy, myy);
                ms = fma(gv, sq, ms);
                mx = fma(wq, dx, mx);
                my = fma(wq, dy, my);
            }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                m0 += __shfl_xor_sync(0xffffffffu, m0, d);
                mxx += __shfl_xor_sync(0xffffffffu, mxx, d);
                mxy += __shfl_xor_sync(0xffffffffu, mxy, d);
                myy += __shfl_xor_sync(0xffffffffu, myy, d);
                ms += __shfl_xor_sync(0xffffffffu, ms, d);
                mx += __shfl_xor_sync(0xffffffffu, mx, d);
                my += __shfl_xor_sync(0xffffffffu, my, d);
            }
            const double A = M[5], iA = 1.0 / A;
            const double qC = M[0] * mxx + 2.0 * M[1] * mxy + M[2] * myy - m0;                       // <C>
            // t = 2 sqrt(disc) / A;  d(disc)/dcx = -2 M_xz Bq + 2 A (M_xx dx + M_xy dy)  (dx = x - cx)
            const double qB = M[3] * mx + M[4] * my;                                                 // <Bq>
            gt = 2.0 * ms * iA;
            gcx = 2.0 * (A * (M[0] * mx + M[1] * my) - M[3] * qB) * iA;
            gcy = 2.0 * (A * (M[1] * mx + M[2] * my) - M[4] * qB) * iA;
#pragma unroll
            for (int p = 0; p < 7; ++p) {
                double dM[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) {
                    if (p < 3) {
                        dM[c] = R[3 * ra[c] + p] * (-2.0 * D[p] / e[p]) * R[3 * rb[c] + p];
                    } else {
                        double v = 0.0;
#pragma unroll
                        for (int k = 0; k < 3; ++k)
                            v += (dR[p - 3][3 * ra[c] + k] * R[3 * rb[c] + k] + R[3 * ra[c] + k] * dR[p - 3][3 * rb[c] + k]) * D[k];
                        dM[c] = v;
                    }
                }
                const double qBdB = M[3] * dM[3] * mxx + (M[3] * dM[4] + M[4] * dM[3]) * mxy + M[4] * dM[4] * myy;   // <Bq dBq>
                const double qdC = dM[0] * mxx + 2.0 * dM[1] * mxy + dM[2] * myy;                                      // <dC>
                acc[p] = (2.0 * qBdB - dM[5] * qC - A * qdC) * iA - 2.0 * dM[5] * ms * iA * iA;
            }
        } else {
            // The 12 planes are 6 centrally symmetric slabs (A, B = -A): with u = n_x / n_z, v = n_y / n_z, c = b / |n_z| of plane A,
            // the slab's exit plane is z = c - u dx - v dy and its entry plane z = -c - u dx - v dy (exit = A iff n_z > 0).
            // Vertical slab (n_z = 0): inside iff |n_x dx + n_y dy| <= b.
            const int slabA[6] = {0, 2, 4, 5, 8, 9};
            double su[6], sv[6], sc[6];
            uint32_t vmask = 0u;
#pragma unroll
            for (int sl = 0; sl < 6; ++sl) {
                double nb[3], bk, dnb[3][3], db[3];
                prism_plane(slabA[sl], e[0], e[1], e[2], nb, &bk, dnb, db);
                const double nx = R[0] * nb[0] + R[1] * nb[1] + R[2] * nb[2], ny = R[3] * nb[0] + R[4] * nb[1] + R[5] * nb[2];
                const double nz = R[6] * nb[0] + R[7] * nb[1] + R[8] * nb[2];
                if (nz == 0.0) { vmask |= 1u << sl; su[sl] = nx; sv[sl] = ny; sc[sl] = bk; }
                else { const double inz = 1.0 / nz; su[sl] = nx * inz; sv[sl] = ny * inz; sc[sl] = bk * fabs(inz); }
            }
            double (*mom)[32] = s_mom[wid];                       // [(slab * 2 + (exit, entry)) * 3 + (0, x, y)][lane]
#pragma unroll
            for (int m = 0; m < 36; ++m) mom[m][lane] = 0.0;
            int i = i0 + lane / bw, j = j0 + lane % bw;
            auto walk = [&](auto vert) {                         // vert: the prism has a vertical slab (rare)
            for (int q = lane; q < np; q += 32) {
                const double dx = (j + 0.5) * a.pitch - cx, dy = (i + 0.5) * a.pitch - cy;
                const double gv = (double)g[(size_t)i * a.W + j];
                j += 32;
                while (j > j1) { j -= bw; ++i; }
                double ex = 1.0e300, en = -1.0e300;
                int ke = 0, kf = 0;
                bool out = false;
#pragma unroll
                for (int sl = 0; sl < 6; ++sl) {
                    const double m = fma(su[sl], dx, sv[sl] * dy);
                    if (decltype(vert)::value && ((vmask >> sl) & 1u)) {
                        out = out || fabs(m) > sc[sl];
                    } else {
                        const double ze = sc[sl] - m, zn = -sc[sl] - m;
                        if (ze < ex) { ex = ze; ke = sl; }
                        if (zn > en) { en = zn; kf = sl; }
                    }
                }
                if (out || !(ex - en > 0.0)) continue;
                const double gx = gv * dx, gy = gv * dy;
                double* me = &mom[6 * ke][lane];
                double* mf = &mom[6 * kf + 3][lane];
                me[0] += gv; me[32] += gx; me[64] += gy;
                mf[0] += gv; mf[32] += gx; mf[64] += gy;
            }
            };
            if (vmask) walk(std::true_type{}); else walk(std::false_type{});
            __syncwarp();
            // the 36 moments summed over the lanes (shuffle tree: a fixed order), then the parameters, slab by slab
#pragma unroll
            for (int sl = 0; sl < 6; ++sl) {
                double S[6];
#pragma unroll
                for (int m = 0; m < 6; ++m) {
                    S[m] = mom[6 * sl + m][lane];
#pragma unroll
                    for (int d = 16; d > 0; d >>= 1) S[m] += __shfl_xor_sync(0xffffffffu, S[m], d);
                }
                if ((vmask >> sl) & 1u) continue;                // vertical slabs bound the silhouette only
                double nb[3], bk, dnb[3][3], db[3];
                prism_plane(slabA[sl], e[0], e[1], e[2], nb, &bk, dnb, db);
                const double nz = R[6] * nb[0] + R[7] * nb[1] + R[8] * nb[2];
                const double sg = nz > 0.0 ? 1.0 : -1.0, ianz = 1.0 / fabs(nz);
                const double Sze = sc[sl] * S[0] - su[sl] * S[1] - sv[sl] * S[2];      // sum G z over the exit set
                const double Szf = -sc[sl] * S[3] - su[sl] * S[4] - sv[sl] * S[5];     // ... over the entry set
                gt += Sze - Szf;                                  // t = z_exit - z_entry
                gcx = fma(su[sl], S[0] - S[3], gcx);              // dz/dcx = +u for both planes of the slab (dx = x - cx)
                gcy = fma(sv[sl], S[0] - S[3], gcy);
#pragma unroll
                for (int p = 0; p < 7; ++p) {
                    double dnx, dny, dnz, dbk;                   // derivatives of plane A's normal and offset
                    if (p < 3) {
                        dbk = db[p];
                        dnx = R[0] * dnb[p][0] + R[1] * dnb[p][1] + R[2] * dnb[p][2];
                        dny = R[3] * dnb[p][0] + R[4] * dnb[p][1] + R[5] * dnb[p][2];
                        dnz = R[6] * dnb[p][0] + R[7] * dnb[p][1] + R[8] * dnb[p][2];
                    } else {
                        dbk = 0.0;
                        const double* d = dR[p - 3];
                        dnx = d[0] * nb[0] + d[1] * nb[1] + d[2] * nb[2];
                        dny = d[3] * nb[0] + d[4] * nb[1] + d[5] * nb[2];
                        dnz = d[6] * nb[0] + d[7] * nb[1] + d[8] * nb[2];
                    }
                    // exit plane E = sg A (n_E,z = |n_z|):  sum G dz_E = (db S0 - sg Xe) / |n_z|;  entry plane F = -sg A (n_F,z = -|n_z|):
                    // -sum G dz_F = (db S0' + sg Xf) / |n_z|
                    const double Xe = dnx * S[1] + dny * S[2] + dnz * Sze, Xf = dnx * S[4] + dny * S[5] + dnz * Szf;
                    acc[p] = fma(dbk * (S[0] + S[3]) + sg * (Xf - Xe), ianz, acc[p]);
                }
            }
        }
    }
    if (lane == 0) {
        if (a.gpar != nullptr) {
#pragma unroll
            for (int p = 0; p < 7; ++p) a.gpar[(size_t)n * 7 + p] = (float)(dn_idx * acc[p]);
        }
        if (a.gnp != nullptr) a.gnp[n] = (float)gt;
        if (a.gc != nullptr) a.gc[n] = make_float2((float)(dn_idx * gcx), (float)(dn_idx * gcy));
    }
}

cudaError_t launch_backward_params(osog_ctx* c, const osog_particles* p, long long N, double pitch, double n_medium,
                                   const float* d_gopd, float* d_gpar, float* d_gnp, float* d_gc)
{
    if (N == 0) return cudaSuccess;
    ParamGradArgs a;
    a.cx = p->cx; a.cy = p->cy; a.qw = p->qw; a.qx = p->qx; a.qy = p->qy; a.qz = p->qz;
    a.d0 = p->d0; a.d1 = p->d1; a.d2 = p->d2; a.n_p = p->n_p; a.kind = p->kind;
    a.recs = c->rec; a.tbox = c->tbox; a.pframe = c->pframe; a.N = N; a.H = c->H; a.W = c->W;
    a.pitch = pitch; a.n_medium = n_medium; a.gopd = d_gopd; a.gpar = d_gpar;
    a.gnp = d_gnp; a.gc = reinterpret_cast<float2*>(d_gc);
    const long long threads = N * 32;
    k_backward_params<<<(unsigned)((threads + kPgThreads - 1) / kPgThreads), kPgThreads, 0, c->stream>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_backward_centre(osog_ctx* c, long long N, double pitch, const float* d_gopd, float* d_gc)
{
    if (N == 0) return cudaSuccess;
    const long long threads = N * 32;
    k_backward_centre<<<(unsigned)((threads + 255) / 256), 256, 0, c->stream>>>(c->rec, c->tbox, c->pframe, N, c->H, c->W,
                                                                               1.0 / pitch, d_gopd,
                                                                               reinterpret_cast<float2*>(d_gc));
    return cudaGetLastError();
}

cudaError_t launch_backward_np(osog_ctx* c, long long N, const float* d_gopd, float* d_gnp)
{
    if (N == 0) return cudaSuccess;
    const long long threads = N * 32;
    k_backward_np<<<(unsigned)((threads + 255) / 256), 256, 0, c->stream>>>(c->rec, c->tbox, c->pframe, N, c->H, c->W, d_gopd,
                                                                           d_gnp);
    return cudaGetLastError();
}

cudaError_t launch_compose_atomic(osog_ctx* c, long long N, int B, float* d_opd)
{
    cudaError_t e = cudaMemsetAsync(d_opd, 0, sizeof(float) * (size_t)B * c->H * c->W, c->stream);
    if (e != cudaSuccess || N == 0) return e;
    const long long threads = N * 32;
    k_compose_atomic<<<(unsigned)((threads + 255) / 256), 256, 0, c->stream>>>(c->rec, c->tbox, c->pframe, N, c->H, c->W,
                                                                              d_opd);
    return cudaGetLastError();
}

}  // namespace osog
