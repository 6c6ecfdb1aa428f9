// Microbenchmark of per-SM instruction issue rates on B200: the measured denominators of the ALU roofline that bench.py
// reports for k_compose_tile (results in profiles/r2_issue_rates.md).  Not part of libosog.so.
//     python -m paper_2606_21381_b200.build --issue-rates      (builds paper_2606_21381_b200/issue_rates)
//     ./paper_2606_21381_b200/issue_rates
// Each kernel: 1 CTA of NT threads per SM, every thread runs 2000 iterations of 64 inline-PTX ops on 8 independent register
// chains whose operands come from the other chains (so ptxas can neither fold nor drop them; the SASS mix of every
// kernel was checked with cuobjdump); cycles from clock64 around the loop (max over CTAs).  Output: thread-ops / clk / SM
// and warp-instructions / clk / SM sub-partition.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#include <cuda_runtime.h>

#define REP8(X) X(0) X(1) X(2) X(3) X(4) X(5) X(6) X(7)

struct Out { unsigned long long cyc; };

#define KERNEL_BEGIN(NAME)                                                                                   \
    __global__ void __launch_bounds__(1024, 1) NAME(Out* out, float* sink, int iters, float fb, float fc, double db, double dc, int ib) { \
        const unsigned long long lb = 0x3f8000013f800001ull, lc = 0x3f0000003f000000ull; float a[8]; double d[8]; unsigned long long l[8]; int n[8]; float m[8];                                         \
        for (int i = 0; i < 8; ++i) { a[i] = threadIdx.x * 1e-3f + i; d[i] = a[i]; l[i] = threadIdx.x + i; n[i] = threadIdx.x + i; m[i] = a[i] * 0.5f; }  \
        __shared__ float4 sm4[64]; if (threadIdx.x < 64) sm4[threadIdx.x] = make_float4(fb, fc, fb, fc); __syncthreads();   \
        const unsigned sbase = (unsigned)__cvta_generic_to_shared(sm4);                                      \
        (void)sbase; (void)m;                                                                                \
        long long t0 = clock64();                                                                            \
        for (int it = 0; it < iters; ++it) {
#define KERNEL_END                                                                                           \
        }                                                                                                    \
        long long t1 = clock64();                                                                            \
        float s = 0; for (int i = 0; i < 8; ++i) s += a[i] + (float)d[i] + (float)l[i] + (float)n[i] + m[i];             \
        if (s == 1234.5678f) sink[0] = s;                                                                    \
        if (threadIdx.x == 0) out[blockIdx.x].cyc = (unsigned long long)(t1 - t0);                           \
    }

#define X8(OPM) REP8(OPM) REP8(OPM) REP8(OPM) REP8(OPM) REP8(OPM) REP8(OPM) REP8(OPM) REP8(OPM)

#define OP_FFMA(i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(fb), "f"(fc));
#define OP_FFMA3R(i) asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(a[i]) : "f"(a[(i + 1) & 7]), "f"(a[(i + 3) & 7]));
#define OP_FFMA2ACC(i) asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(l[i]) : "l"(lb), "l"(lc));
#define OP_FMUL(i) asm volatile("mul.rn.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(fb));
#define OP_FADD(i) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(fc));
#define OP_FADDSAT(i) asm volatile("add.sat.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(fc));
#define OP_FFMA2(i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[i]) : "l"(l[(i + 1) & 7]), "l"(l[(i + 2) & 7]));
#define OP_FADD2(i) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(l[i]) : "l"(l[(i + 1) & 7]));
#define OP_FMNMX(i) asm volatile("min.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(a[(i + 1) & 7]));
#define OP_FMNMX3(i) asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(a[(i + 1) & 7]), "f"(a[(i + 2) & 7]));
#define OP_DFMA(i) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[i]) : "d"(db), "d"(dc));
#define OP_DADD(i) asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(d[i]) : "d"(dc));
#define OP_F2F_32_64(i) { float t; asm volatile("cvt.rn.f32.f64 %0, %1;" : "=f"(t) : "d"(d[i])); asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(t)); asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(d[i]) : "d"(dc)); }
#define OP_F2F_64_32(i) { double t; asm volatile("cvt.f64.f32 %0, %1;" : "=d"(t) : "f"(a[i])); asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(d[i]) : "d"(t)); asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(fc)); }
#define OP_SQRT(i) asm volatile("sqrt.approx.ftz.f32 %0, %0;" : "+f"(a[i]));
#define OP_RSQRT(i) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(a[i]));
#define OP_IADD(i) asm volatile("add.s32 %0, %0, %1;" : "+r"(n[i]) : "r"(n[(i + 1) & 7]));
#define OP_LOP(i) asm volatile("xor.b32 %0, %0, %1;" : "+r"(n[i]) : "r"(n[(i + 1) & 7]));
#define OP_SHF(i) asm volatile("shf.l.wrap.b32 %0, %0, %1, %2;" : "+r"(n[i]) : "r"(n[(i + 1) & 7]), "r"(ib));
#define OP_IMAD(i) asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(n[i]) : "r"(ib), "r"(n[(i + 1) & 7]));
#define OP_I2F(i) { float t; asm volatile("cvt.rn.f32.s32 %0, %1;" : "=f"(t) : "r"(n[i])); asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(t)); asm volatile("add.s32 %0, %0, %1;" : "+r"(n[i]) : "r"(n[(i + 1) & 7])); }
#define OP_F2I(i) { int t; asm volatile("cvt.rzi.s32.f32 %0, %1;" : "=r"(t) : "f"(a[i])); asm volatile("add.s32 %0, %0, %1;" : "+r"(n[i]) : "r"(t)); asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(fc)); }
#define OP_IMNMX(i) asm volatile("max.s32 %0, %0, %1;" : "+r"(n[i]) : "r"(n[(i + 1) & 7]));
#define OP_LDS128(i) { float x, y, z, w; asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(x), "=f"(y), "=f"(z), "=f"(w) : "r"(sbase + 16u * ((i + it) & 63))); a[i] += x; }
#define OP_LDS32(i) { float x; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x) : "r"(sbase + 4u * ((i + it) & 63))); a[i] += x; }
// mixes: even slots one op, odd slots another (independent chains: a[] vs m[] / d[] / l[])
#define OP_MIX_FFMA2_FMNMX3(i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[i]) : "l"(l[(i + 1) & 7]), "l"(l[(i + 2) & 7])); asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(a[(i + 1) & 7]), "f"(a[(i + 2) & 7]));
#define OP_MIX_FFMA_FMNMX(i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(m[i]) : "f"(fb), "f"(fc)); asm volatile("min.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(a[(i + 1) & 7]));
#define OP_MIX_FFMA_DFMA(i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(m[i]) : "f"(fb), "f"(fc)); asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[i]) : "d"(db), "d"(dc));
#define OP_MIX_FFMA_IADD(i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(m[i]) : "f"(fb), "f"(fc)); asm volatile("add.s32 %0, %0, %1;" : "+r"(n[i]) : "r"(n[(i + 1) & 7]));
#define OP_MIX_FMNMX_IADD(i) asm volatile("min.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(a[(i + 1) & 7])); asm volatile("add.s32 %0, %0, %1;" : "+r"(n[i]) : "r"(n[(i + 1) & 7]));
#define OP_MIX_FFMA_SQRT7(i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(m[i]) : "f"(fb), "f"(fc)); if (i == 0) asm volatile("sqrt.approx.ftz.f32 %0, %0;" : "+f"(a[0]));
#define OP_MIX_FFMA2_FFMA(i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[i]) : "l"(l[(i + 1) & 7]), "l"(l[(i + 2) & 7])); asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(m[i]) : "f"(fb), "f"(fc));
#define OP_MIX_FMNMX_DFMA(i) asm volatile("min.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(a[(i + 1) & 7])); asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[i]) : "d"(db), "d"(dc));
// the shape of the planned prism inner loop per pixel: 6 FFMA2, 4 FMNMX3, 2 FMNMX, 1 FADD.SAT, 1 FFMA  (14 instr)
#define OP_PRISMPX(i) \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[0]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[1]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[2]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[3]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[4]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[5]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("min.f32 %0, %1, %2, %3;" : "=f"(a[0]) : "f"(m[0]), "f"(m[1]), "f"(m[2])); \
    asm volatile("min.f32 %0, %1, %2, %3;" : "=f"(a[1]) : "f"(m[3]), "f"(m[4]), "f"(m[5])); \
    asm volatile("max.f32 %0, %1, %2, %3;" : "=f"(a[2]) : "f"(m[0]), "f"(m[1]), "f"(m[2])); \
    asm volatile("max.f32 %0, %1, %2, %3;" : "=f"(a[3]) : "f"(m[3]), "f"(m[4]), "f"(m[5])); \
    asm volatile("min.f32 %0, %1, %2;" : "=f"(a[4]) : "f"(a[0]), "f"(a[1])); \
    asm volatile("max.f32 %0, %1, %2;" : "=f"(a[5]) : "f"(a[2]), "f"(a[3])); \
    asm volatile("sub.sat.f32 %0, %1, %2;" : "=f"(a[6]) : "f"(a[4]), "f"(a[5])); \
    asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(a[7]) : "f"(a[6]), "f"(fb));
// the current prism inner loop per pixel: 6 FFMA2, 4 FMNMX3, 2 FMNMX, FADD, FMNMX, SHF+IADD+SHF (f2d), DFMA (18 instr)
#define OP_PRISMPX_OLD(i) \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[0]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[1]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[2]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[3]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[4]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(l[5]) : "l"(l[6]), "l"(l[7])); \
    asm volatile("min.f32 %0, %1, %2, %3;" : "=f"(a[0]) : "f"(m[0]), "f"(m[1]), "f"(m[2])); \
    asm volatile("min.f32 %0, %1, %2, %3;" : "=f"(a[1]) : "f"(m[3]), "f"(m[4]), "f"(m[5])); \
    asm volatile("max.f32 %0, %1, %2, %3;" : "=f"(a[2]) : "f"(m[0]), "f"(m[1]), "f"(m[2])); \
    asm volatile("max.f32 %0, %1, %2, %3;" : "=f"(a[3]) : "f"(m[3]), "f"(m[4]), "f"(m[5])); \
    asm volatile("min.f32 %0, %1, %2;" : "=f"(a[4]) : "f"(a[0]), "f"(a[1])); \
    asm volatile("max.f32 %0, %1, %2;" : "=f"(a[5]) : "f"(a[2]), "f"(a[3])); \
    asm volatile("sub.rn.f32 %0, %1, %2;" : "=f"(a[6]) : "f"(a[4]), "f"(a[5])); \
    asm volatile("max.f32 %0, %0, %1;" : "+f"(a[6]) : "f"(fc)); \
    asm volatile("shf.r.wrap.b32 %0, %1, %2, %3;" : "=r"(n[0]) : "r"(__float_as_int(a[6])), "r"(ib), "r"(ib)); \
    asm volatile("add.s32 %0, %0, %1;" : "+r"(n[0]) : "r"(ib)); \
    asm volatile("shf.l.wrap.b32 %0, %1, %2, %3;" : "=r"(n[1]) : "r"(__float_as_int(a[6])), "r"(ib), "r"(ib)); \
    asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(d[0]) : "d"(__hiloint2double(n[0], n[1])), "d"(db));

#define DEF(NAME, OPM) KERNEL_BEGIN(NAME) X8(OPM) KERNEL_END
DEF(k_ffma, OP_FFMA) DEF(k_ffma3r, OP_FFMA3R) DEF(k_ffma2acc, OP_FFMA2ACC) DEF(k_fmul, OP_FMUL) DEF(k_fadd, OP_FADD) DEF(k_faddsat, OP_FADDSAT) DEF(k_ffma2, OP_FFMA2) DEF(k_fadd2, OP_FADD2)
DEF(k_fmnmx, OP_FMNMX) DEF(k_fmnmx3, OP_FMNMX3) DEF(k_dfma, OP_DFMA) DEF(k_dadd, OP_DADD) DEF(k_f2f3264, OP_F2F_32_64)
DEF(k_f2f6432, OP_F2F_64_32) DEF(k_sqrt, OP_SQRT) DEF(k_rsqrt, OP_RSQRT) DEF(k_iadd, OP_IADD) DEF(k_lop, OP_LOP) DEF(k_shf, OP_SHF)
DEF(k_imad, OP_IMAD) DEF(k_i2f, OP_I2F) DEF(k_f2i, OP_F2I) DEF(k_imnmx, OP_IMNMX) DEF(k_lds128, OP_LDS128) DEF(k_lds32, OP_LDS32)
DEF(k_mix_ffma2_fmnmx3, OP_MIX_FFMA2_FMNMX3) DEF(k_mix_ffma_fmnmx, OP_MIX_FFMA_FMNMX) DEF(k_mix_ffma_dfma, OP_MIX_FFMA_DFMA)
DEF(k_mix_ffma_iadd, OP_MIX_FFMA_IADD) DEF(k_mix_fmnmx_iadd, OP_MIX_FMNMX_IADD) DEF(k_mix_ffma_sqrt7, OP_MIX_FFMA_SQRT7)
DEF(k_mix_ffma2_ffma, OP_MIX_FFMA2_FFMA) DEF(k_mix_fmnmx_dfma, OP_MIX_FMNMX_DFMA)

typedef void (*kern_t)(Out*, float*, int, float, float, double, double, int);
struct Case { const char* name; kern_t k; int ops_per_iter; const char* note; };

int main(int argc, char** argv)
{
    int dev = 0; cudaSetDevice(dev);
    cudaDeviceProp prop; cudaGetDeviceProperties(&prop, dev);
    const int nsm = prop.multiProcessorCount;
    int iters = 2000;
    Out* d_out; float* d_sink;
    cudaMalloc(&d_out, sizeof(Out) * nsm); cudaMalloc(&d_sink, 16);
    std::vector<Out> h(nsm);
    Case cases[] = {
        {"FFMA", k_ffma, 64, "fma.rn.f32 d=d*b+c, b c loop-invariant"}, {"FFMA 3 regs", k_ffma3r, 64, "d=a*b+d, a b other chains"}, {"FFMA2 acc", k_ffma2acc, 64, "d=a*b+d, a b loop-invariant (instr)"}, {"FMUL", k_fmul, 64, ""}, {"FADD", k_fadd, 64, ""}, {"FADD.SAT", k_faddsat, 64, "add.sat.f32"},
        {"FFMA2", k_ffma2, 64, "fma.rn.f32x2 (instr; x2 for FMAs)"}, {"FADD2", k_fadd2, 64, "add.rn.f32x2 (instr)"},
        {"FMNMX", k_fmnmx, 64, "min.f32"}, {"FMNMX3", k_fmnmx3, 64, "3-input min.f32"}, {"DFMA", k_dfma, 64, ""}, {"DADD", k_dadd, 64, ""},
        {"F2F.F32.F64 (+FADD+DADD)", k_f2f3264, 64, "rate in F2F"}, {"F2F.F64.F32 (+DADD+FADD)", k_f2f6432, 64, "rate in F2F"},
        {"MUFU.SQRT", k_sqrt, 64, "sqrt.approx.ftz.f32"}, {"MUFU.RSQ", k_rsqrt, 64, ""},
        {"IADD", k_iadd, 64, ""}, {"LOP", k_lop, 64, "xor.b32"}, {"SHF", k_shf, 64, "funnel shift"}, {"IMAD", k_imad, 64, ""},
        {"I2F (+FADD+IADD)", k_i2f, 64, "rate in I2F"}, {"F2I (+IADD+FADD)", k_f2i, 64, "rate in F2I"}, {"IMNMX", k_imnmx, 64, "max.s32"},
        {"LDS.128(+FADD)", k_lds128, 64, "broadcast ld.shared.v4 + 1 FADD each; rate in LDS"}, {"LDS.32(+FADD)", k_lds32, 64, ""},
        {"mix FFMA2+FMNMX3", k_mix_ffma2_fmnmx3, 128, "1:1, instr"}, {"mix FFMA+FMNMX", k_mix_ffma_fmnmx, 128, "1:1"},
        {"mix FFMA+DFMA", k_mix_ffma_dfma, 128, "1:1"}, {"mix FFMA+IADD", k_mix_ffma_iadd, 128, "1:1"},
        {"mix FMNMX+IADD", k_mix_fmnmx_iadd, 128, "1:1 (same pipe?)"}, {"mix 8 FFMA+1 SQRT", k_mix_ffma_sqrt7, 72, "8:1"},
        {"mix FFMA2+FFMA", k_mix_ffma2_ffma, 128, "1:1 instr"}, {"mix FMNMX+DFMA", k_mix_fmnmx_dfma, 128, "1:1"},
    };
    printf("device %s, %d SMs\n", prop.name, nsm);
    printf("%-30s %8s %14s %14s %10s  %s\n", "op", "threads", "ops/clk/SM", "warp-instr/clk/SMSP", "MHz", "note");
    for (const Case& c : cases) {
        for (int nt : {1024, 256}) {
            c.k<<<nsm, nt>>>(d_out, d_sink, 50, 1.0001f, 0.5f, 1.0000001, 0.5, 3);   // warm-up
            cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
            cudaEventRecord(e0);
            c.k<<<nsm, nt>>>(d_out, d_sink, iters, 1.0001f, 0.5f, 1.0000001, 0.5, 3);
            cudaEventRecord(e1);
            cudaError_t e = cudaDeviceSynchronize();
            if (e != cudaSuccess) { printf("%s: %s\n", c.name, cudaGetErrorString(e)); return 1; }
            float ms; cudaEventElapsedTime(&ms, e0, e1);
            cudaMemcpy(h.data(), d_out, sizeof(Out) * nsm, cudaMemcpyDeviceToHost);
            unsigned long long mx = 0; for (auto& o : h) mx = std::max(mx, o.cyc);
            const double ops = (double)c.ops_per_iter * iters * nt;
            printf("%-30s %8d %14.2f %14.3f %10.0f  %s\n", c.name, nt, ops / (double)mx, ops / 32.0 / 4.0 / (double)mx, (double)mx / (ms * 1e3), c.note);
        }
    }
    return 0;
}
