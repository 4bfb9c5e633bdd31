// probe.cu -- register-only micro-kernels that measure the FP32 / XU / LDS issue rates of the
// GPU the bench runs on (include/tfstat_probe.h).  They give the ALU roofline its denominator.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tfstat.h"
#include "../../include/tfstat_probe.h"

namespace {

__device__ __forceinline__ float exp2f_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

constexpr int kNT = 256;
constexpr int kIters = 4096;  // multiple of the unroll factor below
constexpr int kChains = 16;

template <int KIND>
__global__ void __launch_bounds__(kNT) probe_kernel(const float *__restrict__ in,
                                                    float *__restrict__ out,
                                                    long long *__restrict__ cycles)
{
    __shared__ float4 s_v[64];
    const float a = in[0], b = in[1];
    if (threadIdx.x < 64) s_v[threadIdx.x] = make_float4(a, b, a, b);
    __syncthreads();
    float acc[kChains];
#pragma unroll
    for (int j = 0; j < kChains; ++j) acc[j] = a * (float)(threadIdx.x + j);
    unsigned long long acc2[kChains / 2];
#pragma unroll
    for (int j = 0; j < kChains / 2; ++j)
        acc2[j] = ((unsigned long long)__float_as_uint(acc[2 * j + 1]) << 32) |
                  __float_as_uint(acc[2 * j]);
    const unsigned long long ab2 =
        ((unsigned long long)__float_as_uint(b) << 32) | __float_as_uint(a);
    // operand forms of fma.rn.f32x2 (kinds 8-10): two distinct register pairs, a broadcast scalar
    // and a pair, two broadcast scalars (what the multiplicands of exp_direct.cu's loop are)
    // (per-thread values, so that the operands live in the register file as in the kernel: a
    // block-uniform operand would go to a uniform register, which every form takes at full rate)
    const float sw = in[2] + 1e-9f * (float)threadIdx.x, sx = in[3] * (float)(threadIdx.x + 1);
    unsigned long long ba2, ww2, xx2, ab2v;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ba2) : "f"(b + sw), "f"(a + sx));
    asm("mov.b64 %0, {%1, %2};" : "=l"(ab2v) : "f"(a + sx), "f"(b + sx));
    asm("mov.b64 %0, {%1, %1};" : "=l"(ww2) : "f"(sw));
    asm("mov.b64 %0, {%1, %1};" : "=l"(xx2) : "f"(sx));
    double dacc[kChains / 2];
#pragma unroll
    for (int j = 0; j < kChains / 2; ++j) dacc[j] = (double)acc[j];
    const double da = (double)a, db = (double)b;
    int sidx = threadIdx.x >> 5;
    float xu0 = -a, xu1 = -b;

    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    const long long c0 = clock64();
#pragma unroll 8
    for (int it = 0; it < kIters; ++it) {
        if (KIND == TFSTAT_PROBE_FFMA) {
#pragma unroll
            for (int j = 0; j < kChains; ++j) acc[j] = fmaf(a, b, acc[j]);
        } else if (KIND == TFSTAT_PROBE_FADD) {
#pragma unroll
            for (int j = 0; j < kChains; ++j) acc[j] = acc[j] + a;
        } else if (KIND == TFSTAT_PROBE_MUFU_EX2) {
#pragma unroll
            for (int j = 0; j < kChains; ++j)
                asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(acc[j]));
        } else if (KIND == TFSTAT_PROBE_FFMA2) {
#pragma unroll
            for (int j = 0; j < kChains / 2; ++j)
                asm volatile("fma.rn.f32x2 %0, %1, %1, %0;" : "+l"(acc2[j]) : "l"(ab2));
        } else if (KIND == TFSTAT_PROBE_FFMA2_PAIRS) {
#pragma unroll
            for (int j = 0; j < kChains / 2; ++j)
                asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc2[j]) : "l"(ab2v), "l"(ba2));
        } else if (KIND == TFSTAT_PROBE_FFMA2_SCALAR_PAIR) {
#pragma unroll
            for (int j = 0; j < kChains / 2; ++j)
                asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc2[j]) : "l"(ww2), "l"(ab2v));
        } else if (KIND == TFSTAT_PROBE_FFMA2_SCALARS) {
#pragma unroll
            for (int j = 0; j < kChains / 2; ++j)
                asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc2[j]) : "l"(ww2), "l"(xx2));
        } else if (KIND == TFSTAT_PROBE_FADD2) {
#pragma unroll
            for (int j = 0; j < kChains / 2; ++j)
                asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(acc2[j]) : "l"(ab2));
        } else if (KIND == TFSTAT_PROBE_FFMA_MUFU) {
#pragma unroll
            for (int j = 0; j < kChains; ++j) acc[j] = fmaf(a, b, acc[j]);
            asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(xu0));
            asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(xu1));
        } else if (KIND == TFSTAT_PROBE_LDS128) {
#pragma unroll
            for (int j = 0; j < kChains / 4; ++j) {
                const float4 v = s_v[(sidx + j) & 63];
                acc[4 * j] += v.x;
                sidx += (int)v.y;  // b == 0 at run time; keeps the address data-dependent
            }
        } else if (KIND == TFSTAT_PROBE_DFMA) {
#pragma unroll
            for (int j = 0; j < kChains / 2; ++j) dacc[j] = fma(da, db, dacc[j]);
        }
    }
    const long long c1 = clock64();
    float r = 0.f;
#pragma unroll
    for (int j = 0; j < kChains; ++j) r += acc[j];
#pragma unroll
    for (int j = 0; j < kChains / 2; ++j)
        r += __uint_as_float((unsigned)acc2[j]) + __uint_as_float((unsigned)(acc2[j] >> 32)) +
             (float)dacc[j];
    out[(size_t)blockIdx.x * kNT + threadIdx.x] = r + (float)sidx + xu0 + xu1;
    // warps are not scheduled fairly, so one warp's elapsed clocks say nothing: take the span
    // from the first start to the last end over every warp that ran on SM 0
    if (smid == 0 && (threadIdx.x & 31) == 0) {
        atomicMin(reinterpret_cast<unsigned long long *>(cycles), (unsigned long long)c0);
        atomicMax(reinterpret_cast<unsigned long long *>(cycles) + 1, (unsigned long long)c1);
    }
}

int ops_per_iter(int kind)
{
    switch (kind) {
    case TFSTAT_PROBE_FFMA:
    case TFSTAT_PROBE_FADD:
    case TFSTAT_PROBE_MUFU_EX2:
    case TFSTAT_PROBE_FFMA2:
    case TFSTAT_PROBE_FFMA2_PAIRS:
    case TFSTAT_PROBE_FFMA2_SCALAR_PAIR:
    case TFSTAT_PROBE_FFMA2_SCALARS:
    case TFSTAT_PROBE_FADD2: return kChains;
    case TFSTAT_PROBE_FFMA_MUFU: return kChains + 2;
    case TFSTAT_PROBE_LDS128: return kChains / 4;
    case TFSTAT_PROBE_DFMA: return kChains / 2;
    }
    return 0;
}

template <int KIND>
void launch(int grid, const float *in, float *out, long long *cyc)
{
    probe_kernel<KIND><<<grid, kNT>>>(in, out, cyc);
}

}  // namespace

// ---- the isolated core loop of the direct exponential sum, in two operand forms ---------------
// (what bounds exp_direct_kernel once everything around the loop is taken away)
namespace {

typedef unsigned long long u64p;
__device__ __forceinline__ u64p pk2(float lo, float hi)
{
    u64p r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(u64p v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ void fma2(u64p &d, u64p a, u64p b)
{
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b));
}
constexpr int kLoopAtoms = 192;

// FORM 0: accumulators paired by CHANNEL of one cell, (A,B) (Re Fa,Im Fa) (Re Fb,Im Fb) (C_c,C_c+1):
//         FFMA2 acc, w.F32 (broadcast), x pair
// FORM 1: accumulators paired by CELL, (X_c, X_c+1) for each of the 7 channels:
//         FFMA2 acc, w.F32, x.F32 (two broadcast scalars)
template <int FORM, int C, int MINB>
__global__ void __launch_bounds__(128, MINB)
    probe_loop_kernel(const ulonglong2 *__restrict__ g, float *__restrict__ out, const int reps,
                      const float kexp0, long long *__restrict__ cycles)
{
    __shared__ ulonglong2 s[2 * kLoopAtoms];
    for (int i = threadIdx.x; i < 2 * kLoopAtoms; i += 128) s[i] = g[i];
    __syncthreads();
    const float kexp = kexp0 * (1.0f + 1e-3f * threadIdx.x), cexp = 0.1f;
    u64p acc[7 * C / 2];
#pragma unroll
    for (int i = 0; i < 7 * C / 2; ++i) acc[i] = 0ull;
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    const long long c0 = clock64();
    for (int r = 0; r < reps; ++r) {
#pragma unroll 24
        for (int i = 0; i < kLoopAtoms; ++i) {
            const ulonglong2 ra = s[2 * i], rb = s[2 * i + 1];
            if (FORM >= 2) {
                // FORM 2 / 3: two / four more broadcast LDS.128 per atom whose results nobody
                // uses -- 8 / 16 more register write-backs and nothing else (do they cost what
                // the FMA pipe's own write-backs cost?)
#pragma unroll
                for (int e = 0; e < 2 * (FORM - 1); ++e) {
                    float d0, d1, d2, d3;
                    asm volatile("ld.volatile.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                                 : "=f"(d0), "=f"(d1), "=f"(d2), "=f"(d3)
                                 : "r"((unsigned)__cvta_generic_to_shared(&s[(2 * i + e) % (2 * kLoopAtoms)])));
                }
            }
            float x[7], dt;
            upk2(ra.x, dt, x[2]);
            upk2(ra.y, x[0], x[1]);
            upk2(rb.x, x[3], x[4]);
            upk2(rb.y, x[5], x[6]);
            // (as exp_direct.cu: w^2 from a second MUFU.EX2 on the exponent-bumped argument)
            const float arg = fmaf(dt, kexp, cexp);
            const float w = exp2f_approx(arg);
            const float w2 = exp2f_approx(__int_as_float(__float_as_int(arg) + 0x00800000));
            const u64p ww = pk2(w, w), w2w2 = pk2(w2, w2);
            if (FORM == 0) {
                const u64p abab = pk2(x[2], x[2]);
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    fma2(acc[3 * c], w2w2, ra.y);
                    fma2(acc[3 * c + 1], ww, rb.x);
                    fma2(acc[3 * c + 2], ww, rb.y);
                }
#pragma unroll
                for (int p = 0; p < C / 2; ++p) fma2(acc[3 * C + p], w2w2, abab);
            } else {
#pragma unroll
                for (int k = 0; k < 7; ++k) {
                    const u64p xx = pk2(x[k], x[k]);
#pragma unroll
                    for (int p = 0; p < C / 2; ++p) fma2(acc[k * (C / 2) + p], k < 3 ? w2w2 : ww, xx);
                }
            }
        }
    }
    const long long c1 = clock64();
    float sum = 0.0f;
#pragma unroll
    for (int i = 0; i < 7 * C / 2; ++i) {
        float a, b;
        upk2(acc[i], a, b);
        sum += a + b;
    }
    out[(size_t)blockIdx.x * 128 + threadIdx.x] = sum;
    if (smid == 0 && (threadIdx.x & 31) == 0) {
        atomicMin(reinterpret_cast<unsigned long long *>(cycles), (unsigned long long)c0);
        atomicMax(reinterpret_cast<unsigned long long *>(cycles) + 1, (unsigned long long)c1);
    }
}

}  // namespace

extern "C" int tfstat_probe_direct_loop(int form, int cells, int reps, double *terms_per_clk_sm,
                                        double *terms_per_s)
{
    if (form < 0 || form > 3 || (cells != 8 && cells != 16) || !terms_per_clk_sm)
        return TFSTAT_EINVAL;
    if (reps < 1) reps = 200;
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return TFSTAT_ECUDA;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return TFSTAT_ECUDA;
    const int per_sm = cells == 8 ? 4 : 3;
    const int grid = n_sm * per_sm;
    ulonglong2 *g = nullptr;
    float *out = nullptr;
    long long *cyc = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = TFSTAT_ECUDA;
    do {
        if (cudaMalloc(&g, sizeof(ulonglong2) * 2 * kLoopAtoms) != cudaSuccess) break;
        if (cudaMalloc(&out, sizeof(float) * (size_t)grid * 128) != cudaSuccess) break;
        if (cudaMalloc(&cyc, 2 * sizeof(long long)) != cudaSuccess) break;
        float h[8 * kLoopAtoms];
        for (int i = 0; i < kLoopAtoms; ++i) {
            h[8 * i] = (float)i;
            for (int k = 1; k < 8; ++k) h[8 * i + k] = 0.01f * k;
        }
        if (cudaMemcpy(g, h, sizeof(h), cudaMemcpyHostToDevice) != cudaSuccess) break;
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) break;
        float ms = 0.0f;
        for (int pass = 0; pass < 2; ++pass) {  // warm-up, then the timed launch
            const unsigned long long init[2] = {~0ull, 0ull};
            cudaMemcpy(cyc, init, sizeof(init), cudaMemcpyHostToDevice);
            cudaEventRecord(e0);
            const int n = pass ? reps : 4;
            if (form == 0 && cells == 8) probe_loop_kernel<0, 8, 4><<<grid, 128>>>(g, out, n, -1e-3f, cyc);
            if (form == 1 && cells == 8) probe_loop_kernel<1, 8, 4><<<grid, 128>>>(g, out, n, -1e-3f, cyc);
            if (form == 0 && cells == 16) probe_loop_kernel<0, 16, 3><<<grid, 128>>>(g, out, n, -1e-3f, cyc);
            if (form == 1 && cells == 16) probe_loop_kernel<1, 16, 3><<<grid, 128>>>(g, out, n, -1e-3f, cyc);
            if (form == 2 && cells == 8) probe_loop_kernel<2, 8, 4><<<grid, 128>>>(g, out, n, -1e-3f, cyc);
            if (form == 3 && cells == 8) probe_loop_kernel<3, 8, 4><<<grid, 128>>>(g, out, n, -1e-3f, cyc);
            if (form == 2 && cells == 16) probe_loop_kernel<2, 16, 3><<<grid, 128>>>(g, out, n, -1e-3f, cyc);
            if (form == 3 && cells == 16) probe_loop_kernel<3, 16, 3><<<grid, 128>>>(g, out, n, -1e-3f, cyc);
            cudaEventRecord(e1);
            if (cudaEventSynchronize(e1) != cudaSuccess) break;
            cudaEventElapsedTime(&ms, e0, e1);
        }
        if (cudaGetLastError() != cudaSuccess || ms <= 0.0f) break;
        unsigned long long span[2] = {0, 0};
        if (cudaMemcpy(span, cyc, sizeof(span), cudaMemcpyDeviceToHost) != cudaSuccess) break;
        const double terms_sm = (double)per_sm * 128 * cells * kLoopAtoms * reps;
        *terms_per_clk_sm = terms_sm / (double)(span[1] - span[0]);
        if (terms_per_s) *terms_per_s = terms_sm * n_sm / (ms * 1e-3);
        rc = TFSTAT_OK;
    } while (0);
    cudaFree(g);
    cudaFree(out);
    cudaFree(cyc);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    return rc;
}

extern "C" int tfstat_probe_alu(int kind, int reps, double *lane_ops_per_s,
                                double *ops_per_clk_sm, double *sm_mhz)
{
    if (kind < 0 || kind >= TFSTAT_PROBE_KINDS || !lane_ops_per_s) return TFSTAT_EINVAL;
    if (reps < 1) reps = 3;
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return TFSTAT_ECUDA;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return TFSTAT_ECUDA;
    const int ctas_per_sm = 4;  // 1024 threads / SM, 8 warps per scheduler
    const int grid = n_sm * ctas_per_sm;
    float *in = nullptr, *out = nullptr;
    long long *cyc = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = TFSTAT_ECUDA;
    do {
        if (cudaMalloc(&in, 4 * sizeof(float)) != cudaSuccess) break;
        if (cudaMalloc(&out, sizeof(float) * (size_t)grid * kNT) != cudaSuccess) break;
        if (cudaMalloc(&cyc, 2 * sizeof(long long)) != cudaSuccess) break;
        const float h_in[4] = {kind == TFSTAT_PROBE_MUFU_EX2 ? -0.5f : 1.0000001f,
                               kind == TFSTAT_PROBE_LDS128 ? 0.0f : 1e-9f, 0.9999999f, 1e-9f};
        if (cudaMemcpy(in, h_in, sizeof(h_in), cudaMemcpyHostToDevice) != cudaSuccess) break;
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) break;
        float best_ms = 1e30f;
        for (int r = 0; r <= reps; ++r) {
            const unsigned long long init[2] = {~0ull, 0ull};
            cudaMemcpy(cyc, init, sizeof(init), cudaMemcpyHostToDevice);
            cudaEventRecord(e0);
            switch (kind) {
            case 0: launch<0>(grid, in, out, cyc); break;
            case 1: launch<1>(grid, in, out, cyc); break;
            case 2: launch<2>(grid, in, out, cyc); break;
            case 3: launch<3>(grid, in, out, cyc); break;
            case 4: launch<4>(grid, in, out, cyc); break;
            case 5: launch<5>(grid, in, out, cyc); break;
            case 6: launch<6>(grid, in, out, cyc); break;
            case 7: launch<7>(grid, in, out, cyc); break;
            case 8: launch<8>(grid, in, out, cyc); break;
            case 9: launch<9>(grid, in, out, cyc); break;
            case 10: launch<10>(grid, in, out, cyc); break;
            }
            cudaEventRecord(e1);
            if (cudaEventSynchronize(e1) != cudaSuccess) break;
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (r > 0 && ms < best_ms) best_ms = ms;
        }
        if (cudaGetLastError() != cudaSuccess || best_ms > 1e29f) break;
        unsigned long long h_span[2] = {0, 0};
        if (cudaMemcpy(h_span, cyc, sizeof(h_span), cudaMemcpyDeviceToHost) != cudaSuccess) break;
        const long long h_cyc = (long long)(h_span[1] - h_span[0]);
        const double ops = (double)grid * kNT * (double)kIters * ops_per_iter(kind);
        *lane_ops_per_s = ops / (best_ms * 1e-3);
        if (ops_per_clk_sm)
            *ops_per_clk_sm = (double)ctas_per_sm * kNT * kIters * ops_per_iter(kind) / (double)h_cyc;
        if (sm_mhz) *sm_mhz = (double)h_cyc / (best_ms * 1e-3) * 1e-6;
        rc = TFSTAT_OK;
    } while (0);
    cudaFree(in);
    cudaFree(out);
    cudaFree(cyc);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    return rc;
}
