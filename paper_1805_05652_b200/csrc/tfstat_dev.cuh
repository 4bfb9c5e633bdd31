// tfstat_dev.cuh -- shared device-side definitions for libtfstat (sm_100a).
//
// Notation follows the paper: atoms alpha with start times t_alpha; grid t0_m, tau_n; window
// support W(m,n) = {alpha : t0_m <= t_alpha < t0_m + k tau_n}, k = 1 (rect, eq. 3) or 3 (exp,
// eq. 4); sums A,B,C,Fa,Fb; D = AB - C^2 and eq. (7).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tfstat.h"

namespace tfstat {

// ---------------------------------------------------------------------------------------
// problem description passed by value to every kernel
// ---------------------------------------------------------------------------------------
struct Grid {
    int32_t t0_min, dt0, N_t0;
    int32_t tau_min, dtau, N_tau;
    int32_t k;  // window length in units of tau: 1 rect, 3 exp
};

// Step a1: window -> atom-index bounds.
//   lo[m]   = first alpha with t_alpha >= t0_m
//   hi(m,n) = first alpha with t_alpha >= t0_m + k tau_n
// All window end times lie on the lattice base + j*g, g = gcd(dt0, k dtau), so one table
// edge[j] = lower_bound(t, base + j g), j = m*e_m + n*e_n, serves every cell (and every
// template: timestamps are shared).  If the lattice is too fine (edge == nullptr) kernels
// fall back to a binary search per cell.
struct Bounds {
    const int32_t *t;     // [n_atoms] timestamps
    const int32_t *lo;    // [N_t0]
    const int32_t *edge;  // [J] or nullptr
    int32_t n_atoms;
    int32_t e_m, e_n;
    int32_t J;
};

__device__ __forceinline__ int lower_bound_t(const int32_t *__restrict__ t, int n, long long x)
{
    int a = 0, b = n;  // first index with t[i] >= x
    while (a < b) {
        const int mid = (a + b) >> 1;
        if ((long long)__ldg(t + mid) < x) a = mid + 1;
        else b = mid;
    }
    return a;
}

__device__ __forceinline__ long long t0_of(const Grid &g, int m)
{
    return (long long)g.t0_min + (long long)m * g.dt0;
}
__device__ __forceinline__ long long tau_of(const Grid &g, int n)
{
    return (long long)g.tau_min + (long long)n * g.dtau;
}

__device__ __forceinline__ int hi_index(const Bounds &b, const Grid &g, int m, int n)
{
    if (b.edge) return __ldg(b.edge + (long long)m * b.e_m + (long long)n * b.e_n);
    return lower_bound_t(b.t, b.n_atoms, t0_of(g, m) + (long long)g.k * tau_of(g, n));
}

// ---------------------------------------------------------------------------------------
// step a4: cell closure, eq. (7).  Sums come in as fp32 (exp path) or fp64 (rect path); the
// closure itself runs in fp64 because D = AB - C^2 and the numerator both cancel by the
// conditioning number D/(AB).
// ---------------------------------------------------------------------------------------
struct Sums64 {
    double A, B, C, far, fai, fbr, fbi;
};

__device__ __forceinline__ float closure_2F(const Sums64 &s, int cnt, int min_atoms,
                                            uint32_t &flags)
{
    const double D = s.A * s.B - s.C * s.C;
    flags = (cnt < min_atoms ? 1u : 0u) | (!(D > 0.0) ? 2u : 0u);
    if (flags) return 0.0f;
    const double na = s.far * s.far + s.fai * s.fai;
    const double nb = s.fbr * s.fbr + s.fbi * s.fbi;
    const double re = s.far * s.fbr + s.fai * s.fbi;
    const double num = s.B * na + s.A * nb - 2.0 * s.C * re;
    return (float)(2.0 * num / D);
}

// Exponential-window cell from fp32 sums: fp32 closure where the cell is well conditioned
// (D > AB/64: the cancellation in D = AB - C^2 and in the numerator amplifies the fp32 rounding of
// the sums by at most ~64, i.e. <= ~1e-5 relative on 2F), fp64 closure otherwise, with a safety
// net for ill-conditioned SHORT windows.
// fp32 sums carry ~6e-8 relative rounding per channel, which D = AB - C^2 amplifies by AB/D: a
// window of one or two atoms can have AB/D ~ 1e4..1e6 (a single two-detector atom reaches 3e6),
// and then no fp32 accumulation meets the 1e-3 contract.  Such cells are cheap to do properly:
// if D <= AB/64 and the window holds at most kRedoMaxAtoms atoms, its sums are recomputed in
// fp64 straight from the atoms (libm-grade exp), exactly as the oracle defines them.  Long
// windows (more atoms than that) mix many antenna phases and are well conditioned in practice;
// they keep the fp32 sums and the fp64 closure.
constexpr int kRedoMaxAtoms = 64;

static __device__ __forceinline__ Sums64 exp_resum64_inline(const float *__restrict__ base, const int64_t ld,
                                           const int32_t *__restrict__ t, const int lo,
                                           const int hi, const long long t0, const double tau)
{
    Sums64 s;
    s.A = s.B = s.C = s.far = s.fai = s.fbr = s.fbi = 0.0;
#pragma unroll 1
    for (int al = lo; al < hi; ++al) {
        const double w = exp(-(double)((long long)__ldg(t + al) - t0) / tau);
        const double w2 = w * w;
        s.A += w2 * (double)__ldg(base + al);
        s.B += w2 * (double)__ldg(base + ld + al);
        s.C += w2 * (double)__ldg(base + 2 * ld + al);
        s.far += w * (double)__ldg(base + 3 * ld + al);
        s.fai += w * (double)__ldg(base + 4 * ld + al);
        s.fbr += w * (double)__ldg(base + 5 * ld + al);
        s.fbi += w * (double)__ldg(base + 6 * ld + al);
    }
    return s;
}

static __device__ __noinline__ Sums64 exp_resum64_call(const float *__restrict__ base,
                                                       const int64_t ld,
                                                       const int32_t *__restrict__ t, const int lo,
                                                       const int hi, const long long t0,
                                                       const double tau)
{
    return exp_resum64_inline(base, ld, t, lo, hi, t0, tau);
}

// REDO_INLINE: how the rare fp64 re-sum is attached.  Measured on B200: as a call it costs the
// direct kernel nothing (3.76e12 terms/s; inlined 3.59e12, the allocator gives the fp64 loop
// registers the packed accumulators need), while the sliding kernel, whose closure sits inside
// the t0 loop, is better off with it inlined (96 registers instead of 121).
template <bool REDO_INLINE>
__device__ __forceinline__ float closure_2F_exp(const float A, const float B, const float C,
                                                const float far, const float fai,
                                                const float fbr, const float fbi, const int lo,
                                                const int cnt, const int min_atoms,
                                                uint32_t &flags, const float *__restrict__ base,
                                                const int64_t ld, const int32_t *__restrict__ t,
                                                const long long t0, const double tau)
{
    const float p = A * B;
    const float D = fmaf(-C, C, p);
    // (1e-30 < p < 1e30: with atoms scaled far down D would be subnormal and the fast divide inf,
    // scaled far up __fdividef returns 0 for D > 2^126 and the numerator overflows)
    if (D > 0.015625f * p && p > 1.0e-30f && p < 1.0e30f && cnt >= min_atoms) {
        const float na = fmaf(far, far, fai * fai);
        const float nb = fmaf(fbr, fbr, fbi * fbi);
        const float re = fmaf(far, fbr, fai * fbi);
        float num = B * na;
        num = fmaf(A, nb, num);
        num = fmaf(-2.0f * C, re, num);
        const float r = 2.0f * __fdividef(num, D);
        if (fabsf(r) < 3.0e38f) {  // atoms scaled far up overflow the numerator: fp64 below
            flags = 0u;
            return r;
        }
    }
    Sums64 s;
    if (cnt >= 1 && cnt <= kRedoMaxAtoms) {  // also cells with too few atoms: their D flag counts
        s = REDO_INLINE ? exp_resum64_inline(base, ld, t, lo, lo + cnt, t0, tau)
                        : exp_resum64_call(base, ld, t, lo, lo + cnt, t0, tau);
    } else {
        s.A = A;
        s.B = B;
        s.C = C;
        s.far = far;
        s.fai = fai;
        s.fbr = fbr;
        s.fbi = fbi;
    }
    return closure_2F(s, cnt, min_atoms, flags);
}

// ---------------------------------------------------------------------------------------
// step a5: marginalisation state (max 2F with lowest-index argmax; online log-sum-exp)
// ---------------------------------------------------------------------------------------
struct Marg {
    float best;    // max 2F so far (-inf if none)
    int32_t idx;   // flat index of best (INT_MAX if none)
    float M;       // running max of F = 2F/2 (-inf if none)
    float S;       // sum exp(F - M)
    int32_t nvalid;
};

struct __align__(16) Partial {  // one per CTA in the workspace, 32 bytes
    float best;
    int32_t idx;
    float M;
    float S;
    int32_t nvalid;
    int32_t pad[3];
};

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

#define TFSTAT_LOG2E_F 1.4426950408889634f

// packed fp32x2 arithmetic (sm_100: SASS FFMA2 / FMUL2), two lanes of one 64-bit register
typedef unsigned long long u64;

__device__ __forceinline__ u64 pack2(const float lo, const float hi)
{
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(const u64 v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ void ffma2(u64 &d, const u64 a, const u64 b)
{
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b));
}
__device__ __forceinline__ u64 fmul2(const u64 a, const u64 b)
{
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}


__device__ __forceinline__ void marg_init(Marg &a)
{
    a.best = -INFINITY;
    a.idx = 0x7fffffff;
    a.M = -INFINITY;
    a.S = 0.0f;
    a.nvalid = 0;
}

__device__ __forceinline__ void marg_add(Marg &a, float twoF, int32_t flat)
{
    if (twoF > a.best || (twoF == a.best && flat < a.idx)) {
        a.best = twoF;
        a.idx = flat;
    }
    const float F = 0.5f * twoF;
    if (F > a.M) {
        a.S = a.S * ex2_approx((a.M - F) * TFSTAT_LOG2E_F) + 1.0f;  // M = -inf: S*0 + 1
        a.M = F;
    } else {
        a.S += ex2_approx((F - a.M) * TFSTAT_LOG2E_F);
    }
    a.nvalid += 1;
}

__device__ __forceinline__ void marg_merge(Marg &a, const Marg &b)
{
    if (b.best > a.best || (b.best == a.best && b.idx < a.idx)) {
        a.best = b.best;
        a.idx = b.idx;
    }
    const float M = fmaxf(a.M, b.M);
    if (M > -INFINITY) {
        a.S = a.S * ex2_approx((a.M - M) * TFSTAT_LOG2E_F) +
              b.S * ex2_approx((b.M - M) * TFSTAT_LOG2E_F);
        a.M = M;
    }
    a.nvalid += b.nvalid;
}

__device__ __forceinline__ Marg marg_shfl_xor(const Marg &a, int lane_mask)
{
    Marg b;
    b.best = __shfl_xor_sync(0xffffffffu, a.best, lane_mask);
    b.idx = __shfl_xor_sync(0xffffffffu, a.idx, lane_mask);
    b.M = __shfl_xor_sync(0xffffffffu, a.M, lane_mask);
    b.S = __shfl_xor_sync(0xffffffffu, a.S, lane_mask);
    b.nvalid = __shfl_xor_sync(0xffffffffu, a.nvalid, lane_mask);
    return b;
}

__device__ __forceinline__ void marg_warp_reduce(Marg &a)
{
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        const Marg b = marg_shfl_xor(a, s);
        marg_merge(a, b);
    }
}

// Block reduce; result valid in thread 0.  `scratch` holds >= 32 Marg.
template <int NT>
__device__ __forceinline__ void marg_block_reduce(Marg &a, Marg *scratch)
{
    marg_warp_reduce(a);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) scratch[warp] = a;
    __syncthreads();
    if (warp == 0) {
        if (lane < NT / 32) a = scratch[lane];
        else marg_init(a);
        marg_warp_reduce(a);
    }
}

__device__ __forceinline__ void partial_store(Partial *p, const Marg &a)
{
    p->best = a.best;
    p->idx = a.idx;
    p->M = a.M;
    p->S = a.S;
    p->nvalid = a.nvalid;
}

// ---------------------------------------------------------------------------------------
// Kernel launches.  The kernels of one call form a chain on the caller's stream (bounds -> pack
// -> sums -> finalize) in plain stream order.
//
// Programmatic dependent launch (griddepcontrol: a kernel is set up while its predecessor
// drains and waits before it reads what the predecessor wrote) was in here for two rounds and
// has been WITHDRAWN.  It bought 1-5 us per call on launch-bound calls, cost 15 % where the
// early-launched grid was big (its CTAs hold their registers while they wait), and it was
// behind a rare illegal-address fault, seen mostly where the library runs on non-blocking
// streams (3 of 20 runs of the GPU suite; 0 of 24 + 24 without it): every kernel here reads
// its predecessor's output through the read-only path (ld.global.nc, which `const __restrict__`
// lets the compiler pick), and that path's contract -- the memory is not written while the
// kernel lives -- does not hold for a kernel that is resident before its predecessor is done.
// ---------------------------------------------------------------------------------------
template <typename... KArgs, typename... Args>
inline cudaError_t launch_k(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem,
                            cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// ---------------------------------------------------------------------------------------
// Packed atoms (pack.cu) and the bulk asynchronous copy that stages them: cp.async.bulk
// global -> shared, completion signalled on an mbarrier (the 1-D TMA path of sm_90+/sm_100).
// ---------------------------------------------------------------------------------------
constexpr int kPackBlock = 768;  // atoms per block of the packed time base; divisible by every
                                 // staging chunk (128, 192, 256, 384), so a chunk has ONE base

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(const uint32_t bar, const uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
// makes the barrier initialisation visible to the async proxy (the copy engine)
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
// arm the barrier for `bytes` and issue the copy; src, dst 16-byte aligned, bytes % 16 == 0
__device__ __forceinline__ void bulk_load(const uint32_t dst, const void *src, const uint32_t bytes,
                                          const uint32_t bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(dst), "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void mbar_wait(const uint32_t bar, const uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "MBAR_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra MBAR_DONE_%=;\n"
        "bra MBAR_WAIT_%=;\n"
        "MBAR_DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

// ---------------------------------------------------------------------------------------
// host-side launchers (one per .cu file)
// ---------------------------------------------------------------------------------------
struct Problem {
    const float *atoms;        // [T][7][ld]
    int64_t template_stride;   // floats
    int64_t ld;
    int32_t n_templates;
    int32_t min_atoms;
    Grid grid;
    Bounds bounds;
    tfstat_result *out;        // [T] or nullptr
    float *out_maps;           // [T][N_t0][N_tau] or nullptr
    uint8_t *out_flags;        // same shape or nullptr
};

}  // namespace tfstat
