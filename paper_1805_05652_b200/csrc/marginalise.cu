// marginalise.cu -- step a5 on a map already in HBM (tfstat_marginalise) and the final
// cross-CTA combine of the fused kernels' partial marginals.
//
// max 2F with lowest-flat-index argmax and logB = log sum_valid exp(2F/2) (eq. 5, PAPER.md:56;
// DESIGN.md R13, R14).  Streaming, HBM-bound: 4 B (+1 B flags) per cell.
#include "plan.h"

namespace tfstat {

namespace {

constexpr int kMargNT = 256;
constexpr int kMargUnroll = 4;

// Per-thread running marginals in the cheap form: max with a RARE branch for the argmax, and the
// log-sum-exp as sum 2^(F log2e - ref2) against a reference exponent that only moves when a value
// exceeds it by more than 2^60 (so nothing overflows and the common path is FFMA + MUFU.EX2 + FADD
// per cell).  Converted to a Marg at the end.
struct StreamMarg {
    float best;    // running max of 2F
    int64_t qbest; // index of the 16-byte group that holds it (first one on ties)
    float ref2;
    float sum;
    int32_t nv;
};
constexpr float kHalfLog2eM = 0.72134752044448170368f;  // log2(e) / 2: F log2e = 2F * this

__device__ __forceinline__ uint32_t flag_bytes_to_count(const uint32_t fl4)
{
    return ((fl4 & 0xffu) != 0u) + ((fl4 & 0xff00u) != 0u) + ((fl4 & 0xff0000u) != 0u) +
           ((fl4 & 0xff000000u) != 0u);
}

// Four cells.  The max only remembers WHICH 16-byte group held it (two selects, no branch: with
// ~10 groups per thread a branch on "new maximum" is taken by some lane of almost every warp);
// the cell inside the group is found once, at the end, by re-reading that group.
template <bool FLAGS>
__device__ __forceinline__ void stream_add4(StreamMarg &a, const float4 v, const uint32_t fl4,
                                            const int64_t q)
{
    float x[4] = {v.x, v.y, v.z, v.w};
    if (FLAGS) {
        if (fl4 != 0u) {  // flagged cells lose every max and add 2^-inf = 0
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (((fl4 >> (8 * j)) & 0xffu) != 0u) x[j] = -INFINITY;
        }
        a.nv += 4 - (int32_t)flag_bytes_to_count(fl4);
    } else {
        a.nv += 4;
    }
    const float m4 = fmaxf(fmaxf(x[0], x[1]), fmaxf(x[2], x[3]));
    const bool up = m4 > a.best;  // ascending q within a thread: '>' keeps the first group
    a.qbest = up ? q : a.qbest;
    a.best = up ? m4 : a.best;
    if (fmaf(m4, kHalfLog2eM, -a.ref2) > 60.0f) {  // rare: move the reference
        a.sum *= ex2_approx(a.ref2 - m4 * kHalfLog2eM);
        a.ref2 = m4 * kHalfLog2eM;
    }
    float acc = 0.0f;
#pragma unroll
    for (int j = 0; j < 4; ++j) acc += ex2_approx(fmaf(x[j], kHalfLog2eM, -a.ref2));
    a.sum += acc;
}

template <bool FLAGS>
__device__ __forceinline__ void marginalise_body(const float *__restrict__ map,
                                                 const uint8_t *__restrict__ flags,
                                                 const int64_t n_cells, Marg &mg)
{
    StreamMarg sm;
    sm.best = -INFINITY;
    sm.qbest = -1;
    sm.ref2 = -1.0e30f;  // finite: a flagged cell (-inf) must give 2^-inf = 0, not inf - inf
    sm.sum = 0.0f;
    sm.nv = 0;
    const bool vec = ((reinterpret_cast<uintptr_t>(map) & 15u) == 0) &&
                     (!FLAGS || (reinterpret_cast<uintptr_t>(flags) & 3u) == 0);
    const int64_t n4 = vec ? n_cells / 4 : 0;
    const int64_t stride = (int64_t)gridDim.x * kMargNT;
    // kMargUnroll independent 16-byte loads in flight per thread (6.5 TB/s x ~1 us of latency
    // is ~45 KB per SM), consumed in ascending index order
    int64_t q = (int64_t)blockIdx.x * kMargNT + threadIdx.x;
    for (; q + (kMargUnroll - 1) * stride < n4; q += kMargUnroll * stride) {
        float4 v[kMargUnroll];
        uint32_t f[kMargUnroll];
#pragma unroll
        for (int k = 0; k < kMargUnroll; ++k) {
            v[k] = __ldcs(reinterpret_cast<const float4 *>(map) + q + k * stride);
            f[k] = FLAGS ? __ldcs(reinterpret_cast<const uint32_t *>(flags) + q + k * stride) : 0u;
        }
#pragma unroll
        for (int k = 0; k < kMargUnroll; ++k)
            stream_add4<FLAGS>(sm, v[k], f[k], q + k * stride);
    }
    for (; q < n4; q += stride) {
        const float4 v = __ldcs(reinterpret_cast<const float4 *>(map) + q);
        const uint32_t f = FLAGS ? __ldcs(reinterpret_cast<const uint32_t *>(flags) + q) : 0u;
        stream_add4<FLAGS>(sm, v, f, q);
    }
    marg_init(mg);
    mg.nvalid = sm.nv;
    if (sm.best > -INFINITY) {
        // the first unflagged cell of group qbest that equals the maximum
        const float4 v = *(reinterpret_cast<const float4 *>(map) + sm.qbest);
        const uint32_t f = FLAGS ? *(reinterpret_cast<const uint32_t *>(flags) + sm.qbest) : 0u;
        const float x[4] = {v.x, v.y, v.z, v.w};
        int jb = 3;
#pragma unroll
        for (int j = 3; j >= 0; --j)
            if (x[j] == sm.best && ((f >> (8 * j)) & 0xffu) == 0u) jb = j;
        mg.best = sm.best;
        mg.idx = (int32_t)(4 * sm.qbest) + jb;
        mg.M = 0.5f * sm.best;
        mg.S = sm.sum * ex2_approx(sm.ref2 - sm.best * kHalfLog2eM);
    }
    // ragged tail (and unaligned maps): the plain per-cell way; indices above all of the above
    for (int64_t i = 4 * n4 + (int64_t)blockIdx.x * kMargNT + threadIdx.x; i < n_cells;
         i += stride) {
        if (!FLAGS || flags[i] == 0) marg_add(mg, map[i], (int32_t)i);
    }
}

// Combine `per_template` partials (fixed order -> deterministic) and write one result.  Called by
// all 256 threads of a CTA.  Plain (coherent) loads: the partials may have been written by other
// CTAs of the same launch (marginalise_fused_kernel).
__device__ __forceinline__ void finalize_body(const Partial *p, const int64_t per_template,
                                              const int32_t N_tau, tfstat_result *__restrict__ out)
{
    __shared__ float s_best[256];
    __shared__ int32_t s_idx[256];
    __shared__ float s_M[256];
    __shared__ double s_S[256];
    __shared__ int32_t s_nv[256];
    const int tid = threadIdx.x;
    float best = -INFINITY, M = -INFINITY;
    int32_t idx = 0x7fffffff, nv = 0;
    for (int64_t i = tid; i < per_template; i += 256) {
        const Partial q = p[i];
        if (q.best > best || (q.best == best && q.idx < idx)) {
            best = q.best;
            idx = q.idx;
        }
        M = fmaxf(M, q.M);
        nv += q.nvalid;
    }
    s_best[tid] = best;
    s_idx[tid] = idx;
    s_M[tid] = M;
    s_nv[tid] = nv;
    __syncthreads();
    for (int s = 128; s >= 1; s >>= 1) {
        if (tid < s) {
            if (s_best[tid + s] > s_best[tid] ||
                (s_best[tid + s] == s_best[tid] && s_idx[tid + s] < s_idx[tid])) {
                s_best[tid] = s_best[tid + s];
                s_idx[tid] = s_idx[tid + s];
            }
            s_M[tid] = fmaxf(s_M[tid], s_M[tid + s]);
            s_nv[tid] += s_nv[tid + s];
        }
        __syncthreads();
    }
    const float Mall = s_M[0];
    double S = 0.0;
    for (int64_t i = tid; i < per_template; i += 256) {
        const Partial q = p[i];
        if (q.nvalid > 0) S += (double)q.S * exp((double)q.M - (double)Mall);
    }
    s_S[tid] = S;
    __syncthreads();
    for (int s = 128; s >= 1; s >>= 1) {
        if (tid < s) s_S[tid] += s_S[tid + s];
        __syncthreads();
    }
    if (tid == 0) {
        tfstat_result r;
        r.n_valid = s_nv[0];
        if (r.n_valid > 0) {
            r.max2F = s_best[0];
            r.m = s_idx[0] / N_tau;
            r.n = s_idx[0] % N_tau;
            r.logB = (float)((double)Mall + log(s_S[0]));
        } else {
            r.max2F = 0.0f;
            r.m = -1;
            r.n = -1;
            r.logB = -INFINITY;
        }
        *out = r;
    }
}

// One CTA per template: combine its partials, write the result.
__global__ void __launch_bounds__(256)
    finalize_kernel(const Partial *__restrict__ partials, const int64_t per_template,
                    const int32_t N_tau, tfstat_result *__restrict__ out)
{
    finalize_body(partials + (int64_t)blockIdx.x * per_template, per_template, N_tau,
                  out + blockIdx.x);
}

// tfstat_marginalise: stream the map into one partial per CTA; finalize_kernel follows.  (One
// launch instead of two was measured and is no faster on B200: a cooperative launch with a grid
// barrier costs 8.6 us per call on a 2 MB map, a memset node for a last-CTA ticket 10.4 us, the
// two kernels chained by programmatic dependent launch 8.8 us: withdrawn since, tfstat_dev.cuh.)
__global__ void __launch_bounds__(kMargNT)
    marginalise_kernel(const float *__restrict__ map, const uint8_t *__restrict__ flags,
                       const int64_t n_cells, Partial *__restrict__ partials)
{
    __shared__ Marg s_red[32];
    Marg mg;
    if (flags) marginalise_body<true>(map, flags, n_cells, mg);
    else marginalise_body<false>(map, flags, n_cells, mg);
    marg_block_reduce<kMargNT>(mg, s_red);
    if (threadIdx.x == 0) partial_store(partials + blockIdx.x, mg);
}

}  // namespace

int32_t marginalise_blocks(int64_t n_cells)
{
    const int64_t per_block = (int64_t)kMargNT * 16;  // >= 16 cells per thread
    int64_t nb = (n_cells + per_block - 1) / per_block;
    if (nb < 1) nb = 1;
    if (nb > 148 * 8) nb = 148 * 8;
    return (int32_t)nb;
}

cudaError_t launch_finalize(const Partial *partials, int64_t partials_per_template,
                            int32_t n_templates, int32_t N_tau, tfstat_result *out,
                            cudaStream_t st)
{
    return launch_k(finalize_kernel, (unsigned)n_templates, 256, 0, st, partials,
                      partials_per_template, N_tau, out);
}

cudaError_t launch_marginalise(const float *map, const uint8_t *flags, int64_t n_cells,
                               int32_t N_tau, Partial *partials, int32_t n_blocks,
                               tfstat_result *out, cudaStream_t st)
{
    marginalise_kernel<<<n_blocks, kMargNT, 0, st>>>(map, flags, n_cells, partials);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return launch_finalize(partials, n_blocks, 1, N_tau, out, st);
}

}  // namespace tfstat
