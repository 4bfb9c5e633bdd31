// marginalise.cu -- step a5 on a map already in HBM (tfstat_marginalise) and the final
// cross-CTA combine of the fused kernels' partial marginals.
//
// max 2F with lowest-flat-index argmax and logB = log sum_valid exp(2F/2) (eq. 5, PAPER.md:56;
// DESIGN.md R13, R14).  Streaming, HBM-bound: 4 B (+1 B flags) per cell.
#include "plan.h"

namespace tfstat {

namespace {

constexpr int kMargNT = 256;

__device__ __forceinline__ void marg_add4(Marg &a, const float4 v, const uint32_t fl4,
                                          const int32_t flat0)
{
    const float x[4] = {v.x, v.y, v.z, v.w};
    float m4 = -INFINITY;
    int nv = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const bool ok = ((fl4 >> (8 * j)) & 0xffu) == 0u;
        if (ok) {
            if (x[j] > a.best) {  // ascending flat index within a thread: '>' keeps the lowest
                a.best = x[j];
                a.idx = flat0 + j;
            }
            m4 = fmaxf(m4, 0.5f * x[j]);
            nv += 1;
        }
    }
    if (nv == 0) return;
    if (m4 > a.M) {
        a.S *= ex2_approx((a.M - m4) * TFSTAT_LOG2E_F);
        a.M = m4;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const bool ok = ((fl4 >> (8 * j)) & 0xffu) == 0u;
        if (ok) a.S += ex2_approx((0.5f * x[j] - a.M) * TFSTAT_LOG2E_F);
    }
    a.nvalid += nv;
}

__global__ void __launch_bounds__(kMargNT)
    marginalise_kernel(const float *__restrict__ map, const uint8_t *__restrict__ flags,
                       const int64_t n_cells, Partial *__restrict__ partials)
{
    __shared__ Marg s_red[32];
    Marg mg;
    marg_init(mg);
    const bool vec = ((reinterpret_cast<uintptr_t>(map) & 15u) == 0) &&
                     (!flags || (reinterpret_cast<uintptr_t>(flags) & 3u) == 0);
    const int64_t n4 = vec ? n_cells / 4 : 0;
    const int64_t stride = (int64_t)gridDim.x * kMargNT;
    // each thread walks ascending indices, so ties inside a thread keep the lowest index
    for (int64_t q = (int64_t)blockIdx.x * kMargNT + threadIdx.x; q < n4; q += stride) {
        const float4 v = __ldcs(reinterpret_cast<const float4 *>(map) + q);
        const uint32_t f = flags ? __ldcs(reinterpret_cast<const uint32_t *>(flags) + q) : 0u;
        marg_add4(mg, v, f, (int32_t)(4 * q));
    }
    for (int64_t i = 4 * n4 + (int64_t)blockIdx.x * kMargNT + threadIdx.x; i < n_cells;
         i += stride) {
        if (!flags || flags[i] == 0) marg_add(mg, map[i], (int32_t)i);
    }
    marg_block_reduce<kMargNT>(mg, s_red);
    if (threadIdx.x == 0) partial_store(partials + blockIdx.x, mg);
}

// One CTA per template: combine its partials (fixed order -> deterministic), write the result.
__global__ void __launch_bounds__(256)
    finalize_kernel(const Partial *__restrict__ partials, const int64_t per_template,
                    const int32_t N_tau, tfstat_result *__restrict__ out)
{
    __shared__ float s_best[256];
    __shared__ int32_t s_idx[256];
    __shared__ float s_M[256];
    __shared__ double s_S[256];
    __shared__ int32_t s_nv[256];
    const Partial *__restrict__ p = partials + (int64_t)blockIdx.x * per_template;
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
        out[blockIdx.x] = r;
    }
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
    finalize_kernel<<<n_templates, 256, 0, st>>>(partials, partials_per_template, N_tau, out);
    return cudaGetLastError();
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
