// bounds.cu -- step a1: window -> atom-index bounds, and the term
// counter N_sums of eqs. (A.5)/(A.6) generalised to gaps.
//
// Membership is the half-open integer predicate t0_m <= t_alpha < t0_m + k tau_n
// (R3, R11).  Timestamps are shared by all templates, so this runs once per call.
#include "plan.h"

namespace tfstat {

// One lower_bound per t0 and per lattice point.  A plain binary search is a chain of ~log2(N)
// dependent global loads; here every CTA first stages a coarse sample of the timestamps (the
// last one of every `stride` atoms, at most kMaxSamples of them) in shared memory, searches
// that, and finishes with independent loads inside one block of atoms: two global round
// trips instead of log2(N).
constexpr int kBoundsNT = 256;
constexpr int kMaxSamples = 4096;

__device__ __forceinline__ int sampled_lower_bound(const int32_t *__restrict__ t, const int n,
                                                   const int32_t *__restrict__ s_t,
                                                   const int n_samples, const int stride,
                                                   const long long x)
{
    int a = 0, b = n_samples;  // first sample >= x
    while (a < b) {
        const int mid = (a + b) >> 1;
        if ((long long)s_t[mid] < x) a = mid + 1;
        else b = mid;
    }
    if (a == n_samples) return n;
    int lo = a * stride, hi = min(lo + stride, n);  // the answer is in [lo, hi)
    while (hi - lo > 16) {
        const int mid = (lo + hi) >> 1;
        if ((long long)__ldg(t + mid) < x) lo = mid + 1;
        else hi = mid;
    }
    int v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = (lo + i < hi) ? __ldg(t + lo + i) : INT32_MAX;
    int cnt = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) cnt += (lo + i < hi && (long long)v[i] < x) ? 1 : 0;
    return lo + cnt;
}

__global__ void __launch_bounds__(kBoundsNT)
    bounds_kernel(const int32_t *__restrict__ t, int n_atoms, Grid g, int64_t lat_g, int64_t J,
                  int stride, int n_samples, int32_t *__restrict__ lo,
                  int32_t *__restrict__ edge, int32_t *__restrict__ zero, int64_t n_zero)
{
    // scan flags of the rectangular path (rect.cu), zeroed here to save a memset node
    for (int64_t z = (int64_t)blockIdx.x * kBoundsNT + threadIdx.x; z < n_zero;
         z += (int64_t)gridDim.x * kBoundsNT)
        zero[z] = 0;
    __shared__ int32_t s_t[kMaxSamples];
    for (int i = threadIdx.x; i < n_samples; i += kBoundsNT)
        s_t[i] = __ldg(t + min((i + 1) * stride - 1, n_atoms - 1));
    __syncthreads();
    const int64_t i = (int64_t)blockIdx.x * kBoundsNT + threadIdx.x;
    if (i < g.N_t0)
        lo[i] = sampled_lower_bound(t, n_atoms, s_t, n_samples, stride, t0_of(g, (int)i));
    if (i < J) {
        const long long base = (long long)g.t0_min + (long long)g.k * g.tau_min;
        edge[i] =
            sampled_lower_bound(t, n_atoms, s_t, n_samples, stride, base + (long long)i * lat_g);
    }
}

cudaError_t launch_bounds(const Plan &pl, const int32_t *t_atoms, void *ws, cudaStream_t st)
{
    int32_t *lo = reinterpret_cast<int32_t *>(static_cast<char *>(ws) + pl.off_lo);
    int32_t *edge = reinterpret_cast<int32_t *>(static_cast<char *>(ws) + pl.off_edge);
    const int64_t n = pl.J > pl.grid.N_t0 ? pl.J : pl.grid.N_t0;
    int stride = 16;
    while ((pl.n_atoms + stride - 1) / stride > kMaxSamples) stride <<= 1;
    const int n_samples = (pl.n_atoms + stride - 1) / stride;
    bounds_kernel<<<(unsigned)((n + kBoundsNT - 1) / kBoundsNT), kBoundsNT, 0, st>>>(
        t_atoms, pl.n_atoms, pl.grid, pl.g, pl.J, stride, n_samples, lo, edge,
        reinterpret_cast<int32_t *>(static_cast<char *>(ws) + pl.off_flags),
        (int64_t)(pl.flags_bytes / sizeof(int32_t)));
    return cudaGetLastError();
}

// Opt-in validator of the precondition "time stamps strictly increasing" (include/tfstat.h).
__global__ void validate_timestamps_kernel(const int32_t *__restrict__ t, const int n,
                                           unsigned *__restrict__ first_bad)
{
    unsigned bad = 0xffffffffu;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x + 1; i < n;
         i += (int64_t)gridDim.x * blockDim.x)
        if (__ldg(t + i) <= __ldg(t + i - 1)) bad = min(bad, (unsigned)i);
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) bad = min(bad, __shfl_xor_sync(0xffffffffu, bad, s));
    if ((threadIdx.x & 31) == 0 && bad != 0xffffffffu) atomicMin(first_bad, bad);
}

cudaError_t launch_validate_timestamps(const int32_t *t_atoms, int32_t n_atoms,
                                       int32_t *out_first_bad, cudaStream_t st)
{
    // -1 = 0xffffffff is also the identity of the unsigned minimum
    cudaError_t e = cudaMemsetAsync(out_first_bad, 0xff, sizeof(int32_t), st);
    if (e != cudaSuccess) return e;
    const int nt = 256;
    int nb = (n_atoms + nt - 1) / nt;
    if (nb > 148 * 8) nb = 148 * 8;
    validate_timestamps_kernel<<<nb, nt, 0, st>>>(t_atoms, n_atoms,
                                                  reinterpret_cast<unsigned *>(out_first_bad));
    return cudaGetLastError();
}

__global__ void count_terms_kernel(Grid g, Bounds b, unsigned long long *out)
{
    const int64_t n_cells = (int64_t)g.N_t0 * g.N_tau;
    unsigned long long acc = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_cells;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int m = (int)(i / g.N_tau), n = (int)(i % g.N_tau);
        const int lo = __ldg(b.lo + m);
        const int hi = hi_index(b, g, m, n);
        acc += (unsigned long long)(hi > lo ? hi - lo : 0);
    }
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
    if ((threadIdx.x & 31) == 0 && acc) atomicAdd(out, acc);
}

cudaError_t launch_count_terms(const Plan &pl, const Bounds &b, int64_t *out_terms,
                               cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(out_terms, 0, sizeof(int64_t), st);
    if (e != cudaSuccess) return e;
    const int64_t n_cells = (int64_t)pl.grid.N_t0 * pl.grid.N_tau;
    const int nt = 256;
    int64_t nb = (n_cells + nt - 1) / nt;
    if (nb > 148 * 16) nb = 148 * 16;
    count_terms_kernel<<<(unsigned)nb, nt, 0, st>>>(  // follows a memset node: plain launch
        pl.grid, b, reinterpret_cast<unsigned long long *>(out_terms));
    return cudaGetLastError();
}

}  // namespace tfstat
