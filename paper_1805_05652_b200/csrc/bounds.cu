// bounds.cu -- step a1: window -> atom-index bounds, and the term
// counter N_sums of eqs. (A.5)/(A.6) generalised to gaps.
//
// Membership is the half-open integer predicate t0_m <= t_alpha < t0_m + k tau_n
// (R3, R11).  Timestamps are shared by all templates, so this runs once per call.
#include "plan.h"

namespace tfstat {

__global__ void bounds_kernel(const int32_t *__restrict__ t, int n_atoms, Grid g, int64_t lat_g,
                              int64_t J, int32_t *__restrict__ lo, int32_t *__restrict__ edge)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < g.N_t0) lo[i] = lower_bound_t(t, n_atoms, t0_of(g, (int)i));
    if (i < J) {
        const long long base = (long long)g.t0_min + (long long)g.k * g.tau_min;
        edge[i] = lower_bound_t(t, n_atoms, base + (long long)i * lat_g);
    }
}

cudaError_t launch_bounds(const Plan &pl, const int32_t *t_atoms, void *ws, cudaStream_t st)
{
    int32_t *lo = reinterpret_cast<int32_t *>(static_cast<char *>(ws) + pl.off_lo);
    int32_t *edge = reinterpret_cast<int32_t *>(static_cast<char *>(ws) + pl.off_edge);
    const int64_t n = pl.J > pl.grid.N_t0 ? pl.J : pl.grid.N_t0;
    const int nt = 256;
    bounds_kernel<<<(unsigned)((n + nt - 1) / nt), nt, 0, st>>>(t_atoms, pl.n_atoms, pl.grid,
                                                                pl.g, pl.J, lo, edge);
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
    count_terms_kernel<<<(unsigned)nb, nt, 0, st>>>(
        pl.grid, b, reinterpret_cast<unsigned long long *>(out_terms));
    return cudaGetLastError();
}

}  // namespace tfstat
