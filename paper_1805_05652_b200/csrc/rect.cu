// rect.cu -- steps a2 + a4 + a5 for the rectangular window (eq. 3).
//
// The paper keeps running partial sums over tau per t0 (N_t0 workers).  Here every
// cell is independent: S(m,n) = P[hi(m,n)] - P[lo(m)] with P the exclusive prefix sums of the
// 7 atom channels.  P is kept in fp64: an fp32 prefix over a year of atoms cancels
// catastrophically for short windows far from the origin, fp64 differences of
// fp32 data are exact to ~1e-13.  The closure (eq. 7) runs in fp64 on those differences.
#include "plan.h"

namespace tfstat {

namespace {

constexpr int kPrefixNT = 1024;

// P[tpl][i][ch], i = 0..n_atoms, ch = 0..7 (7 used): 64 B per entry.
__global__ void __launch_bounds__(kPrefixNT)
    rect_prefix_kernel(const Problem pr, double *__restrict__ prefix)
{
    __shared__ double s_warp[7][32];
    const int tpl = blockIdx.x;
    const int N = pr.bounds.n_atoms;
    const float *__restrict__ base = pr.atoms + (int64_t)tpl * pr.template_stride;
    double *__restrict__ P = prefix + (int64_t)tpl * (N + 1) * 8;
    const int seg = (N + kPrefixNT - 1) / kPrefixNT;
    const int a0 = min((int)threadIdx.x * seg, N), a1 = min(a0 + seg, N);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    double tot[7];
#pragma unroll
    for (int ch = 0; ch < 7; ++ch) {
        double s = 0.0;
        for (int al = a0; al < a1; ++al) s += (double)__ldg(base + ch * pr.ld + al);
        tot[ch] = s;
    }
    // inclusive scan of the per-thread totals across the block
    double incl[7];
#pragma unroll
    for (int ch = 0; ch < 7; ++ch) {
        double v = tot[ch];
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) {
            const double u = __shfl_up_sync(0xffffffffu, v, s);
            if (lane >= s) v += u;
        }
        incl[ch] = v;
        if (lane == 31) s_warp[ch][warp] = v;
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int ch = 0; ch < 7; ++ch) {
            double v = s_warp[ch][lane];
#pragma unroll
            for (int s = 1; s < 32; s <<= 1) {
                const double u = __shfl_up_sync(0xffffffffu, v, s);
                if (lane >= s) v += u;
            }
            s_warp[ch][lane] = v;
        }
    }
    __syncthreads();
#pragma unroll
    for (int ch = 0; ch < 7; ++ch) {
        double run = incl[ch] - tot[ch] + (warp > 0 ? s_warp[ch][warp - 1] : 0.0);
        for (int al = a0; al < a1; ++al) {
            run += (double)__ldg(base + ch * pr.ld + al);
            P[(int64_t)(al + 1) * 8 + ch] = run;
            if (ch == 6) P[(int64_t)(al + 1) * 8 + 7] = 0.0;  // pad lane of the 64-B entry
        }
    }
    if (threadIdx.x < 8) P[threadIdx.x] = 0.0;
}

constexpr int kCellNT = 256;

__global__ void __launch_bounds__(kCellNT)
    rect_cells_kernel(const Problem pr, const double *__restrict__ prefix,
                      Partial *__restrict__ partials, const int blocks_per_template)
{
    __shared__ Marg s_red[32];
    const Grid g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int tpl = blockIdx.x / blocks_per_template;
    const int blk = blockIdx.x % blocks_per_template;
    const int64_t n_cells = (int64_t)g.N_t0 * g.N_tau;
    const int64_t i = (int64_t)blk * kCellNT + threadIdx.x;
    Marg mg;
    marg_init(mg);
    if (i < n_cells) {
        const int m = (int)(i / g.N_tau), n = (int)(i % g.N_tau);
        const int lo = __ldg(bd.lo + m);
        const int hi = max(hi_index(bd, g, m, n), lo);
        const double2 *__restrict__ P = reinterpret_cast<const double2 *>(
            prefix + (int64_t)tpl * (bd.n_atoms + 1) * 8);
        const double2 l0 = __ldg(P + (int64_t)lo * 4), l1 = __ldg(P + (int64_t)lo * 4 + 1),
                      l2 = __ldg(P + (int64_t)lo * 4 + 2), l3 = __ldg(P + (int64_t)lo * 4 + 3);
        const double2 h0 = __ldg(P + (int64_t)hi * 4), h1 = __ldg(P + (int64_t)hi * 4 + 1),
                      h2 = __ldg(P + (int64_t)hi * 4 + 2), h3 = __ldg(P + (int64_t)hi * 4 + 3);
        Sums64 s;
        s.A = h0.x - l0.x;
        s.B = h0.y - l0.y;
        s.C = h1.x - l1.x;
        s.far = h1.y - l1.y;
        s.fai = h2.x - l2.x;
        s.fbr = h2.y - l2.y;
        s.fbi = h3.x - l3.x;
        uint32_t fl;
        const float twoF = closure_2F(s, hi - lo, pr.min_atoms, fl);
        const int64_t o = (int64_t)tpl * n_cells + i;
        if (pr.out_maps) pr.out_maps[o] = twoF;
        if (pr.out_flags) pr.out_flags[o] = (uint8_t)fl;
        if (!fl) marg_add(mg, twoF, (int32_t)i);
    }
    if (partials) {
        marg_block_reduce<kCellNT>(mg, s_red);
        if (threadIdx.x == 0) partial_store(partials + blockIdx.x, mg);
    }
}

}  // namespace

cudaError_t launch_rect(const Plan &pl, const Problem &pr, double *prefix, Partial *partials,
                        cudaStream_t st)
{
    rect_prefix_kernel<<<pl.n_templates, kPrefixNT, 0, st>>>(pr, prefix);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const int64_t n_ctas = (int64_t)pl.cell_blocks_per_template * pl.n_templates;
    rect_cells_kernel<<<(unsigned)n_ctas, kCellNT, 0, st>>>(pr, prefix, partials,
                                                            pl.cell_blocks_per_template);
    return cudaGetLastError();
}

}  // namespace tfstat
