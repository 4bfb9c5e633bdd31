// exp_direct.cu -- steps a0 + a3 + a4 + a5 for the exponential window, direct truncated sum
// ("brute-force grid", eq. (4) PAPER.md:44, 3 tau cut PAPER.md:52/238), fused with
// the cell closure (eq. 7) and the marginalisation, batched over templates.
//
// B200 design:
//  * one thread owns C cells (m0..m0+C-1, n): same tau, C consecutive t0.  For fixed tau the
//    weight exp(-(t - t0_c)/tau) = exp(-(t - t_ref)/tau) * const_c, and F is invariant under a
//    per-cell rescaling of the window (A,B,C ~ k^2, Fa,Fb ~ k), so ONE weight
//    w = exp(-(t - t_ref)/tau), t_ref = t0_{m0}, serves all C cells: 1 FMUL + 1 MUFU.EX2 +
//    1 FMUL per atom instead of per term, and 7 FFMA per term.
//  * lanes of a warp hold consecutive tau_n, so every lane reads the SAME atom: the atoms are
//    staged once per CTA in shared memory as two float4 per atom (dt, a2, b2, ab | Fa, Fb) and
//    read with broadcast LDS.128; int->float conversion of the timestamps happens once in the
//    staging, not in the loop (I2F shares the XU pipe with MUFU).
//  * the window of a CTA is streamed through shared memory in chunks of KC atoms, so a
//    1-year atom set (13 140 atoms, 420 KB) needs no more shared memory than a 1-day one.
//  * ragged window edges: atoms in [lo_{C-1}, min_lanes hi_0) belong to every cell of every
//    lane and are summed without predicates; only the short head and tail are predicated.
//  * CTAs are ordered heaviest (largest tau) first within a template.
#include "plan.h"

namespace tfstat {

namespace {

template <int C>
struct Acc {
    float A[C], B[C], Cc[C], far[C], fai[C], fbr[C], fbi[C];
};

template <int C, bool PRED>
__device__ __forceinline__ void accumulate(Acc<C> &acc, const float4 a, const float4 b,
                                           const float kexp, const int alpha,
                                           const int (&lo)[C], const int (&hi)[C])
{
    const float w = ex2_approx(a.x * kexp);
    const float w2 = w * w;
#pragma unroll
    for (int c = 0; c < C; ++c) {
        if (!PRED || (alpha >= lo[c] && alpha < hi[c])) {
            acc.A[c] = fmaf(w2, a.y, acc.A[c]);
            acc.B[c] = fmaf(w2, a.z, acc.B[c]);
            acc.Cc[c] = fmaf(w2, a.w, acc.Cc[c]);
            acc.far[c] = fmaf(w, b.x, acc.far[c]);
            acc.fai[c] = fmaf(w, b.y, acc.fai[c]);
            acc.fbr[c] = fmaf(w, b.z, acc.fbr[c]);
            acc.fbi[c] = fmaf(w, b.w, acc.fbi[c]);
        }
    }
}

template <int C, int NT, int KC>
__global__ void __launch_bounds__(NT)
    exp_direct_kernel(const Problem pr, Partial *__restrict__ partials, const int n_mtiles,
                      const int n_nblocks)
{
    __shared__ float4 s_a[KC];
    __shared__ float4 s_b[KC];
    __shared__ Marg s_red[32];

    const Grid g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int64_t tiles = (int64_t)n_mtiles * n_nblocks;
    const int tpl = (int)(blockIdx.x / tiles);
    const int tile = (int)(blockIdx.x % tiles);
    const int nb = n_nblocks - 1 - tile / n_mtiles;  // heaviest (largest tau) first
    const int m0 = (tile % n_mtiles) * C;
    const int n_raw = nb * NT + threadIdx.x;
    const bool n_ok = n_raw < g.N_tau;
    const int n = n_ok ? n_raw : g.N_tau - 1;  // clamped duplicate, result discarded

    int lo[C], hi[C];
#pragma unroll
    for (int c = 0; c < C; ++c) {
        const int mc = min(m0 + c, g.N_t0 - 1);
        lo[c] = __ldg(bd.lo + mc);
        hi[c] = max(hi_index(bd, g, mc, n), lo[c]);
    }
    // atom range of the CTA
    const int a_begin = lo[0];
    const int a_end = hi_index(bd, g, min(m0 + C - 1, g.N_t0 - 1),
                               min(nb * NT + NT - 1, g.N_tau - 1));
    const int core_b = lo[C - 1];
    const int core_e = __reduce_min_sync(0xffffffffu, hi[0]);

    const long long t_ref = t0_of(g, m0);
    const float kexp = (float)(-1.4426950408889634 / (double)tau_of(g, n));

    const float *__restrict__ base = pr.atoms + (int64_t)tpl * pr.template_stride;
    const int64_t ld = pr.ld;

    Acc<C> acc;
#pragma unroll
    for (int c = 0; c < C; ++c)
        acc.A[c] = acc.B[c] = acc.Cc[c] = acc.far[c] = acc.fai[c] = acc.fbr[c] = acc.fbi[c] = 0.f;

    for (int cs = a_begin; cs < a_end; cs += KC) {
        const int ce = min(cs + KC, a_end);
        // ---- a0: stage atoms [cs, ce) -------------------------------------------------
        for (int i = threadIdx.x; i < ce - cs; i += NT) {
            const int al = cs + i;
            float4 a, b;
            a.x = (float)((long long)__ldg(bd.t + al) - t_ref);
            a.y = __ldg(base + al);
            a.z = __ldg(base + ld + al);
            a.w = __ldg(base + 2 * ld + al);
            b.x = __ldg(base + 3 * ld + al);
            b.y = __ldg(base + 4 * ld + al);
            b.z = __ldg(base + 5 * ld + al);
            b.w = __ldg(base + 6 * ld + al);
            s_a[i] = a;
            s_b[i] = b;
        }
        __syncthreads();
        // ---- a3: weighted sums over this chunk -----------------------------------------
        const int x0 = max(cs, lo[0]);
        const int x3 = min(ce, hi[C - 1]);
        const int s1 = min(x3, max(x0, core_b));
        const int s2 = min(x3, max(s1, core_e));
        for (int al = x0; al < s1; ++al)
            accumulate<C, true>(acc, s_a[al - cs], s_b[al - cs], kexp, al, lo, hi);
#pragma unroll 4
        for (int al = s1; al < s2; ++al)
            accumulate<C, false>(acc, s_a[al - cs], s_b[al - cs], kexp, al, lo, hi);
        for (int al = s2; al < x3; ++al)
            accumulate<C, true>(acc, s_a[al - cs], s_b[al - cs], kexp, al, lo, hi);
        __syncthreads();
    }

    // ---- a4 closure + a5 marginals ----------------------------------------------------
    Marg mg;
    marg_init(mg);
    const int64_t map_base = (int64_t)tpl * g.N_t0 * g.N_tau;
#pragma unroll
    for (int c = 0; c < C; ++c) {
        const int m = m0 + c;
        if (n_ok && m < g.N_t0) {
            Sums64 s;
            s.A = acc.A[c];
            s.B = acc.B[c];
            s.C = acc.Cc[c];
            s.far = acc.far[c];
            s.fai = acc.fai[c];
            s.fbr = acc.fbr[c];
            s.fbi = acc.fbi[c];
            uint32_t fl;
            const float twoF = closure_2F(s, hi[c] - lo[c], pr.min_atoms, fl);
            const int32_t flat = m * g.N_tau + n;
            if (pr.out_maps) pr.out_maps[map_base + flat] = twoF;
            if (pr.out_flags) pr.out_flags[map_base + flat] = (uint8_t)fl;
            if (!fl) marg_add(mg, twoF, flat);
        }
    }
    if (partials) {
        marg_block_reduce<NT>(mg, s_red);
        if (threadIdx.x == 0) partial_store(partials + blockIdx.x, mg);
    }
}

template <int C, int NT>
cudaError_t launch_one(const Plan &pl, const Problem &pr, Partial *partials, cudaStream_t st)
{
    const int64_t n_ctas = pl.tiles_per_template * pl.n_templates;
    exp_direct_kernel<C, NT, 1024><<<(unsigned)n_ctas, NT, 0, st>>>(pr, partials, pl.n_mtiles,
                                                                    pl.n_nblocks);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_exp_direct(const Plan &pl, const Problem &pr, Partial *partials,
                              cudaStream_t st)
{
    if (pl.tile.C == 8 && pl.tile.NT == 256) return launch_one<8, 256>(pl, pr, partials, st);
    if (pl.tile.C == 4 && pl.tile.NT == 128) return launch_one<4, 128>(pl, pr, partials, st);
    if (pl.tile.C == 2 && pl.tile.NT == 64) return launch_one<2, 64>(pl, pr, partials, st);
    return cudaErrorInvalidValue;
}

}  // namespace tfstat
