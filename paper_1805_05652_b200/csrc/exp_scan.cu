// exp_scan.cu -- steps a0 + a3' + a4 + a5: the exponential window in its exact FACTORISED,
// SLIDING form (SURVEY.md 8(a) row a3', BASELINE.json north_star "exact factorised form
// exp(-(t-t0)/tau) = exp(t0/tau) exp(-t/tau) ... kept only if it matches the oracle").
//
// The paper sums every cell's window on its own ("brute-force grid").  But for a
// fixed tau_n the weights of all t0 share one series:
//     exp(-(t_a - t0_m)/tau) = exp(-(t_a - t_ref)/tau) * exp(-(t_ref - t0_m)/tau),
// and eq. (7) is invariant under a per-cell rescaling of the window (A,B,C ~ k^2, Fa,Fb ~ k;
// DESIGN.md invariant I3), so the per-cell factor never has to be applied.  With
//     E_a = exp(-(t_a - t_ref)/tau)
// the window sums of cell m are  W_m = sum_{a in [lo_m, hi_mn)} E_a x_a  (E_a^2 for a2,b2,ab),
// and neighbouring cells differ by the few atoms that enter at the low end and leave at the
// high end:
//     W_{m-1} = W_m + sum_{[lo_{m-1}, lo_m)} E_a x_a - sum_{[hi_{m-1,n}, hi_{m,n})} E_a x_a.
// One thread owns one tau_n and slides BACKWARDS in t0 (the stable direction: entering atoms
// carry the largest weights of the window, leaving atoms the smallest, ~e^-3 of them, so the
// subtraction never cancels the bulk of the sum).  Every weight is computed directly from its
// time stamp (no multiplicative recurrence, hence no drift), an atom leaves with the same weight
// it entered with, and t_ref is moved (accumulators rescaled by one exp) whenever
// (t_ref - t0_m)/tau exceeds kReanchor so nothing overflows.  If a window loses most of its
// weight (gaps, end of data) or does not overlap its neighbour, it is summed afresh.
//
// Work per (template, tau): |window of the last t0| + 2 atoms per t0 step, instead of
// |window| atoms per cell: 60x fewer weighted terms on BASELINE.json config 4, 300x on
// config 5.  Terms/s reported for this path are EFFECTIVE terms (eq. A.6 count / time).
//
// Layout: lanes of a warp hold consecutive tau_n (same template), so the initial window is
// streamed through shared memory and broadcast exactly like exp_direct.cu; a CTA is
// (template, block of NT tau, segment of t0).  Long t0 grids with few tau (config 5) are cut
// into segments, each with its own initial sum, to fill the GPU.
#include "plan.h"

// unroll of the initial-window loop: swept 2..32 on B200, 16 is 4-5 % faster than 4
constexpr int kWindowUnroll = 16;
namespace tfstat {

namespace {

constexpr float kReanchor = 4.0f;  // move t_ref when (t_ref - t0_m)/tau exceeds this
constexpr float kGuard = 64.0f;    // re-sum a window whose A fell below 1/kGuard of its maximum

struct SlideAcc {
    u64 ab;  // (A, B)
    u64 fa;  // (Re Fa, Im Fa)
    u64 fb;  // (Re Fb, Im Fb)
    float c;
};

__device__ __forceinline__ void acc_zero(SlideAcc &a)
{
    a.ab = a.fa = a.fb = 0ull;
    a.c = 0.0f;
}

// acc += s * E x  (s = +1 entering, -1 leaving): w carries the sign, w2 = w * |w|
__device__ __forceinline__ void acc_add(SlideAcc &a, const float w, const float w2, const u64 a2b2,
                                        const float ab, const u64 fa, const u64 fb)
{
    const u64 ww = pack2(w, w);
    ffma2(a.ab, pack2(w2, w2), a2b2);
    ffma2(a.fa, ww, fa);
    ffma2(a.fb, ww, fb);
    a.c = fmaf(w2, ab, a.c);
}

// atom `al` straight from global memory (entering / leaving / re-summed atoms), one weight for
// the TPC templates of the CTA
template <int TPC>
__device__ __forceinline__ void acc_add_global(SlideAcc (&a)[TPC],
                                               const float *__restrict__ const (&base)[TPC],
                                               const int64_t ld, const int32_t *__restrict__ t,
                                               const int al, const long long t_ref,
                                               const float kexp, const float sign)
{
    const float dt = (float)((long long)__ldg(t + al) - t_ref);
    const float e = ex2_approx(dt * kexp);
    const float w = sign * e;
    const float w2 = w * e;
#pragma unroll
    for (int q = 0; q < TPC; ++q) {
        const float *__restrict__ bq = base[q];
        acc_add(a[q], w, w2, pack2(__ldg(bq + al), __ldg(bq + ld + al)), __ldg(bq + 2 * ld + al),
                pack2(__ldg(bq + 3 * ld + al), __ldg(bq + 4 * ld + al)),
                pack2(__ldg(bq + 5 * ld + al), __ldg(bq + 6 * ld + al)));
    }
}

__device__ __forceinline__ void acc_scale(SlideAcc &a, const float c)
{
    const float c2 = c * c;
    a.ab = fmul2(a.ab, pack2(c2, c2));
    a.fa = fmul2(a.fa, pack2(c, c));
    a.fb = fmul2(a.fb, pack2(c, c));
    a.c *= c2;
}

// TPC templates per CTA: the weights E_a depend on (atom, tau) only, not on the template, so one
// MUFU.EX2 (+ the argument and E^2 multiplies) serves TPC templates; per (atom, template) the
// initial window sum costs 2 LDS.128 + 4 multiply-adds + 3 / TPC instead of + 3.
// Resident CTAs per SM asked of ptxas (measured on B200, config 4 x 2048 templates): one
// template per CTA 5.26 ms unconstrained (96 registers), 5.09 at 5 CTAs, 4.85 at 6 (80 registers);
// two templates 4.56 unconstrained (128 registers), 4.47 at 5 (96), 5.10 at 6 (spills).
template <int NT, int KC, int TPC>
__global__ void __launch_bounds__(NT, TPC == 1 ? (NT == 128 ? 6 : 1) : TPC == 2 ? (NT == 128 ? 5 : 1) : 1)
    exp_slide_kernel(const Problem pr, Partial *__restrict__ partials, const int n_nblocks,
                     const int n_segs, const int seg_len)
{
    __shared__ ulonglong2 s_a[TPC][KC];  // {(dt, ab), (a2, b2)}
    __shared__ ulonglong2 s_b[TPC][KC];  // {(Re Fa, Im Fa), (Re Fb, Im Fb)}
    __shared__ Marg s_red[32];
    pdl_trigger();
    pdl_wait();  // bounds_kernel's lo / edge tables

    const Grid g = pr.grid;
    const Bounds &bd = pr.bounds;
    // blockIdx.x = (tplgrp * n_segs + seg) * n_nblocks + j, heaviest tau block (largest tau) first
    const int j = (int)(blockIdx.x % n_nblocks);
    const int seg = (int)((blockIdx.x / n_nblocks) % n_segs);
    const int tpl0 = (int)(blockIdx.x / ((int64_t)n_nblocks * n_segs)) * TPC;
    const int nb = n_nblocks - 1 - j;
    const int n_first = nb * NT;
    const int n_count = min(NT, g.N_tau - n_first);
    const bool n_ok = (int)threadIdx.x < n_count;
    const int n = n_first + (n_ok ? (int)threadIdx.x : 0);
    const int m_beg = seg * seg_len;
    const int m_end = min(m_beg + seg_len, g.N_t0);

    // templates beyond the batch (ragged last group) alias the last real one; nothing of theirs
    // is stored
    const float *__restrict__ base[TPC];
#pragma unroll
    for (int q = 0; q < TPC; ++q)
        base[q] = pr.atoms + (int64_t)min(tpl0 + q, pr.n_templates - 1) * pr.template_stride;
    const int64_t ld = pr.ld;
    const double tau = (double)tau_of(g, n);
    const float kexp = (float)(-1.4426950408889634 / tau);
    const float inv_tau = (float)(1.0 / tau);

    // ---- initial window: cell (m_end - 1, n), streamed through shared memory -----------------
    int m = m_end - 1;
    int lo_m = __ldg(bd.lo + m);
    int hi = n_ok ? max(hi_index(bd, g, m, n), lo_m) : lo_m;
    long long t_ref = t0_of(g, m);
    const int cta_e = max(hi_index(bd, g, m, n_first + n_count - 1), lo_m);  // hi is monotone in n

    SlideAcc acc[TPC];
#pragma unroll
    for (int q = 0; q < TPC; ++q) acc_zero(acc[q]);
#pragma unroll 1
    for (int cs = lo_m; cs < cta_e; cs += KC) {
        const int n_stage = min(KC, cta_e - cs);
        for (int i = threadIdx.x; i < n_stage; i += NT) {
            const int al = cs + i;
            const float dt = (float)((long long)__ldg(bd.t + al) - t_ref);
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                const float *__restrict__ bq = base[q];
                ulonglong2 ra, rb;
                ra.x = pack2(dt, __ldg(bq + 2 * ld + al));
                ra.y = pack2(__ldg(bq + al), __ldg(bq + ld + al));
                rb.x = pack2(__ldg(bq + 3 * ld + al), __ldg(bq + 4 * ld + al));
                rb.y = pack2(__ldg(bq + 5 * ld + al), __ldg(bq + 6 * ld + al));
                s_a[q][i] = ra;
                s_b[q][i] = rb;
            }
        }
        __syncthreads();
        const int x1 = min(cs + n_stage, hi) - cs;
#pragma unroll kWindowUnroll
        for (int i = 0; i < x1; ++i) {
            float e = 0.0f, e2 = 0.0f;
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                const ulonglong2 ra = s_a[q][i], rb = s_b[q][i];
                float dt, ab;
                unpack2(ra.x, dt, ab);
                if (q == 0) {
                    e = ex2_approx(dt * kexp);
                    e2 = e * e;
                }
                acc_add(acc[q], e, e2, ra.y, ab, rb.x, rb.y);
            }
        }
        __syncthreads();
    }
    float A_max[TPC];
#pragma unroll
    for (int q = 0; q < TPC; ++q) {
        float A, B;
        unpack2(acc[q].ab, A, B);
        A_max[q] = A;
    }

    // ---- slide backwards in t0: closure of cell m, then step to m - 1 ------------------------
    Marg mg[TPC];
#pragma unroll
    for (int q = 0; q < TPC; ++q) marg_init(mg[q]);
    const int64_t cells = (int64_t)g.N_t0 * g.N_tau;
#pragma unroll 1
    for (;;) {
        if (n_ok) {
            const int32_t flat = m * g.N_tau + n;
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                if (tpl0 + q >= pr.n_templates) continue;
                float A, B, far, fai, fbr, fbi;
                unpack2(acc[q].ab, A, B);
                unpack2(acc[q].fa, far, fai);
                unpack2(acc[q].fb, fbr, fbi);
                uint32_t fl;
                // one closure per t0 step is a quarter of this kernel's instructions in fp64
                const float twoF =
                    closure_2F_exp<true>(A, B, acc[q].c, far, fai, fbr, fbi, lo_m, hi - lo_m,
                                   pr.min_atoms, fl, base[q], ld, bd.t, t0_of(g, m), tau);
                const int64_t o = (int64_t)(tpl0 + q) * cells + flat;
                if (pr.out_maps) pr.out_maps[o] = twoF;
                if (pr.out_flags) pr.out_flags[o] = (uint8_t)fl;
                if (!fl) marg_add(mg[q], twoF, flat);
            }
        }
        if (m == m_beg) break;
        const int m2 = m - 1;
        const int lo2 = __ldg(bd.lo + m2);
        const int hi2 = n_ok ? max(hi_index(bd, g, m2, n), lo2) : lo2;
        const long long t0_2 = t0_of(g, m2);
        bool fresh = (hi2 <= lo_m) || (hi2 == lo2);  // no overlap with window m, or empty
        if (!fresh) {
            const float sh = (float)(t_ref - t0_2);
            if (sh * inv_tau > kReanchor) {  // keep the weights of entering atoms <= e^kReanchor
                const float c = ex2_approx(sh * kexp);
#pragma unroll
                for (int q = 0; q < TPC; ++q) {
                    acc_scale(acc[q], c);
                    A_max[q] *= c * c;
                }
                t_ref = t0_2;
            }
            for (int al = lo2; al < lo_m; ++al)  // entering at the low end
                acc_add_global<TPC>(acc, base, ld, bd.t, al, t_ref, kexp, 1.0f);
            for (int al = max(hi2, lo_m); al < hi; ++al)  // leaving at the high end
                acc_add_global<TPC>(acc, base, ld, bd.t, al, t_ref, kexp, -1.0f);
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                float A, B;
                unpack2(acc[q].ab, A, B);
                A_max[q] = fmaxf(A_max[q], A);
                // a window that lost most of its weight is re-summed (for all TPC templates:
                // a fresh sum is always right)
                // (written so that a NaN / inf atom in the running sums also forces a fresh
                // sum: once it has left the window it must not linger)
                fresh = fresh || !(A * kGuard >= A_max[q]);
            }
        }
        if (fresh) {
#pragma unroll
            for (int q = 0; q < TPC; ++q) acc_zero(acc[q]);
            t_ref = t0_2;
            for (int al = lo2; al < hi2; ++al)
                acc_add_global<TPC>(acc, base, ld, bd.t, al, t_ref, kexp, 1.0f);
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                float A, B;
                unpack2(acc[q].ab, A, B);
                A_max[q] = A;
            }
        }
        m = m2;
        lo_m = lo2;
        hi = hi2;
    }
    if (partials) {
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
            if (q > 0) __syncthreads();  // s_red is reused
            marg_block_reduce<NT>(mg[q], s_red);
            if (threadIdx.x == 0 && tpl0 + q < pr.n_templates)
                partial_store(partials + ((int64_t)(tpl0 + q) * n_segs + seg) * n_nblocks + j,
                              mg[q]);
        }
    }
}

template <int NT, int TPC>
cudaError_t launch_tpc(const Plan &pl, const Problem &pr, Partial *partials, cudaStream_t st)
{
    const int64_t groups = (pl.n_templates + TPC - 1) / TPC;
    const int64_t n_ctas = (int64_t)pl.n_nblocks * pl.n_segs * groups;
    return launch_pdl(exp_slide_kernel<NT, (TPC == 4 ? 256 : 512), TPC>, (unsigned)n_ctas, NT, 0,
                      st, pr, partials, pl.n_nblocks, pl.n_segs, pl.seg_len);
}

template <int NT>
cudaError_t launch_nt(const Plan &pl, const Problem &pr, Partial *partials, cudaStream_t st)
{
    switch (pl.slide_tpc) {
    case 4: return launch_tpc<NT, 4>(pl, pr, partials, st);
    case 2: return launch_tpc<NT, 2>(pl, pr, partials, st);
    default: return launch_tpc<NT, 1>(pl, pr, partials, st);
    }
}

}  // namespace

cudaError_t launch_exp_scan(const Plan &pl, const Problem &pr, const void *packed,
                            Partial *partials, cudaStream_t st)
{
    (void)packed;
    switch (pl.tile.NT) {
    case 128: return launch_nt<128>(pl, pr, partials, st);
    case 64: return launch_nt<64>(pl, pr, partials, st);
    case 32: return launch_nt<32>(pl, pr, partials, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace tfstat
