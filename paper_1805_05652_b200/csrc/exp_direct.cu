// exp_direct.cu -- steps a0 + a3 + a4 + a5 for the exponential window, direct truncated sum
// ("brute-force grid", eq. (4) PAPER.md:44, 3 tau cut PAPER.md:52/238), fused with
// the cell closure (eq. 7) and the marginalisation, batched over templates.
//
// B200 design:
//  * one thread owns C cells (m0..m0+C-1, n): same tau, C consecutive t0.  For fixed tau the
//    weight exp(-(t - t0_c)/tau) = exp(-(t - t_ref)/tau) * const_c, and F is invariant under a
//    per-cell rescaling of the window (A,B,C ~ k^2, Fa,Fb ~ k), so ONE weight
//    w = exp(-(t - t_ref)/tau), t_ref = t0_{m0}, serves all C cells: 1 FMUL + 1 MUFU.EX2 per
//    atom instead of per term.  The plan only picks C > 1 when (C-1) dt0 <= 8 tau_min, so the
//    dropped factor const_c stays within e^-8..1 and nothing underflows.
//  * every term is still accumulated on its own: 7 fp32 FMAs per (cell, atom) pair.  They are
//    issued as packed fma.rn.f32x2 (SASS FFMA2, sm_100): the accumulator pairs are (A,B),
//    (Re Fa, Im Fa), (Re Fb, Im Fb) of one cell and (C_c, C_c+1) of two cells, so the atom
//    operands (a2,b2), (Re Fa, Im Fa), (Re Fb, Im Fb) are the natural 64-bit halves of the
//    staged atom record.  FFMA2 has the lane throughput of FFMA at half the issue slots
//    (measured by tfstat_probe_alu), which leaves room to issue the LDS/MUFU/loop instructions
//    beside a saturated FMA pipe.
//  * lanes of a warp hold consecutive tau_n, so every lane reads the SAME atom: atoms are
//    staged per CTA in shared memory as two 16-byte records (dt, ab | a2, b2) and
//    (Re Fa, Im Fa | Re Fb, Im Fb) and read with broadcast LDS.128; the int->float conversion
//    of the timestamps happens once in the staging, not in the loop.
//  * the window of a CTA is streamed through shared memory in chunks of KC atoms, so a 1-year
//    atom set (13 140 atoms) needs no more shared memory than a 1-day one.
//  * ragged window edges: the atoms [lo_{C-1}, hi_0) belong to all C cells of a thread and are
//    summed with per-thread loop bounds and no predicates; the few head atoms [lo_0, lo_{C-1})
//    and tail atoms [hi_0, hi_{C-1}) are read straight from global memory with 0/1 weights.
//  * a CTA is (one t0 tile) x (NT consecutive tau); the ragged tau block is the one with the
//    SHORTEST windows, and CTAs are launched heaviest (largest tau) first.
#include "plan.h"

// Tuning constants of the core loop, swept on B200 (config 4, 592 templates): staging chunk KC in
// {256, 512, 1024} atoms x unroll in {2 .. 64}.  Unrolling is what matters (unroll 4: 3.79e12
// terms/s, 8: 3.94, 16: 4.10, 24..32: 4.12-4.17, 64: 4.11; the loop counter, the shared-memory address
// arithmetic and the branch are per iteration, and the scheduler gets more independent LDS /
// MUFU to hoist above the FFMA2 stream); KC = 1024 adds ~1 % over 512 (half the barriers).
constexpr int kStageAtoms = 1024;
constexpr int kCoreUnroll = 24;
namespace tfstat {

namespace {

template <int C>
struct Acc {
    u64 ab[C];            // (A, B)
    u64 fa[C];            // (Re Fa, Im Fa)
    u64 fb[C];            // (Re Fb, Im Fb)
    u64 cc[(C + 1) / 2];  // (C of cell 2p, C of cell 2p+1)
};

// one staged atom: rec_a = {(dt, ab), (a2, b2)}, rec_b = {(Re Fa, Im Fa), (Re Fb, Im Fb)}
template <int C>
__device__ __forceinline__ void accumulate_core(Acc<C> &acc, const ulonglong2 ra,
                                                const ulonglong2 rb, const float kexp)
{
    float dt, ab;
    unpack2(ra.x, dt, ab);
    const float w = ex2_approx(dt * kexp);
    const float w2 = w * w;
    // Multiplier as a broadcast scalar, atom operand as a register pair.  Measured on B200
    // (DESIGN.md "FFMA2 operand forms"): this form and the pre-multiplied FADD2 form both end
    // at ~13 terms/clk/SM once the LDS write-backs share the register file with the
    // accumulator updates; two-pair forms (w2 as a pair from FMUL2) are ~2 % slower.
    const u64 ww = pack2(w, w);
    const u64 w2w2 = pack2(w2, w2);
    const u64 abab = pack2(ab, ab);
#pragma unroll
    for (int c = 0; c < C; ++c) {
        ffma2(acc.ab[c], w2w2, ra.y);
        ffma2(acc.fa[c], ww, rb.x);
        ffma2(acc.fb[c], ww, rb.y);
    }
#pragma unroll
    for (int p = 0; p < (C + 1) / 2; ++p) ffma2(acc.cc[p], w2w2, abab);
}

template <int C, int NT, int KC>
__global__ void __launch_bounds__(NT, ((C > 8 ? 384 : 512) / NT) > 12 ? 12 : ((C > 8 ? 384 : 512) / NT))
    exp_direct_kernel(const Problem pr, Partial *__restrict__ partials, const int n_mtiles,
                      const int n_nblocks)
{
    __shared__ ulonglong2 s_a[KC];
    __shared__ ulonglong2 s_b[KC];
    __shared__ Marg s_red[32];
    pdl_trigger();
    pdl_wait();  // bounds_kernel's lo / edge tables

    const Grid g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int64_t tiles = (int64_t)n_mtiles * n_nblocks;
    const int tpl = (int)(blockIdx.x / tiles);
    const int tile = (int)(blockIdx.x % tiles);
    const int nb = n_nblocks - 1 - tile / n_mtiles;  // heaviest (largest tau) first
    const int m0 = (tile % n_mtiles) * C;
    // tau blocks: block 0 holds the N_tau % NT shortest windows (if any), the others are full
    const int ragged = g.N_tau % NT;
    const int n_first = (ragged && nb > 0) ? ragged + (nb - 1) * NT : nb * NT;
    const int n_count = (ragged && nb == 0) ? ragged : NT;
    const bool n_ok = (int)threadIdx.x < n_count;
    const int n = n_first + (n_ok ? (int)threadIdx.x : 0);
    const int m_last = min(m0 + C - 1, g.N_t0 - 1);  // cells beyond N_t0 duplicate the last one

    // per-thread ranges: head [h0, cb) and tail [ce, h1) take 0/1 weights per cell, the core
    // [cb, ce) belongs to all C cells
    const int lo_first = __ldg(bd.lo + m0);
    const int lo_last = __ldg(bd.lo + m_last);
    int h0 = 0, cb = 0, ce = 0, h1 = 0;
    if (n_ok) {
        h0 = lo_first;
        h1 = max(hi_index(bd, g, m_last, n), lo_last);
        cb = lo_last;
        ce = max(hi_index(bd, g, m0, n), lo_first);
        if (ce <= cb) cb = ce = h1;  // no common core: everything goes through the head loop
    }
    // atom range the CTA streams through shared memory: the union of its threads' cores
    const int cta_b = lo_last;
    const int cta_e = hi_index(bd, g, m0, n_first + n_count - 1);

    const long long t_ref = t0_of(g, m0);
    const float kexp = (float)(-1.4426950408889634 / (double)tau_of(g, n));

    const float *__restrict__ base = pr.atoms + (int64_t)tpl * pr.template_stride;
    const int64_t ld = pr.ld;

    Acc<C> acc;
#pragma unroll
    for (int c = 0; c < C; ++c) acc.ab[c] = acc.fa[c] = acc.fb[c] = 0ull;
#pragma unroll
    for (int p = 0; p < (C + 1) / 2; ++p) acc.cc[p] = 0ull;

    // ---- head and tail: atoms that belong to some of the thread's cells only ----------------
#pragma unroll 1
    for (int ph = 0; ph < 2; ++ph) {
        const int xb = ph ? ce : h0, xe = ph ? h1 : cb;
        if (xb >= xe) continue;
        int lo[C], hi[C];
#pragma unroll
        for (int c = 0; c < C; ++c) {
            const int mc = min(m0 + c, g.N_t0 - 1);
            lo[c] = __ldg(bd.lo + mc);
            hi[c] = max(hi_index(bd, g, mc, n), lo[c]);
        }
#pragma unroll 1
        for (int al = xb; al < xe; ++al) {
            const float dt = (float)((long long)__ldg(bd.t + al) - t_ref);
            const float w = ex2_approx(dt * kexp);
            const u64 a2b2 = pack2(__ldg(base + al), __ldg(base + ld + al));
            const float ab = __ldg(base + 2 * ld + al);
            const u64 fa = pack2(__ldg(base + 3 * ld + al), __ldg(base + 4 * ld + al));
            const u64 fb = pack2(__ldg(base + 5 * ld + al), __ldg(base + 6 * ld + al));
            // cells that do not hold this atom are SKIPPED, not weighted by zero: 0 x NaN of a
            // non-finite atom (a bad SFT) would spoil windows it is not part of
            const u64 ww = pack2(w, w);
            const u64 w2 = fmul2(ww, ww);
            const float w2ab = w * w * ab;
#pragma unroll
            for (int c = 0; c < C; ++c) {
                if (al >= lo[c] && al < hi[c]) {
                    ffma2(acc.ab[c], w2, a2b2);
                    ffma2(acc.fa[c], ww, fa);
                    ffma2(acc.fb[c], ww, fb);
                    float c0, c1;
                    unpack2(acc.cc[c / 2], c0, c1);
                    if (c & 1) c1 += w2ab;
                    else c0 += w2ab;
                    acc.cc[c / 2] = pack2(c0, c1);
                }
            }
        }
    }

    // ---- core: atoms common to all C cells, streamed through shared memory ------------------
#pragma unroll 1
    for (int cs = cta_b; cs < cta_e; cs += KC) {
        const int n_stage = min(KC, cta_e - cs);
        // a0: stage atoms [cs, cs + n_stage)
        for (int i = threadIdx.x; i < n_stage; i += NT) {
            const int al = cs + i;
            const float dt = (float)((long long)__ldg(bd.t + al) - t_ref);
            ulonglong2 ra, rb;
            ra.x = pack2(dt, __ldg(base + 2 * ld + al));
            ra.y = pack2(__ldg(base + al), __ldg(base + ld + al));
            rb.x = pack2(__ldg(base + 3 * ld + al), __ldg(base + 4 * ld + al));
            rb.y = pack2(__ldg(base + 5 * ld + al), __ldg(base + 6 * ld + al));
            s_a[i] = ra;
            s_b[i] = rb;
        }
        __syncthreads();
        // a3: weighted sums over this chunk, per-thread bounds
        const int x0 = max(cs, cb) - cs;
        const int x1 = min(cs + n_stage, ce) - cs;
#pragma unroll kCoreUnroll
        for (int i = x0; i < x1; ++i) accumulate_core<C>(acc, s_a[i], s_b[i], kexp);
        __syncthreads();
    }

    // ---- a4 closure + a5 marginals ----------------------------------------------------------
    Marg mg;
    marg_init(mg);
    const int64_t map_base = (int64_t)tpl * g.N_t0 * g.N_tau;
#pragma unroll
    for (int c = 0; c < C; ++c) {
        const int m = m0 + c;
        if (n_ok && m < g.N_t0) {
            float A, B, Cc, cc0, cc1, far, fai, fbr, fbi;
            unpack2(acc.ab[c], A, B);
            unpack2(acc.fa[c], far, fai);
            unpack2(acc.fb[c], fbr, fbi);
            unpack2(acc.cc[c / 2], cc0, cc1);
            Cc = (c & 1) ? cc1 : cc0;
            const int lo_c = __ldg(bd.lo + m);
            const int cnt = max(hi_index(bd, g, m, n) - lo_c, 0);
            uint32_t fl;
            // the sums carry the weight of the tile's first cell; eq. (7) does not care, and the
            // fp64 redo of short ill-conditioned windows uses the cell's own t0
            const float twoF = closure_2F_exp<false>(A, B, Cc, far, fai, fbr, fbi, lo_c, cnt,
                                              pr.min_atoms, fl, base, ld, bd.t, t0_of(g, m),
                                              (double)tau_of(g, n));
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
    return launch_pdl(exp_direct_kernel<C, NT, kStageAtoms>, (unsigned)n_ctas, NT, 0, st, pr, partials,
                      pl.n_mtiles, pl.n_nblocks);
}

template <int C>
cudaError_t launch_c(const Plan &pl, const Problem &pr, Partial *partials, cudaStream_t st)
{
    if (pl.tile.NT == 256) return launch_one<C, 256>(pl, pr, partials, st);
    if (pl.tile.NT == 128) return launch_one<C, 128>(pl, pr, partials, st);
    if (pl.tile.NT == 64) return launch_one<C, 64>(pl, pr, partials, st);
    if (pl.tile.NT == 32) return launch_one<C, 32>(pl, pr, partials, st);
    return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t launch_exp_direct(const Plan &pl, const Problem &pr, Partial *partials,
                              cudaStream_t st)
{
    switch (pl.tile.C) {
    case 16: return launch_c<16>(pl, pr, partials, st);
    case 8: return launch_c<8>(pl, pr, partials, st);
    case 4: return launch_c<4>(pl, pr, partials, st);
    case 2: return launch_c<2>(pl, pr, partials, st);
    case 1: return launch_c<1>(pl, pr, partials, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace tfstat
