// exp_direct.cu -- steps a0 + a3 + a4 + a5 for the exponential window, direct truncated sum
// ("brute-force grid", eq. (4) PAPER.md:44, 3 tau cut PAPER.md:52/238), fused with
// the cell closure (eq. 7) and the marginalisation, batched over templates.
//
// B200 design:
//  * one thread owns C cells (m0..m0+C-1, n): same tau, C consecutive t0.  For fixed tau the
//    weight exp(-(t - t0_c)/tau) = exp(-(t - t_ref)/tau) * const_c, and F is invariant under a
//    per-cell rescaling of the window (A,B,C ~ k^2, Fa,Fb ~ k), so ONE weight
//    w = exp(-(t - t_ref)/tau), t_ref = t0_{m0}, serves all C cells: its argument (1 FFMA) and
//    two MUFU.EX2 (w and w^2) per atom instead of per term.  The plan only picks C > 1 when
//    (C-1) dt0 <= 8 tau_min, so the dropped factor const_c stays within e^-8..1 and nothing
//    underflows.
//  * every term is still accumulated on its own: 7 fp32 FMAs per (cell, atom) pair, issued as
//    packed fma.rn.f32x2 (SASS FFMA2, sm_100) on accumulator pairs of two CELLS of one channel:
//    both multiplicands (weight, atom channel) are then broadcast scalars, the one FFMA2
//    operand form that issues every 2 cycles (a pair x a scalar takes 2.4: tfstat_probe).
//  * lanes of a warp hold consecutive tau_n, so every lane reads the SAME atom: the atoms come
//    as the packed 32-byte records of pack.cu, (dtc, ab | a2, b2) and (Re Fa, Im Fa | Re Fb,
//    Im Fb), and are read with two broadcast LDS.128.
//  * every WARP streams the atoms of its own windows through its own ring of kStages slots of
//    kChunkAtoms records, filled by bulk asynchronous copies (cp.async.bulk + mbarrier): no
//    thread moves atom data, there is no CTA barrier in the loop, and a 1-year atom set needs no
//    more shared memory than a 1-day one.
//  * ragged window edges: the atoms [lo_{C-1}, hi_0) belong to all C cells of a thread and are
//    summed with per-thread loop bounds and no predicates; the few head atoms [lo_0, lo_{C-1})
//    and tail atoms [hi_0, hi_{C-1}) are read straight from global memory and added per cell
//    under a predicate.
//  * a CTA is (one t0 tile) x (NT consecutive tau); the ragged tau block is the one with the
//    SHORTEST windows, and CTAs are launched heaviest (largest tau) first.  SPLIT (single maps):
//    the warps of a CTA share 32 tau values and split the atoms of their windows instead.
#include "plan.h"

// Tuning constants of the core loop, swept on B200 (config 4).  Unrolling is what matters (round
// 1's loop: unroll 4: 3.79e12 terms/s, 8: 3.94, 16: 4.10, 24..32: 4.12-4.17, 64: 4.11; the loop
// counter, the shared-memory address arithmetic and the branch are per iteration, and the
// scheduler gets more independent LDS / MUFU to hoist above the FFMA2 stream).
constexpr int kChunkAtoms = 192;  // atoms per bulk copy (6 KB); divides kPackBlock
constexpr int kStages = 2;        // ring slots per warp
constexpr int kCoreUnroll = 24;   // divides kChunkAtoms
namespace tfstat {

namespace {

static_assert(kPackBlock % kChunkAtoms == 0, "a staged chunk must lie inside one packed time block");
static_assert(kChunkAtoms % kCoreUnroll == 0, "whole unrolled trips per full chunk");

// Accumulators: channel k of the cells (2p, 2p + 1) as one packed fp32x2 pair.
//   k: 0 A, 1 B, 2 C, 3 Re Fa, 4 Im Fa, 5 Re Fb, 6 Im Fb
// The C cells of a thread share the weight AND the atom, so a pair of CELLS is updated by one
// fma.rn.f32x2 whose two multiplicands are both broadcast scalars (SASS: FFMA2 Racc, Rw.F32,
// Rx.F32, Racc).  Measured on B200 (profiles/r02_ffma2_forms.md): this is the one packed form
// that issues every 2 clocks; a register-pair multiplicand (channel pairs of ONE cell: the
// round-1 layout) takes 2.4.  Isolated loop, C = 8: 15.85 against 15.20 terms/clk/SM; C = 16:
// 16.60 against 15.98.
template <int C>
struct Acc {
    u64 ch[7][(C + 1) / 2];
};

template <int C>
__device__ __forceinline__ void acc_zero(Acc<C> &acc)
{
#pragma unroll
    for (int k = 0; k < 7; ++k)
#pragma unroll
        for (int p = 0; p < (C + 1) / 2; ++p) acc.ch[k][p] = 0ull;
}

// one staged atom: rec_a = {(dtc, ab), (a2, b2)}, rec_b = {(Re Fa, Im Fa), (Re Fb, Im Fb)};
// weight argument (t - t_ref) kexp = dtc kexp + cexp (pack.cu)
template <int C>
__device__ __forceinline__ void accumulate_core(Acc<C> &acc, const ulonglong2 ra,
                                                const ulonglong2 rb, const float kexp,
                                                const float cexp)
{
    float x[7], dt;
    unpack2(ra.x, dt, x[2]);
    unpack2(ra.y, x[0], x[1]);
    unpack2(rb.x, x[3], x[4]);
    unpack2(rb.y, x[5], x[6]);
    const float arg = fmaf(fabsf(dt), kexp, cexp);  // (sign bit of dtc: a flag, pack.cu)
    const float w = ex2_approx(arg);
    // w^2 = 2^(2 arg) by a second MUFU.EX2 on the argument with its exponent field bumped by one
    // (an integer add on the ALU pipe): takes the multiply w * w off the FMA pipe, which is what
    // this loop is bound by (measured on B200, config 4: 4.43e12 -> 4.49e12 terms/s).  arg = 0
    // becomes 2^-126 and 2^that = 1, as it must.  A NaN argument (a bad SFT: pack.cu) does NOT
    // survive the integer add -- w is NaN, w2 is not: close_cell flags the cell.
    const float w2 = ex2_approx(__int_as_float(__float_as_int(arg) + 0x00800000));
    const u64 ww = pack2(w, w);
    const u64 w2w2 = pack2(w2, w2);
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        const u64 xx = pack2(x[k], x[k]);
#pragma unroll
        for (int p = 0; p < (C + 1) / 2; ++p) ffma2(acc.ch[k][p], k < 3 ? w2w2 : ww, xx);
    }
}

// cell c alone (head / tail atoms that belong to some of the thread's cells only): a scalar FMA on
// one half of the pair
template <int C>
__device__ __forceinline__ void accumulate_cell(Acc<C> &acc, const int c, const float w,
                                                const float w2, const float (&x)[7])
{
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        float lo, hi;
        unpack2(acc.ch[k][c / 2], lo, hi);
        if (c & 1) hi = fmaf(k < 3 ? w2 : w, x[k], hi);
        else lo = fmaf(k < 3 ? w2 : w, x[k], lo);
        acc.ch[k][c / 2] = pack2(lo, hi);
    }
}

// Staging: every WARP streams the atoms of its own windows through its own ring
// of kStages slots of kChunkAtoms packed atoms, filled by bulk asynchronous copies
// (cp.async.bulk global -> shared, one elected lane issues them, completion on the slot's
// mbarrier).  No thread moves atom data, and there is no CTA barrier in the loop: a warp waits
// for its own data only, never for the other warps of the CTA (whose windows -- larger tau --
// are longer).
//
// SPLIT (single maps: too few CTAs to fill 148 SMs several times over): the NW warps of a CTA
// share the SAME 32 tau values and split the atoms of their windows between them, chunk k to warp
// k mod NW; their partial sums meet in shared memory at the end and the cells are closed by
// the warps in turn.  Same arithmetic per term; a CTA's critical path is NW times shorter and
// every warp of it carries the same load, so the tail of a small grid shrinks accordingly
// (config 2: 0.176 -> see DESIGN.md 6.1).
template <int C, int NT, int KW, int NS, bool SPLIT>
__global__ void __launch_bounds__(NT, (C > 8 ? 384 : 512) / NT)
    exp_direct_kernel(const Problem pr, const ulonglong2 *__restrict__ packed, const int n_pad,
                      Partial *__restrict__ partials, const int n_mtiles, const int n_nblocks)
{
    constexpr int NW = NT / 32;
    extern __shared__ __align__(128) unsigned char smem_raw[];  // rings: [NW][NS][2 KW] x 16 B
    __shared__ __align__(8) unsigned long long s_bar[NW][NS];
    __shared__ Marg s_red[32];

    const Grid g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t tiles = (int64_t)n_mtiles * n_nblocks;
    const int tpl = (int)(blockIdx.x / tiles);
    const int tile = (int)(blockIdx.x % tiles);
    const int nb = n_nblocks - 1 - tile / n_mtiles;  // heaviest (largest tau) first
    const int m0 = (tile % n_mtiles) * C;
    // Warp w of a CTA runs on scheduler w of its SM, and the windows of a CTA grow with the warp
    // index (32 more tau values each): left alone, scheduler 0 of every SM would get the lightest
    // quarter of every resident CTA and scheduler NW-1 the heaviest.  Rotating the quarter a warp
    // takes with the CTA index evens the schedulers out.
    const int tq = SPLIT ? lane : ((warp + (int)(blockIdx.x % NW)) % NW) * 32 + lane;  // tau slot
    // tau blocks: block 0 holds the N_tau % TPB shortest windows (if any), the others are full
    constexpr int TPB = SPLIT ? 32 : NT;  // tau values per CTA
    const int ragged = g.N_tau % TPB;
    const int n_first = (ragged && nb > 0) ? ragged + (nb - 1) * TPB : nb * TPB;
    const int n_count = (ragged && nb == 0) ? ragged : TPB;
    const bool n_ok = tq < n_count;
    const int n = n_first + (n_ok ? tq : 0);
    const int m_last = min(m0 + C - 1, g.N_t0 - 1);  // cells beyond N_t0 duplicate the last one

    const uint32_t bar0 = smem_u32(&s_bar[warp][0]);
    constexpr uint32_t kChunkBytes = 2 * KW * sizeof(ulonglong2);
    const ulonglong2 *s_ring = reinterpret_cast<const ulonglong2 *>(smem_raw) + warp * (NS * 2 * KW);
    const uint32_t ring0 = smem_u32(s_ring);
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(bar0 + 8 * s, 1);
        mbar_fence_init();
    }
    __syncwarp();

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
    }
    const bool has_core = ce > cb;  // else: windows shorter than the tile's t0 span (or no cell)
    // atom range the WARP streams through its ring: the union of its threads' cores, in whole
    // chunks of KW atoms aligned to multiples of KW (one packed time base per chunk)
    const int warp_b = lo_last;
    const int warp_e = __reduce_max_sync(0xffffffffu, has_core ? ce : 0);
    const int q0 = warp_b / KW;
    const int nq = warp_e > warp_b ? (warp_e + KW - 1) / KW - q0 : 0;
    constexpr int KSTEP = SPLIT ? NW : 1;  // this warp's chunks: k0, k0 + KSTEP, ...
    const int k0 = SPLIT ? warp : 0;
    const ulonglong2 *__restrict__ rec = packed + (int64_t)tpl * n_pad * 2;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s)
            if (k0 + s * KSTEP < nq)
                bulk_load(ring0 + s * kChunkBytes, rec + (int64_t)(q0 + k0 + s * KSTEP) * KW * 2,
                          kChunkBytes, bar0 + 8 * s);
    }

    const long long t_ref = t0_of(g, m0);
    const float kexp = (float)(-1.4426950408889634 / (double)tau_of(g, n));

    const float *__restrict__ base = pr.atoms + (int64_t)tpl * pr.template_stride;
    const int64_t ld = pr.ld;

    Acc<C> acc;
    acc_zero<C>(acc);

    // ---- head and tail: atoms that belong to some of the thread's cells only ----------------
    // (measured on B200, config 4: an unrolled "staircase" -- the atoms in [lo_c, lo_c+1) belong
    // to cells 0..c, so every step adds to a fixed set of cells without predicates -- is 2.4 %
    // SLOWER than this plain predicated loop: twice the code, one short loop per step)
#pragma unroll 1
    for (int ph = 0; ph < 2; ++ph) {
        if (SPLIT && warp != (ph ? NW - 1 : 0)) continue;  // head: first warp, tail: last warp
        const int xb = has_core ? (ph ? ce : h0) : (ph ? h1 : h0);
        const int xe = has_core ? (ph ? h1 : cb) : h1;
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
            const float w2 = w * w;
            float x[7];
#pragma unroll
            for (int k = 0; k < 7; ++k) x[k] = __ldg(base + k * ld + al);
            // cells that do not hold this atom are SKIPPED, not weighted by zero: 0 x NaN of a
            // non-finite atom (a bad SFT) would spoil windows it is not part of
#pragma unroll
            for (int c = 0; c < C; ++c)
                if (al >= lo[c] && al < hi[c]) accumulate_cell<C>(acc, c, w, w2, x);
        }
    }

    // ---- core: atoms common to all C cells, streamed through the warp's ring ----------------
#pragma unroll 1
    for (int k = k0, j = 0; k < nq; k += KSTEP, ++j) {
        const int s = j % NS;
        const int cs = (q0 + k) * KW;  // first atom of the chunk
        // weight argument of atom i: dtc_i kexp + cexp, dtc_i relative to the chunk's time base
        const int tb = __ldg(bd.t + cs - cs % kPackBlock);
        const float cexp = (float)((long long)tb - t_ref) * kexp;
        const int x0 = max(cs, cb) - cs;
        const int x1 = has_core ? min(cs + KW, ce) - cs : x0;
        mbar_wait(bar0 + 8 * s, (uint32_t)(j / NS) & 1u);
        const ulonglong2 *__restrict__ slot = s_ring + s * (2 * KW);
#pragma unroll kCoreUnroll
        for (int i = x0; i < x1; ++i)
            accumulate_core<C>(acc, slot[2 * i], slot[2 * i + 1], kexp, cexp);
        __syncwarp();  // every lane is done with the slot: refill it
        if (lane == 0 && k + NS * KSTEP < nq)
            bulk_load(ring0 + s * kChunkBytes, rec + (int64_t)(q0 + k + NS * KSTEP) * KW * 2,
                      kChunkBytes, bar0 + 8 * s);
    }

    // ---- a4 closure + a5 marginals ----------------------------------------------------------
    Marg mg;
    marg_init(mg);
    const int64_t map_base = (int64_t)tpl * g.N_t0 * g.N_tau;
    auto close_cell = [&](const int c, const float(&S)[7]) {
        const int m = m0 + c;
        if (n_ok && m < g.N_t0) {
            const int lo_c = __ldg(bd.lo + m);
            const int cnt = max(hi_index(bd, g, m, n) - lo_c, 0);
            uint32_t fl;
            // the sums carry the weight of the tile's first cell; eq. (7) does not care, and the
            // fp64 redo of short ill-conditioned windows uses the cell's own t0
            float twoF = closure_2F_exp<false>(S[0], S[1], S[2], S[3], S[4], S[5], S[6], lo_c,
                                                     cnt, pr.min_atoms, fl, base, ld, bd.t,
                                                     t0_of(g, m), (double)tau_of(g, n));
            // a bad SFT among the core atoms made w NaN but not w2 (accumulate_core): Fa, Fb are
            // NaN while D is fine, and eq. (7) comes out NaN: the cell is degenerate (flag bit 1),
            // as it is when D itself is NaN.  (Carrying the NaN over to A in front of the closure
            // instead cost 1.8 %: the register allocation of the loop is that touchy.)
            if (twoF != twoF) {
                twoF = 0.0f;
                fl = 2u;
            }
            const int32_t flat = m * g.N_tau + n;
            if (pr.out_maps) pr.out_maps[map_base + flat] = twoF;
            if (pr.out_flags) pr.out_flags[map_base + flat] = (uint8_t)fl;
            if (!fl) marg_add(mg, twoF, flat);
        }
    };
    constexpr int CP = (C + 1) / 2;
    if (SPLIT) {
        // the warps' partial sums meet in shared memory (the rings are done with), pair p of
        // every channel is summed and closed by warp p mod NW
        __syncthreads();
        u64 *red = reinterpret_cast<u64 *>(smem_raw);  // [NW][7][CP][32]
#pragma unroll
        for (int k = 0; k < 7; ++k)
#pragma unroll
            for (int p = 0; p < CP; ++p) red[((warp * 7 + k) * CP + p) * 32 + lane] = acc.ch[k][p];
        __syncthreads();
#pragma unroll
        for (int p = 0; p < CP; ++p) {
            if (p % NW != warp) continue;
            float S0[7], S1[7];
#pragma unroll
            for (int k = 0; k < 7; ++k) {
                float e = 0.0f, o = 0.0f;
#pragma unroll
                for (int w = 0; w < NW; ++w) {
                    float pe, po;
                    unpack2(red[((w * 7 + k) * CP + p) * 32 + lane], pe, po);
                    e += pe;
                    o += po;
                }
                S0[k] = e;
                S1[k] = o;
            }
            close_cell(2 * p, S0);
            if (2 * p + 1 < C) close_cell(2 * p + 1, S1);
        }
    } else {
#pragma unroll
        for (int c = 0; c < C; ++c) {
            float S[7];
#pragma unroll
            for (int k = 0; k < 7; ++k) {
                float e, o;
                unpack2(acc.ch[k][c / 2], e, o);
                S[k] = (c & 1) ? o : e;
            }
            close_cell(c, S);
        }
    }
    if (partials) {
        marg_block_reduce<NT>(mg, s_red);
        if (threadIdx.x == 0) partial_store(partials + blockIdx.x, mg);
    }
}

template <int C, int NT>
cudaError_t launch_one(const Plan &pl, const Problem &pr, const void *packed, Partial *partials,
                       cudaStream_t st)
{
    const int64_t n_ctas = pl.tiles_per_template * pl.n_templates;
    const size_t smem = (size_t)(NT / 32) * kStages * 2 * kChunkAtoms * sizeof(ulonglong2);
    auto go = [&](auto kern) -> cudaError_t {
        cudaError_t e =
            cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        return launch_k(kern, (unsigned)n_ctas, NT, smem, st, pr,
                          static_cast<const ulonglong2 *>(packed), pl.n_pad, partials, pl.n_mtiles,
                          pl.n_nblocks);
    };
    if constexpr (C <= 8 && NT == 128) {  // the partial sums of the split form fit in the rings
        static_assert((size_t)(NT / 32) * 7 * ((C + 1) / 2) * 32 * 8 <=
                      (size_t)(NT / 32) * kStages * 2 * kChunkAtoms * sizeof(ulonglong2));
        if (pl.tile.split) return go(exp_direct_kernel<C, NT, kChunkAtoms, kStages, true>);
    }
    return go(exp_direct_kernel<C, NT, kChunkAtoms, kStages, false>);
}

template <int C>
cudaError_t launch_c(const Plan &pl, const Problem &pr, const void *packed, Partial *partials,
                     cudaStream_t st)
{
    if (pl.tile.NT == 256) return launch_one<C, 256>(pl, pr, packed, partials, st);
    if (pl.tile.NT == 128) return launch_one<C, 128>(pl, pr, packed, partials, st);
    if (pl.tile.NT == 64) return launch_one<C, 64>(pl, pr, packed, partials, st);
    if (pl.tile.NT == 32) return launch_one<C, 32>(pl, pr, packed, partials, st);
    return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t launch_exp_direct(const Plan &pl, const Problem &pr, const void *packed,
                              Partial *partials, cudaStream_t st)
{
    switch (pl.tile.C) {
    case 16: return launch_c<16>(pl, pr, packed, partials, st);
    case 8: return launch_c<8>(pl, pr, packed, partials, st);
    case 4: return launch_c<4>(pl, pr, packed, partials, st);
    case 2: return launch_c<2>(pl, pr, packed, partials, st);
    case 1: return launch_c<1>(pl, pr, packed, partials, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace tfstat
