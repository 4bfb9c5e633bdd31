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

namespace tfstat {

namespace {

constexpr float kReanchor = 4.0f;  // move t_ref when (t_ref - t0_m)/tau exceeds this
constexpr float kGuard = 64.0f;    // re-sum a window whose A fell below 1/kGuard of its maximum
constexpr int kSlideChunk = 128;   // atoms per bulk copy and template (4 KB); divides kPackBlock
constexpr int kSlideStages = 3;    // ring slots per CTA
constexpr int kWindowUnroll = 8;   // unroll of the initial-window loop
static_assert(kPackBlock % kSlideChunk == 0, "a staged chunk must lie inside one packed time block");

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

// acc += s * E x  (s = +1 entering, -1 leaving): w carries the sign, w2 = w * |w|;
// ra = {(dtc, ab), (a2, b2)}, rb = {(Re Fa, Im Fa), (Re Fb, Im Fb)}: one packed atom (pack.cu)
__device__ __forceinline__ void acc_add(SlideAcc &a, const float w, const float w2,
                                        const ulonglong2 ra, const ulonglong2 rb)
{
    float dtc, ab;
    unpack2(ra.x, dtc, ab);
    const u64 ww = pack2(w, w);
    ffma2(a.ab, pack2(w2, w2), ra.y);
    ffma2(a.fa, ww, rb.x);
    ffma2(a.fb, ww, rb.y);
    a.c = fmaf(w2, ab, a.c);
}

__device__ __forceinline__ void acc_scale(SlideAcc &a, const float c)
{
    const float c2 = c * c;
    a.ab = fmul2(a.ab, pack2(c2, c2));
    a.fa = fmul2(a.fa, pack2(c, c));
    a.fb = fmul2(a.fb, pack2(c, c));
    a.c *= c2;
}

__device__ __forceinline__ void mbar_expect_tx(const uint32_t bar, const uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(const uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_copy(const uint32_t dst, const void *src, const uint32_t bytes,
                                          const uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(dst), "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}

// ---------------------------------------------------------------------------------------
// exp_slide_kernel: a thread owns RT tau values (n, n + NT, ..) x TPC templates.  The weights E_a
// depend on (atom, tau) only, so one MUFU.EX2 (+ its argument and E^2) serves the TPC templates,
// and one broadcast LDS.128 pair of an atom serves the RT tau values.
//
// The atoms of the initial window (more than 90 % of the weighted terms of this form) come through
// a ring of kSlideStages slots shared by the CTA, filled by bulk asynchronous copies from the
// packed records (cp.async.bulk + mbarrier; thread 0 issues them, a slot is refilled once every
// warp has released it): no thread moves atom data, no CTA barrier in the loop.  While sliding,
// the atoms that enter (the same for every thread of the CTA) and leave (one gather per thread)
// are read from the same records with two 16-byte loads each.
//
// Also measured (B200, config 4): the initial window sums in a kernel of their own with the LANES
// ON ATOMS (a lane loads its own atom, the warp walks 8 tau values in uniform registers, a
// transposing butterfly combines the 56 partial sums per lane): 4.2-4.8 terms/clk/SM against
// ~9.8 for the broadcast form below, whichever way the loads were staged -- one MUFU per term
// and lane instead of one per TPC terms, and half the lanes idle at the window's ragged end.
// ---------------------------------------------------------------------------------------
template <int NT, int RT, int TPC, bool STATS>
__global__ void __launch_bounds__(NT, RT * TPC <= 2 ? (NT == 128 ? 5 : 1) : (NT == 128 ? 3 : 1))
    exp_slide_kernel(const Problem pr, const ulonglong2 *__restrict__ packed, const int n_pad,
                     Partial *__restrict__ partials, const int n_nblocks, const int n_segs,
                     const int seg_len, unsigned long long *__restrict__ stats)
{
    constexpr int KW = kSlideChunk, NS = TPC > 2 ? 2 : kSlideStages, NW = NT / 32;
    constexpr uint32_t kTplBytes = KW * 2 * sizeof(ulonglong2);  // one template's share of a slot
    __shared__ __align__(128) ulonglong2 s_ring[NS][TPC][2 * KW];
    __shared__ __align__(8) unsigned long long s_full[NS], s_empty[NS];
    __shared__ Marg s_red[32];
    pdl_trigger();

    const Grid g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int lane = threadIdx.x & 31;
    // blockIdx.x = (tplgrp * n_segs + seg) * n_nblocks + j, heaviest tau block (largest tau) first
    const int j = (int)(blockIdx.x % n_nblocks);
    const int seg = (int)((blockIdx.x / n_nblocks) % n_segs);
    const int tpl0 = (int)(blockIdx.x / ((int64_t)n_nblocks * n_segs)) * TPC;
    const int nb = n_nblocks - 1 - j;
    const int n_first = nb * (NT * RT);
    const int n_count = min(NT * RT, g.N_tau - n_first);
    const int m_beg = seg * seg_len;
    const int m_end = min(m_beg + seg_len, g.N_t0);

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            mbar_init(smem_u32(&s_full[s]), 1);
            mbar_init(smem_u32(&s_empty[s]), NW);
        }
        mbar_fence_init();
    }
    __syncthreads();
    pdl_wait();  // bounds_kernel's lo / edge tables, pack_atoms_kernel's records

    // templates beyond the batch (ragged last group) alias the last real one; nothing of theirs
    // is stored
    const ulonglong2 *__restrict__ rec[TPC];
    const float *__restrict__ base[TPC];
#pragma unroll
    for (int q = 0; q < TPC; ++q) {
        const int tq = min(tpl0 + q, pr.n_templates - 1);
        rec[q] = packed + (int64_t)tq * n_pad * 2;
        base[q] = pr.atoms + (int64_t)tq * pr.template_stride;
    }
    const int64_t ld = pr.ld;

    // this thread's tau values
    bool n_ok[RT];
    int n[RT];
    float kexp[RT], inv_tau[RT];
#pragma unroll
    for (int r = 0; r < RT; ++r) {
        const int slot = r * NT + (int)threadIdx.x;
        n_ok[r] = slot < n_count;
        n[r] = n_first + (n_ok[r] ? slot : 0);
        const double tau = (double)tau_of(g, n[r]);
        kexp[r] = (float)(-1.4426950408889634 / tau);
        inv_tau[r] = (float)(1.0 / tau);
    }

    // ---- initial window: cell (m_end - 1, n), streamed through the ring ----------------------
    int m = m_end - 1;
    int lo_m = __ldg(bd.lo + m);
    int hi[RT];
    int t_ref[RT];  // seconds (int32: every grid time fits, TFSTAT_EOVERFLOW otherwise)
#pragma unroll
    for (int r = 0; r < RT; ++r) {
        hi[r] = n_ok[r] ? max(hi_index(bd, g, m, n[r]), lo_m) : lo_m;
        t_ref[r] = (int)t0_of(g, m);
    }
    const int cta_e = max(hi_index(bd, g, m, n_first + n_count - 1), lo_m);  // hi is monotone in n
    const int q0 = lo_m / KW;
    const int nq = cta_e > lo_m ? (cta_e + KW - 1) / KW - q0 : 0;
    auto fill = [&](const int k) {  // thread 0: chunk k -> slot k % NS
        const int s = k % NS;
        const uint32_t bar = smem_u32(&s_full[s]);
        mbar_expect_tx(bar, TPC * kTplBytes);
#pragma unroll
        for (int q = 0; q < TPC; ++q)
            bulk_copy(smem_u32(&s_ring[s][q][0]), rec[q] + (int64_t)(q0 + k) * KW * 2, kTplBytes, bar);
    };
    if (threadIdx.x == 0)
        for (int k = 0; k < NS && k < nq; ++k) fill(k);

    SlideAcc acc[RT][TPC];
#pragma unroll
    for (int r = 0; r < RT; ++r)
#pragma unroll
        for (int q = 0; q < TPC; ++q) acc_zero(acc[r][q]);
    unsigned n_term[4] = {0u, 0u, 0u, 0u};  // STATS: window, enter, leave, re-sum (x TPC templates)

    int hi_max = hi[0];
#pragma unroll
    for (int r = 1; r < RT; ++r) hi_max = max(hi_max, hi[r]);
#pragma unroll 1
    for (int k = 0; k < nq; ++k) {
        const int s = k % NS;
        const int cs = (q0 + k) * KW;
        // refill the slot of chunk k - 1 with chunk k - 1 + NS once every warp has released it
        if (threadIdx.x == 0 && k >= 1 && k - 1 + NS < nq) {
            mbar_wait(smem_u32(&s_empty[(k - 1) % NS]), (uint32_t)((k - 1) / NS) & 1u);
            fill(k - 1 + NS);
        }
        const int tb = __ldg(bd.t + cs - cs % kPackBlock);
        float cexp[RT];
#pragma unroll
        for (int r = 0; r < RT; ++r) cexp[r] = (float)(tb - t_ref[r]) * kexp[r];
        const int x0 = max(cs, lo_m) - cs;
        const int x1 = min(cs + KW, hi_max) - cs;
        mbar_wait(smem_u32(&s_full[s]), (uint32_t)(k / NS) & 1u);
#pragma unroll kWindowUnroll
        for (int i = x0; i < x1; ++i) {
            ulonglong2 ra[TPC], rb[TPC];
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                ra[q] = s_ring[s][q][2 * i];
                rb[q] = s_ring[s][q][2 * i + 1];
            }
            float dtc, ab0;
            unpack2(ra[0].x, dtc, ab0);
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                // atoms beyond this tau's own window are skipped, never weighted by zero (0 x NaN)
                if (RT == 1 || cs + i < hi[r]) {
                    const float e = ex2_approx(fmaf(dtc, kexp[r], cexp[r]));
                    const float e2 = e * e;
#pragma unroll
                    for (int q = 0; q < TPC; ++q) acc_add(acc[r][q], e, e2, ra[q], rb[q]);
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&s_empty[s]));
    }
    if (STATS) {
#pragma unroll
        for (int r = 0; r < RT; ++r) n_term[0] += (unsigned)(hi[r] - lo_m);
    }
    float A_max[RT][TPC];
#pragma unroll
    for (int r = 0; r < RT; ++r)
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
            float A, B;
            unpack2(acc[r][q].ab, A, B);
            A_max[r][q] = A;
        }

    // one atom straight from the packed records (entering / leaving / re-summed atoms), one weight
    // for the TPC templates
    auto add_global = [&](const int r, const int al, const float sign) {
        const float dt = (float)(__ldg(bd.t + al) - t_ref[r]);
        const float e = ex2_approx(dt * kexp[r]);
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
            const ulonglong2 ra = __ldg(rec[q] + 2 * (int64_t)al), rb = __ldg(rec[q] + 2 * (int64_t)al + 1);
            float dtc, ab;
            unpack2(ra.x, dtc, ab);
            const float eq = fmaf(dtc, 0.0f, e);  // NaN for an atom that is not finite (pack.cu)
            const float w = sign * eq;
            acc_add(acc[r][q], w, w * eq, ra, rb);
        }
    };

    // ---- slide backwards in t0: closure of cell m, then step to m - 1 ------------------------
    Marg mg[RT][TPC];
#pragma unroll
    for (int r = 0; r < RT; ++r)
#pragma unroll
        for (int q = 0; q < TPC; ++q) marg_init(mg[r][q]);
    const int64_t cells = (int64_t)g.N_t0 * g.N_tau;
#pragma unroll 1
    for (;;) {
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            if (!n_ok[r]) continue;
            const int32_t flat = m * g.N_tau + n[r];
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                if (tpl0 + q >= pr.n_templates) continue;
                float A, B, far, fai, fbr, fbi;
                unpack2(acc[r][q].ab, A, B);
                unpack2(acc[r][q].fa, far, fai);
                unpack2(acc[r][q].fb, fbr, fbi);
                uint32_t fl;
                const float twoF = closure_2F_exp<false>(
                    A, B, acc[r][q].c, far, fai, fbr, fbi, lo_m, hi[r] - lo_m, pr.min_atoms, fl,
                    base[q], ld, bd.t, t0_of(g, m), (double)tau_of(g, n[r]));
                const int64_t o = (int64_t)(tpl0 + q) * cells + flat;
                if (pr.out_maps) pr.out_maps[o] = twoF;
                if (pr.out_flags) pr.out_flags[o] = (uint8_t)fl;
                if (!fl) marg_add(mg[r][q], twoF, flat);
            }
        }
        if (m == m_beg) break;
        const int m2 = m - 1;
        const int lo2 = __ldg(bd.lo + m2);
        const int t0_2 = (int)t0_of(g, m2);
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            const int hi2 = n_ok[r] ? max(hi_index(bd, g, m2, n[r]), lo2) : lo2;
            bool fresh = (hi2 <= lo_m) || (hi2 == lo2);  // no overlap with window m, or empty
            if (!fresh) {
                const float sh = (float)(t_ref[r] - t0_2);
                if (sh * inv_tau[r] > kReanchor) {  // keep the weights of entering atoms <= e^kReanchor
                    const float c = ex2_approx(sh * kexp[r]);
#pragma unroll
                    for (int q = 0; q < TPC; ++q) {
                        acc_scale(acc[r][q], c);
                        A_max[r][q] *= c * c;
                    }
                    t_ref[r] = t0_2;
                }
                for (int al = lo2; al < lo_m; ++al) add_global(r, al, 1.0f);  // entering, low end
                const int lv = max(hi2, lo_m);
                for (int al = lv; al < hi[r]; ++al) add_global(r, al, -1.0f);  // leaving, high end
                if (STATS) {
                    n_term[1] += (unsigned)(lo_m - lo2);
                    n_term[2] += (unsigned)max(hi[r] - lv, 0);
                }
#pragma unroll
                for (int q = 0; q < TPC; ++q) {
                    float A, B;
                    unpack2(acc[r][q].ab, A, B);
                    A_max[r][q] = fmaxf(A_max[r][q], A);
                    // a window that lost most of its weight is re-summed (for all TPC templates:
                    // a fresh sum is always right); written so that a NaN / inf atom in the
                    // running sums also forces a fresh sum: once it has left the window it must
                    // not linger
                    fresh = fresh || !(A * kGuard >= A_max[r][q]);
                }
            }
            if (fresh) {
#pragma unroll
                for (int q = 0; q < TPC; ++q) acc_zero(acc[r][q]);
                t_ref[r] = t0_2;
                for (int al = lo2; al < hi2; ++al) add_global(r, al, 1.0f);
                if (STATS) n_term[3] += (unsigned)(hi2 - lo2);
#pragma unroll
                for (int q = 0; q < TPC; ++q) {
                    float A, B;
                    unpack2(acc[r][q].ab, A, B);
                    A_max[r][q] = A;
                }
            }
            hi[r] = hi2;
        }
        m = m2;
        lo_m = lo2;
    }
    if (STATS) {
        // (terms of out-of-range tau slots and of ragged template groups were not summed for real)
        unsigned long long v[5];
        const unsigned long long ntpl = (unsigned long long)min(TPC, pr.n_templates - tpl0);
        int n_mine = 0;
#pragma unroll
        for (int r = 0; r < RT; ++r) n_mine += n_ok[r] ? 1 : 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = (unsigned long long)n_term[i] * ntpl;
        v[4] = (unsigned long long)n_mine * (unsigned long long)(m_end - m_beg) * ntpl;
#pragma unroll
        for (int i = 0; i < 5; ++i) {
#pragma unroll
            for (int sft = 16; sft >= 1; sft >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], sft);
            if (lane == 0 && v[i]) atomicAdd(stats + i, v[i]);
        }
    }
    if (partials) {
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
            Marg a = mg[0][q];
#pragma unroll
            for (int r = 1; r < RT; ++r) marg_merge(a, mg[r][q]);
            if (q > 0) __syncthreads();  // s_red is reused
            marg_block_reduce<NT>(a, s_red);
            if (threadIdx.x == 0 && tpl0 + q < pr.n_templates)
                partial_store(partials + ((int64_t)(tpl0 + q) * n_segs + seg) * n_nblocks + j, a);
        }
    }
}

template <int NT, int RT, int TPC>
cudaError_t launch_tpc(const Plan &pl, const Problem &pr, const ulonglong2 *packed,
                       Partial *partials, cudaStream_t st)
{
    const int64_t groups = (pl.n_templates + TPC - 1) / TPC;
    const int64_t n_ctas = (int64_t)pl.n_nblocks * pl.n_segs * groups;
    if (pl.stats)
        return launch_pdl(exp_slide_kernel<NT, RT, TPC, true>, (unsigned)n_ctas, NT, 0, st, pr,
                          packed, pl.n_pad, partials, pl.n_nblocks, pl.n_segs, pl.seg_len, pl.stats);
    return launch_pdl(exp_slide_kernel<NT, RT, TPC, false>, (unsigned)n_ctas, NT, 0, st, pr, packed,
                      pl.n_pad, partials, pl.n_nblocks, pl.n_segs, pl.seg_len, pl.stats);
}

template <int NT>
cudaError_t launch_nt(const Plan &pl, const Problem &pr, const ulonglong2 *packed,
                      Partial *partials, cudaStream_t st)
{
    if (pl.slide_rt == 2) {
        if (pl.slide_tpc == 2) return launch_tpc<NT, 2, 2>(pl, pr, packed, partials, st);
        return launch_tpc<NT, 2, 1>(pl, pr, packed, partials, st);
    }
    switch (pl.slide_tpc) {
    case 4: return launch_tpc<NT, 1, 4>(pl, pr, packed, partials, st);
    case 2: return launch_tpc<NT, 1, 2>(pl, pr, packed, partials, st);
    default: return launch_tpc<NT, 1, 1>(pl, pr, packed, partials, st);
    }
}

}  // namespace

cudaError_t launch_exp_scan(const Plan &pl, const Problem &pr, const void *packed,
                            Partial *partials, cudaStream_t st)
{
    const ulonglong2 *rec = static_cast<const ulonglong2 *>(packed);
    switch (pl.tile.NT) {
    case 128: return launch_nt<128>(pl, pr, rec, partials, st);
    case 64: return launch_nt<64>(pl, pr, rec, partials, st);
    case 32: return launch_nt<32>(pl, pr, rec, partials, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace tfstat
